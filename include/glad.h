/*
 * glad.h -- C ABI of libglad: batched joint lensing + dynamics log-likelihood on one
 * NVIDIA B200 (sm_100a).  Method: arXiv 2504.01302 ("GLaD"); "P:n" = PAPER.md line n;
 * "R-xx" = a reading listed in DESIGN.md where the paper prints no formula.
 *
 * Conventions common to every call
 *   - All `d_` pointers are DEVICE pointers owned by the caller.  The library never
 *     allocates or frees caller-visible memory; a context keeps grow-only device scratch.
 *     Static-data pointers passed to glad_set_* are BORROWED: keep them alive and unchanged
 *     until they are replaced or the context is destroyed.
 *   - Batch calls only ENQUEUE work on the context's stream and return; no implicit D2H copy and
 *     no host sync, except that a call which needs MORE context scratch than any call before it
 *     (the first call, or a larger batch) synchronises the context's streams once while the
 *     scratch is re-allocated.  glad_set_kin_data is synchronous (documented there).
 *   - Every call makes the context's device current for its own duration and restores the
 *     caller's current device before returning.  The library reads no environment variable.
 *   - Errors detectable on the host return a negative glad_status at once; a CUDA
 *     launch/runtime error returns GLAD_ECUDA with the CUDA text in glad_last_error().
 *     No exceptions, no exit(), no printing.  There is no CPU fallback.
 *   - A physically invalid parameter VECTOR is not an error: its outputs are
 *     lnL = -INFINITY, chi2 = +INFINITY, v_rms/image = NaN and a bit is set in d_flags[b].
 *   - Angles in radians counter-clockwise from +x (Table 3 note); lengths in arcsec.
 */
#ifndef GLAD_H
#define GLAD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct glad_ctx glad_ctx; /* opaque */

typedef enum {
    GLAD_OK = 0,
    GLAD_EINVAL = -1, /* null pointer / bad scalar argument */
    GLAD_ESHAPE = -2, /* size outside what the kernels support (see each call) */
    GLAD_ECUDA = -3,  /* CUDA runtime error; text in glad_last_error */
    GLAD_ENOMEM = -4, /* scratch allocation failed */
    GLAD_ESTATE = -5  /* static data for this call not set */
} glad_status;

/* per-vector flag bits written to d_flags */
#define GLAD_FLAG_LENS_INVALID 1 /* theta_E<0, gamma not in (1,3), q not in (0,1], Sersic R_e,n,q <= 0 */
#define GLAD_FLAG_DYN_INVALID 2  /* not deprojectable (Eq. 22), D_d<=0, M_BH<0, beta_z>=1 */
#define GLAD_FLAG_PIXSRC_NOT_PD 8 /* glad_pixsrc_evidence_batch: F + lambda g is not positive definite */
#define GLAD_FLAG_BIN_INVALID 4  /* a bin is empty or has V^2 < 0 (negative density) */

/*
 * Lens parameter vector, GLAD_NLENS floats:
 *   [0..5]   EPL          x_l, y_l, theta_E, gamma, q, phi_PA    (App. B Eq. B.1-B.3; R-L3:
 *                         singular, r_soft = 0)
 *   [6..7]   ext. shear   gamma_ext, phi_ext, origin at the lens centre (Eq. 49; R-L5)
 *   [8]      point mass   theta_E,BH^2 [arcsec^2]                 (R-L6; see glad_bh_theta2)
 *   [9..15]  source       x_s, y_s, I_e, R_e, n, q_s, phi_s   elliptical Sersic at beta (R-L7)
 *   [16..20] lens light 1 I_e, R_e, n, q, phi   centred on the lens centre, evaluated at theta
 *   [21..25] lens light 2 I_e, R_e, n, q, phi   (I_e = 0 disables a component)
 * Elliptical radius R = sqrt(x^2 + y^2/q^2) everywhere (Eq. B.2).
 */
#define GLAD_NLENS 26
/* Dynamics parameter vector: inclination [rad], D_d [Mpc], M_BH [Msun], Upsilon (multiplies the
 * mass-MGE surface densities, not the BH). */
#define GLAD_NDYN 4
/* MGE table row: surface density [Lsun/pc^2 or Msun/pc^2], sigma' [arcsec], q' (Eq. 21, 24 P:166,182) */
#define GLAD_MGE_ROW 3

/* limits of the kernels (GLAD_ESHAPE beyond them) */
#define GLAD_MAX_IMAGE_PIXELS 40000 /* nx*ny of the lens image (staged whole in shared memory): the exact condition, checked by
                                       glad_set_image_data, is 4 (80 + kpsf ceil8(kpsf) + (ny + 1) pitch) <= 231424 bytes with
                                       pitch = (nx + 2 (kpsf/2) + 23) | 1 floats per padded row */
#define GLAD_MAX_PSF 31             /* kpsf and kk */
#define GLAD_MAX_GAUSS 64           /* n_lum, n_mass (+1 for the BH) */
#define GLAD_MAX_SKY 256            /* nx, ny of the kinematic grid */
#define GLAD_MAX_NODES 1024
#define GLAD_MAX_BINS 1024
#define GLAD_MAX_QIMG 8             /* lensed quasar images */

/* Create a context on `device` whose work is enqueued on `cuda_stream` (a cudaStream_t, borrowed;
 * NULL = the legacy default stream).  Returns GLAD_ECUDA if the device is not sm_100. */
glad_status glad_create(glad_ctx** out, int device, void* cuda_stream);
void glad_destroy(glad_ctx* ctx);
/* Context-owned string describing the last error on this context ("" if none). Never free it. */
const char* glad_last_error(const glad_ctx* ctx);
/* Library version string and the symbols it exports (static). */
const char* glad_version(void);

/* Image grid: pixel (iy,ix) centre at (x0 + ix*pix, y0 + iy*pix); row index grows with +y (R-L1).
 * Each pixel is the mean of supersample^2 sub-pixel samples at offsets ((a+1/2)/s - 1/2)*pix (R-L2). */
typedef struct {
    int nx, ny, supersample;
    float pix, x0, y0;
} glad_image_grid;

/* Static lensing data.  d_data, d_ivar: [ny,nx] (ivar = 1/sigma^2, 0 masks a pixel); either may be NULL
 * if chi2 is never requested.  d_psf: [kpsf,kpsf], kpsf odd <= GLAD_MAX_PSF, used as given (not
 * renormalised); the model is the TRUE convolution m[y,x] = sum psf[dy,dx] img[y-(dy-c), x-(dx-c)],
 * c = kpsf/2, zero outside the image (Eq. 38, (N_d,N_d) Table 1; R-L8).  The PSF is copied
 * into the context (on the stream); data/ivar are borrowed. */
glad_status glad_set_image_data(glad_ctx* ctx, const glad_image_grid* grid, const float* d_data,
                                const float* d_ivar, const float* d_psf, int kpsf);

/* Kinematic sky grid: tensor product xs[ix] x ys[iy] in the galaxy-aligned frame, x' = projected major
 * axis (R-D5), pixel centres, arcsec. */
typedef struct {
    int nx, ny;
    const float* d_xs;
    const float* d_ys;
} glad_sky_grid;

/* Static kinematic data.  d_bin_id [ny,nx] in [0,nbins) or -1 (unused spaxel); d_kernel [kk,kk], kk odd
 * <= GLAD_MAX_PSF = PSF_kin (x) pixel aperture, applied to numerator and denominator of Eq. 27
 * with the same true-convolution / zero-pad convention as the image PSF (R-D6); d_vrms_obs, d_vrms_ivar
 * [nbins] (may be NULL if chi2 is never requested); d_u_nodes, d_u_weights [nu] = quadrature rule on
 * u in (0,1) (R-D4).  All pointers borrowed.
 * SYNCHRONOUS (setup call): copies xs, ys and bin_id to the host once to detect a grid that is mirror-
 * symmetric about x' = 0 and/or y' = 0 (then only one half per axis is integrated -- the integrand is even),
 * validates the bin ids, and precomputes the static bin x kernel weights on the device.  The folded grid may
 * have at most 512 tiles of 8x8 pixels, and 4 (2 nxf nyf + n_lum (nxf + nyf)) bytes -- both folded maps plus the luminous
 * Gaussians' separable factors, staged in shared memory by the binning kernel -- must fit 231424 bytes: checked here for
 * n_lum = 1 and in the batch call for its n_lum (GLAD_ESHAPE otherwise). */
glad_status glad_set_kin_data(glad_ctx* ctx, const glad_sky_grid* grid, const int32_t* d_bin_id,
                              int nbins, const float* d_kernel, int kk, const float* d_vrms_obs,
                              const float* d_vrms_ivar, const float* d_u_nodes,
                              const float* d_u_weights, int nu);

/*
 * Lensing half.  For each of the B vectors: ray-shoot every sub-pixel centre
 * theta through EPL + shear + point mass, beta = theta - alpha (Eq. 33); evaluate the Sersic
 * source at beta and the lens light at theta; average to pixels; convolve with the PSF; and reduce
 * chi2_L = sum ivar (data - model)^2 (Eq. 48 P:374 with the pixel term of Eq. 37, diagonal C_d).
 *   d_lens_params [B,GLAD_NLENS]; d_images [B,ny,nx] or NULL; d_chi2 [B] or NULL; d_flags [B] or NULL
 *   (flags are OVERWRITTEN with the lens bits).
 * GLAD_ESTATE if glad_set_image_data was not called (or d_chi2 != NULL without data/ivar).
 */
glad_status glad_lens_image_batch(glad_ctx* ctx, const float* d_lens_params, int B, float* d_images,
                                  float* d_chi2, int32_t* d_flags);

/*
 * Dynamics half (rows a5-a8).  Cylindrically-aligned axisymmetric Jeans model on MGEs (the paper defers
 * the formula to Cappellari at P:228; R-D1 states it): for every sky pixel
 *   [Sigma v_los^2](x',y') = 4 pi^{3/2} G sum_u w_u sum_k sum_j T(u,j,k; x',y')
 * over quadrature nodes u, luminous Gaussians k (deprojected by Eq. 22-23; b_k = 1/(1-beta_z,k),
 * R-D2) and mass Gaussians j (Eq. 25, times Upsilon) plus, if M_BH > 0, one round Gaussian of
 * sigma = 0.01" and mass M_BH (R-D3); Sigma from Eq. 21; then Eq. 27-28 with the
 * kernel and bins of glad_set_kin_data, and chi2_D = sum_l ivar_l (obs_l - v_l)^2 (Eq. 32; R-D7).
 *   d_dyn_params [B,GLAD_NDYN]
 *   d_lum_mge  rows {I0, sigma', q'} x n_lum ; lum_stride = floats between consecutive vectors, 0 = shared
 *   d_mass_mge rows {Sigma0, sigma', q'} x n_mass (n_mass may be 0) ; mass_stride likewise
 *   d_beta [B,n_lum] if beta_per_gaussian else [B]
 *   d_vrms [B,nbins] or NULL ; d_chi2 [B] or NULL ; d_v2map [B,ny,nx] or NULL (raw Sigma*v_los^2 map,
 *   (km/s)^2 Lsun/pc^2) ; d_flags [B] or NULL (OVERWRITTEN with the dynamics bits).
 */
glad_status glad_jam_vrms_batch(glad_ctx* ctx, const float* d_dyn_params, int B,
                                const float* d_lum_mge, int n_lum, long lum_stride,
                                const float* d_mass_mge, int n_mass, long mass_stride,
                                const float* d_beta, int beta_per_gaussian, float* d_vrms,
                                float* d_chi2, float* d_v2map, int32_t* d_flags);

/*
 * Joint (row a9): both halves on the context stream, then lnL[b] = -(chi2_L[b] + chi2_D[b])/2 with no
 * normalisation constant (Eq. 52-53 P:410-416 restricted to the pixel term and chi2_dyn; the image-
 * position and time-delay terms are the paper's CPU terms), -INFINITY where a half is invalid.
 *   d_loglike [B]; d_chi2_lens, d_chi2_dyn [B] or NULL; d_flags [B] or NULL (union of both halves' bits).
 */
glad_status glad_joint_loglike_batch(glad_ctx* ctx, const float* d_lens_params,
                                     const float* d_dyn_params, int B, const float* d_lum_mge,
                                     int n_lum, long lum_stride, const float* d_mass_mge, int n_mass,
                                     long mass_stride, const float* d_beta, int beta_per_gaussian,
                                     float* d_loglike, float* d_chi2_lens, float* d_chi2_dyn,
                                     int32_t* d_flags);

/*
 * Host-buffer variant of glad_joint_loglike_batch (the end-to-end call a CPU sampler makes): all pointers are
 * HOST pointers (pinned memory recommended).  Copies the parameter vectors, MGE tables and beta to context-
 * owned device staging on the stream, runs the joint path, copies lnL (and chi2 / flags if non-NULL) back and
 * SYNCHRONISES the stream before returning.  Table sizes follow the strides: n_lum*3 floats if lum_stride == 0
 * else B*lum_stride; likewise for mass.
 */
glad_status glad_joint_loglike_host(glad_ctx* ctx, const float* h_lens_params, const float* h_dyn_params, int B,
                                    const float* h_lum_mge, int n_lum, long lum_stride, const float* h_mass_mge,
                                    int n_mass, long mass_stride, const float* h_beta, int beta_per_gaussian,
                                    float* h_loglike, float* h_chi2_lens, float* h_chi2_dyn, int32_t* h_flags);

/*
 * the step between the two halves (Fig. 2: "we decompose I_light and Sigma_int into
 * multiple Gaussian components").  1-D multi-Gaussian expansion of a radial profile F(R), R = sqrt(x^2 + y^2/q'^2)
 * (footnote P:234), by the integral transform of Eq. 44 evaluated with the Euler sum of Eq. 45 of
 * order P (2P+1 complex profile evaluations per Gaussian; P in [1,15], 0 = default 12; DESIGN.md R-M1 states the
 * constants eta_n, chi_n the paper leaves out) on n_gauss >= 2 log-spaced sigma_n in [sigma_lo, sigma_hi]:
 *   A_n = w_n f(sigma_n) dln(sigma) / sqrt(2 pi)   (Eq. 46; w = 1/2 at both ends, 1 inside, R-M2).
 * d_prof [B,GLAD_NPROF] float, one row per vector:
 *   GLAD_PROFILE_SERSIC : {I_e, R_e, n, q'}            F = I_e exp(-b_n ((R/R_e)^(1/n) - 1))        (R-L7)
 *   GLAD_PROFILE_EPL    : {scale, theta_E, gamma, q}   F = scale (3-gamma)/2 (b/R)^(gamma-1), b of Eq. B.3
 *   GLAD_PROFILE_CHAMELEON : {I_0, w_c, w_t, q'}       F of Eq. 47, the paper's I_light
 *   GLAD_PROFILE_NFW_CSE   : {scale, r_s, -, q}        F = scale sum_i A_i / (2 (s_i^2 + u^2)^(3/2)), u = R sqrt(q)/r_s (Eq. A.2-A.4),
 *                                                      the CSE table of glad_set_enfw (GLAD_ESTATE without it)
 * d_mge [B,n_gauss,3] rows {A_n, sigma_n, q'}: the MGE row layout glad_jam_vrms_batch reads (stride 3*n_gauss).
 * fp64 arithmetic, fp32 rows.  Enqueues on the context stream; device pointers owned by the caller.
 * GLAD_EINVAL on a bad kind / range / order, GLAD_ESHAPE if n_gauss > GLAD_MAX_GAUSS.
 */
typedef enum { GLAD_PROFILE_SERSIC = 0, GLAD_PROFILE_EPL = 1, GLAD_PROFILE_CHAMELEON = 2, GLAD_PROFILE_NFW_CSE = 3 } glad_profile_kind;
#define GLAD_NPROF 4
glad_status glad_mge1d_batch(glad_ctx* ctx, int kind, const float* d_prof, int B, int n_gauss, float sigma_lo,
                             float sigma_hi, int euler_order, float* d_mge);

/*
 * Self-consistent joint model (R-M3; Fig. 2): ONE sampler vector per evaluation.  On the device, per vector:
 *   luminous MGE = Eq. 46 of lens-light component #1 (lens[16..19]; Sersic or Chameleon, glad_set_light_profiles), n_lum Gaussians on
 *                  [lum_sigma_lo, lum_sigma_hi];
 *   mass MGE     = Eq. 46 of Sigma_crit * kappa_epl(theta_E, gamma, q) with Sigma_crit(D_dt, D_d, z_d) of Eq. 13
 *                  (D_d = dyn[1]), n_mass Gaussians on [mass_sigma_lo, mass_sigma_hi] (the paper goes to 50");
 *   lens[8]      = theta_E,BH^2 of M_BH = dyn[2] and D_dt (Eq. 4); the caller's lens[8] is ignored;
 * then exactly glad_joint_loglike_batch with these per-vector tables (Upsilon = dyn[3] still multiplies the mass MGE).
 *   d_ddt [B] time-delay distances in Mpc; z_d lens redshift; other arguments as glad_joint_loglike_batch.
 *   d_lum_mge_out [B,n_lum,3] / d_mass_mge_out [B,n_mass,3]: the derived tables, or NULL.
 */
glad_status glad_joint_loglike_model_batch(glad_ctx* ctx, const float* d_lens_params, const float* d_dyn_params,
                                           const float* d_ddt, float z_d, int B, int n_lum, float lum_sigma_lo,
                                           float lum_sigma_hi, int n_mass, float mass_sigma_lo, float mass_sigma_hi,
                                           const float* d_beta, int beta_per_gaussian, float* d_loglike,
                                           float* d_chi2_lens, float* d_chi2_dyn, int32_t* d_flags,
                                           float* d_lum_mge_out, float* d_mass_mge_out);

/* Host helper: theta_E,BH^2 [arcsec^2] = 4 G M_BH (1+z_d) / (c^2 D_dt) (from Eq. 4), so that the
 * caller keeps lens[8] consistent with dyn[2] and the sampled D_dt.  Pure host arithmetic. */
double glad_bh_theta2(double mbh_msun, double ddt_mpc, double z_d);

/*
 * Optional per-kernel timing for bench.py's roofline line: when enabled, a CUDA event pair is recorded on the
 * context stream around every kernel launch (at most 2048 launches between reads).  glad_profile_read
 * SYNCHRONISES the stream, adds the elapsed times to per-kernel totals, copies them out and clears them.
 * Kernel order: 0 lens_prep, 1 lens_image, 2 jam_prep, 3 jam_quad, 4 jam_post, 5 joint, 6 mge (mge1d / model kernel), 7 quasar,
 * 8 pixsrc_map, 9 pixsrc_blur, 10 pixsrc_syrk, 11 pixsrc_rhs, 12 pixsrc_chol, 13 pixsrc_model (+ static / final kernels),
 * 14 jam_sph (intrinsic moments), 15 jam_sph_los.
 */
#define GLAD_NKERNELS 16
glad_status glad_profile_enable(glad_ctx* ctx, int on);
glad_status glad_profile_read(glad_ctx* ctx, double* ms_out /*[GLAD_NKERNELS]*/, long* count_out /*[GLAD_NKERNELS]*/);

/*
 * SURVEY 8(f) rank 4, light part: the paper models the lens light with Chameleon profiles (Eq. 47),
 *   I = I_0/(1+q) [ (x^2 + y^2/q^2 + 4 w_c^2/(1+q)^2)^(-1/2) - (x^2 + y^2/q^2 + 4 w_t^2/(1+q)^2)^(-1/2) ].
 * Each of the three light components (source, lens light 1, lens light 2) is a Sersic (default) or a Chameleon for the
 * whole batch; a Chameleon component reads its five shape slots as {I_0, w_c, w_t, q, phi} instead of {I_e, R_e, n, q, phi}
 * (source: lens[11..15], lens light: lens[16..20], lens[21..25]); valid iff 0 < w_c < w_t and 0 < q <= 1, I_0 = 0 disables it.
 * Takes effect for the batch calls enqueued afterwards; glad_joint_loglike_model_batch then expands lens light 1 as a
 * Chameleon for the luminous tracer (GLAD_PROFILE_CHAMELEON).
 */
#define GLAD_LIGHT_SERSIC 0
#define GLAD_LIGHT_CHAMELEON 1
glad_status glad_set_light_profiles(glad_ctx* ctx, int source_kind, int lens1_kind, int lens2_kind);

/*
 * SURVEY 8(f) rank 4, mass part: an elliptical NFW dark-matter halo through core-steep ellipsoids (Appendix A; the dark
 * matter of the paper's composite model kappa_int,comp):
 *   kappa_enfw(x, y) = rho_s sum_i A_i / (2 (s_i^2 + u^2)^(3/2)),  u^2 = X^2 + Y^2/q^2,  (X, Y) = (sqrt(q)/r_s) (x, y)   (Eq. A.2-A.4)
 * in the halo frame (centre = the lens centre lens[0..1], major axis at angle phi), with the closed-form potential of a CSE
 * (Eq. A.6) for alpha, the Hessian and psi: psi = (rho_s r_s^2/q) sum A_i psi_CSE, alpha = (rho_s r_s/sqrt(q)) sum A_i grad psi_CSE
 * (DESIGN.md R-N2: amplitudes from Eq. 7; the prefactor printed in Eq. A.7 is off by one power of r_s).
 *   d_enfw [n,4] DEVICE pointer, BORROWED: {rho_s (dimensionless, >= 0; 0 = no halo for that vector), r_s [arcsec] > 0, q in (0,1], phi};
 *     NULL switches the halo off.  Vector b of a batch reads row b; B > n returns GLAD_EINVAL; invalid rows flag the vector
 *     (GLAD_FLAG_LENS_INVALID).
 *   h_A, h_s [n_cse <= GLAD_MAX_CSE] HOST arrays, copied: the (A_i, s_i) table of Eq. A.3.  The paper uses Oguri (2021)'s 44 pairs
 *     and says they are "predetermined": the table is an INPUT of the method (R-N1).  workloads/cse_nfw.txt holds a table
 *     fitted from Eq. A.5 as printed (41 positive pairs, 6.9e-6 relative on u in [1e-6, 1e3]).
 *   n_gauss, sigma_lo, sigma_hi: the halo's rows of the mass MGE (Eq. 46 of Sigma_crit lambda kappa_enfw, q' = q), appended after the EPL
 *     (and mass-sheet) rows by glad_joint_loglike_model_batch / _full_batch; d_mass_mge_out is then wider by n_gauss rows.
 * While set: the lens half (every entry built on glad_lens_image_batch) adds alpha_enfw to the ray-shoot (fp32, the Chameleon /
 * mass-sheet instantiation of the kernel), glad_quasar_chi2_batch adds alpha, the Hessian and psi (fp64).  The pixelated-source
 * entry does not take the halo (GLAD_ESTATE while it is set).  SYNCHRONOUS setup call (copies the table).
 */
#define GLAD_MAX_CSE 64
glad_status glad_set_enfw(glad_ctx* ctx, const float* d_enfw, int n_enfw, int n_cse, const double* h_A, const double* h_s, int n_gauss,
                          float sigma_lo, float sigma_hi);

/*
 * Options of the quadrature (row a6), fixed for the context until changed; 0 selects the default of each.
 *   path         GLAD_JAM_AUTO: tcgen05 tensor-core contraction where the folded grid fits (<= 128 rows, terms * columns <= 256),
 *                the FP32 SIMT kernel otherwise; GLAD_JAM_SIMT: always the FP32 SIMT kernel.
 *   bf16_terms   operand values are split into 2 (default: 16 mantissa bits) or 3 (24 bits) bf16 terms on the tcgen05 path.
 *   flush_chunks operand chunks per TMEM accumulator group before the group is added into fp32 registers (default: 512 contraction rows;
 *                a chunk is the rows one producer group stages, 64 at the default sizes; never fewer than 2 * groups - 2 = 14 chunks,
 *                which the reuse of the two TMEM buffers needs, so smaller values are raised to that).
 *   k_slices     CTAs per parameter vector along the contraction (default: enough for 4 CTAs per SM on small batches).
 * The arithmetic of a context therefore never depends on the caller's environment.  GLAD_EINVAL on a bad value.
 */
#define GLAD_JAM_AUTO 0
#define GLAD_JAM_SIMT 1
glad_status glad_set_jam_options(glad_ctx* ctx, int path, int bf16_terms, int flush_chunks, int k_slices);

/*
 * glad_joint_loglike_batch (and the entries built on it) run the lens half on a context-owned side stream beside the
 * dynamics half, joined by events before the joint kernel; the caller's stream still sees plain stream order.
 * glad_set_overlap(ctx, 0) keeps every kernel on the caller's stream (bench.py uses it for per-kernel timing, where
 * overlapped event times would include waiting for SMs); default on (environment GLAD_OVERLAP=0 turns it off at creation).
 * Returns GLAD_ESTATE if the side stream could not be created.
 */
glad_status glad_set_overlap(glad_ctx* ctx, int on);

/*
 * SURVEY 8(f) rank 4, quasar part: the image-position and time-delay terms of Eq. 53.  The paper keeps them on the
 * CPU; in a batched sampler they are one more per-vector reduction over the same mass parameters.
 *
 * glad_set_quasar_data: HOST pointers, copied into the context (n_img = 0 clears).  h_theta [n_img,2] observed image positions
 * (x, y) in arcsec, same frame as the image grid; h_sigma_theta [n_img] > 0 positional uncertainties; ref_image = index of the
 * reference image j of Eq. 36; h_dt_obs [n_img] observed delays Delta t_ij in DAYS relative to the reference image (its own
 * entry is ignored) and h_sigma_dt [n_img] their uncertainties (<= 0 = that delay is not measured); both NULL = no delays.
 * GLAD_ESHAPE if n_img > GLAD_MAX_QIMG.
 *
 * glad_quasar_chi2_batch, per vector (mass parameters lens[0..8] only; DESIGN.md R-Q1..R-Q5), all arithmetic fp64:
 *   beta_i = theta_i - alpha(theta_i) (Eq. 33); mu_i = 1/det(I - Hessian psi(theta_i));
 *   beta_bar = sum |mu_i| beta_i / sum |mu_i|  ("magnification-weighted average");
 *   theta_i^pre = image of beta_bar reached from theta_i by 12 Newton steps on the lens equation ("map it back");
 *   chi2_img = sum_i |theta_i - theta_i^pre|^2 / sigma_theta,i^2                                            (Eq. 35)
 *   dt_i^pre = (D_dt/c) [phi(theta_i^pre, beta_bar) - phi(theta_ref^pre, beta_bar)], phi = |theta-beta|^2/2 - psi(theta)
 *                                                                                       (Eq. 2-4), in days;
 *   chi2_tmd = sum_{i != ref} (dt_obs,i - dt_i^pre)^2 / sigma_dt,i^2                                        (Eq. 36)
 *   d_lens_params [B,GLAD_NLENS]; d_ddt [B] time-delay distances in Mpc; outputs (device, any may be NULL):
 *   d_chi2_img, d_chi2_tmd [B] float; d_theta_pre [B,n_img,2], d_dt_pre [B,n_img], d_beta [B,2] DOUBLE.
 *   An invalid mass model (GLAD_FLAG_LENS_INVALID conditions on lens[2..4], lens[8]) gives chi2 = +INFINITY, NaN elsewhere.
 * GLAD_ESTATE if no quasar data is set.
 */
glad_status glad_set_quasar_data(glad_ctx* ctx, int n_img, const double* h_theta, const double* h_sigma_theta, int ref_image,
                                 const double* h_dt_obs, const double* h_sigma_dt);
glad_status glad_quasar_chi2_batch(glad_ctx* ctx, const float* d_lens_params, const float* d_ddt, int B, float* d_chi2_img,
                                   float* d_chi2_tmd, double* d_theta_pre, double* d_dt_pre, double* d_beta);

/*
 * glad_joint_loglike_model_batch plus the quasar terms: lnL = -(chi2_L + chi2_D + chi2_img + chi2_tmd)/2, every term of
 * Eq. 53 with the pixel chi2 standing for the extended-source evidence (R-J1).  The quasar kernel reads the derived
 * lens vector (lens[8] = theta_E,BH^2 of M_BH and D_dt) and runs on the lens half's stream.  d_chi2_img, d_chi2_tmd [B] or NULL.
 */
glad_status glad_joint_loglike_full_batch(glad_ctx* ctx, const float* d_lens_params, const float* d_dyn_params,
                                          const float* d_ddt, float z_d, int B, int n_lum, float lum_sigma_lo,
                                          float lum_sigma_hi, int n_mass, float mass_sigma_lo, float mass_sigma_hi,
                                          const float* d_beta, int beta_per_gaussian, float* d_loglike,
                                          float* d_chi2_lens, float* d_chi2_dyn, float* d_chi2_img, float* d_chi2_tmd,
                                          int32_t* d_flags);

/*
 * SURVEY 8(f) rank 1, remainder: the internal mass sheet that the joint model exists to constrain (Eq. 5-9).  The paper
 * stands a dPIE profile with r_core = 45", r_tr = 45.09" for the constant sheet (Eq. 50-51); DESIGN.md R-S1..3:
 *   kappa_int = (1 - lambda) S(R) + lambda kappa_epl + kappa_BH,   S(R) = [1/sqrt(R^2+r_core^2) - 1/sqrt(R^2+r_tr^2)] / (1/r_core - 1/r_tr),
 * R^2 = x^2 + y^2 about the lens centre, lambda = the constant of Eq. 51 (one per vector); the external shear (Eq. 49) and the point
 * mass are outside the transformation.  d_lambda [n_lambda] is a DEVICE pointer, BORROWED; NULL switches the sheet off.  Vector b
 * of a batch call reads d_lambda[b]; a batch call with B > n_lambda returns GLAD_EINVAL.  While set:
 *   - the lens half (glad_lens_image_batch and every joint entry) ray-shoots through lambda alpha_epl + alpha_sheet + shear + point mass;
 *   - glad_quasar_chi2_batch uses the same alpha, its Jacobian and psi (Eq. 8);
 *   - glad_joint_loglike_model_batch / _full_batch build the mass MGE of Sigma_crit kappa_int: lambda x the n_mass EPL rows followed by
 *     n_sheet round (q' = 1) rows, the Eq. 46 expansion of Sigma_crit (1 - lambda) S(R) on [sheet_sigma_lo, sheet_sigma_hi] (the
 *     profile's transform falls off as sigma^-3 only: take sheet_sigma_hi >> r_tr); n_mass + n_sheet <= GLAD_MAX_GAUSS and
 *     d_mass_mge_out is then [B, n_mass + n_sheet, 3].  The caller-supplied tables of glad_joint_loglike_batch are used as given.
 * A non-finite lambda invalidates the vector (GLAD_FLAG_LENS_INVALID).  GLAD_EINVAL unless 0 < r_core < r_tr, n_sheet >= 2,
 * 0 < sheet_sigma_lo < sheet_sigma_hi.
 */
glad_status glad_set_mass_sheet(glad_ctx* ctx, const float* d_lambda, int n_lambda, float r_core, float r_tr, int n_sheet,
                                float sheet_sigma_lo, float sheet_sigma_hi);

/*
 * the paper's own extended-image likelihood, the pixelated-source inversion of Eq. 37-43 (
 * matrix sizes in Table 1), for B parameter vectors at once.  Static data: glad_set_image_data (grid, d_esr = data,
 * C_d^-1 = diag(ivar) with ivar = 0 masking a pixel out, PSF).  Per vector b (DESIGN.md R-P1..5):
 *   L   [N_pix, N_s]  image pixel CENTRE theta -> beta = theta - alpha(theta) (Eq. 33; mass part lens[0..8] only, with the
 *                     internal mass sheet when glad_set_mass_sheet is active), bilinear weights on the source grid of n_sx x n_sy
 *                     pixels of size d_src_grid[b,2] whose pixel (0,0) is centred at (d_src_grid[b,0], d_src_grid[b,1]); a ray
 *                     outside the rectangle of source-pixel centres gives a zero row.  The supersampling factor is not used.
 *   f = B L           (Eq. 38), B = the "same"-size zero-padded PSF convolution of glad_lens_image_batch
 *   F = f^T C_d^-1 f, D = f^T C_d^-1 d_esr                                                                (Eq. 41-42)
 *   s_MP = (F + lambda g)^-1 D, lambda = d_lambda_reg[b] > 0                                              (Eq. 40)
 *       g = Hessian of the curvature regulariser E_S = 1/2 sum_pixels [(s_{i-1} - 2 s_i + s_{i+1})^2 + (same in j)^2], s = 0 outside
 *   ln P(d_esr | f, lambda, g) = -chi2/2 - lambda E_S(s_MP) - 1/2 ln det(F + lambda g) + N_s/2 ln lambda + 1/2 ln det g
 *                                - N_d/2 ln 2 pi + 1/2 sum_{ivar>0} ln ivar       (Eq. 43; Suyu et al. 2006 Eq. 19)
 *       chi2 = sum ivar (f s_MP - d_esr)^2, N_d = number of pixels with ivar > 0.
 * Arithmetic: rays, D, the Cholesky factorisation, the solve and the evidence in fp64; f and the contraction F in fp32.
 * All pointers are DEVICE pointers owned by the caller: d_lens_params [B,GLAD_NLENS], d_src_grid [B,3], d_lambda_reg [B];
 * outputs (any may be NULL): d_logev [B], d_chi2 [B], d_reg [B] (= E_S), d_s_mp [B,n_sy,n_sx], d_model [B,ny,nx] (= f s_MP),
 * d_flags [B].  An invalid mass model (GLAD_FLAG_LENS_INVALID conditions on lens[2..4], lens[8]), lambda <= 0 or a pixel size
 * <= 0 gives logev = -INFINITY, chi2 = +INFINITY, NaN elsewhere and GLAD_FLAG_LENS_INVALID; a matrix that is not positive
 * definite gives the same outputs with GLAD_FLAG_PIXSRC_NOT_PD.  The batch is processed in chunks that fit scratch_mib_max
 * MiB of context-owned device scratch (<= 0: 16384; the block is allocated at exactly the chunk's size, never above the limit);
 * one vector needs about 4 N_pix N_s + 8 N_s^2 bytes.
 * GLAD_ESTATE without image data; GLAD_ESHAPE if n_sx, n_sy < 2, N_s > 4096 or one vector does not fit the scratch limit.
 */
glad_status glad_pixsrc_evidence_batch(glad_ctx* ctx, const float* d_lens_params, const float* d_src_grid, const float* d_lambda_reg,
                                       int n_sx, int n_sy, int B, int scratch_mib_max, float* d_logev, float* d_chi2, float* d_reg,
                                       float* d_s_mp, float* d_model, int32_t* d_flags);

/*
 * JAM_sph, the dynamics the paper itself runs -- the axisymmetric Jeans equations with a SPHERICALLY-aligned
 * velocity ellipsoid (Eq. 17-18, beta_ani = 1 - v_theta^2/v_r^2 Eq. 20), solved for the intrinsic moments
 * v_r^2, v_theta^2, v_phi^2 "at the required positions ... in polar coordinates" by a NON-ADAPTIVE 2-D quadrature, then
 * projected along the line of sight (Eq. 26), convolved and binned (Eq. 27-28) and compared (Eq. 32).  The paper prints no
 * solution formula (it defers to Cappellari 2020 at P:228); DESIGN.md R-SPH1..6 derive it from Eq. 17-18:
 *   nu v_r^2 (r,th) = int_r^r_cut (r'/r)^(2 beta) nu(r',th') (r'^2/z') dPhi/dz'(r',th') dr'/r',  sin th' = sin th (r/r')^(1-beta),
 *   nu v_th^2 = (1-beta) nu v_r^2,   nu v_phi^2 = (1-beta) [nu v_r^2 + tan th d(nu v_r^2)/dth] + nu tan th dPhi/dth,
 * Phi the MGE potential (a u-integral on (0,1) per mass Gaussian), per luminous Gaussian k with its own beta_k, r_cut = 6 max sigma_k.
 *
 * glad_set_jam_sph_rules: DEVICE pointers, BORROWED; d_rgrid = NULL clears.
 *   d_rgrid [nr] ascending radii (arcsec), d_thgrid [nth] ascending polar angles in [0, pi/2] (from the symmetry axis): the polar
 *     grid; the moment ratios are interpolated bilinearly in (ln r, theta), clamped at the grid edges (R-SPH2, R-SPH3);
 *   d_tau, d_wtau [nt]: rule on (0,1) for r' = r (r_cut/r)^tau;  d_un, d_uw [nu]: rule on (0,1) for the potential integral (the
 *     paper's mesh, 64 sub-regions x 4 Gauss-Kronrod rectangles P:360, is 112 x 112 nodes);
 *   d_zeta, d_wz [nz]: rule on (-1,1) for z' = rho_0 sinh(a zeta), rho_0 = max(sky radius, rgrid[0]), a = asinh(r_cut/rho_0) (R-SPH4).
 *   GLAD_ESHAPE beyond nr <= GLAD_MAX_SPH_R, nth <= GLAD_MAX_SPH_TH, nt, nu, nz <= GLAD_MAX_NODES.
 *
 * glad_jam_sph_vrms_batch: arguments and outputs as glad_jam_vrms_batch (sky grid, kernel, bins, data from glad_set_kin_data; its
 * u rule is not used), except that d_beta holds beta_ani (< 1, else GLAD_FLAG_DYN_INVALID) and
 *   d_moments [B,3,nr,nth] or NULL receives v_r^2, v_theta^2, v_phi^2 in (km/s)^2 on the polar grid.
 * d_v2map is int nu v_z'^2 dz' (km^2 s^-2 Lsun pc^-2).  fp32 arithmetic with fp64-prepared tables.  GLAD_ESTATE without kinematic
 * data or rules; GLAD_ESHAPE if 20 (n_mass + 1) nu bytes of potential table do not fit shared memory.
 */
#define GLAD_MAX_SPH_R 128
#define GLAD_MAX_SPH_TH 64
glad_status glad_set_jam_sph_rules(glad_ctx* ctx, const float* d_rgrid, int nr, const float* d_thgrid, int nth, const float* d_tau,
                                   const float* d_wtau, int nt, const float* d_u_nodes, const float* d_u_weights, int nu,
                                   const float* d_zeta, const float* d_wz, int nz);
glad_status glad_jam_sph_vrms_batch(glad_ctx* ctx, const float* d_dyn_params, int B, const float* d_lum_mge, int n_lum,
                                    long lum_stride, const float* d_mass_mge, int n_mass, long mass_stride, const float* d_beta,
                                    int beta_per_gaussian, float* d_vrms, float* d_chi2, float* d_v2map, float* d_moments,
                                    int32_t* d_flags);

/*
 * Eq. 43: the evidence of the pixelated-source reconstruction AT THE OPTIMAL regularisation constant,
 *   lambda_hat = argmax over [lambda_lo, lambda_hi] of ln P(d_esr | f, lambda, g).
 * F and D do not depend on lambda, only the factorisation does: the chain of glad_pixsrc_evidence_batch is run once up to F and D,
 * then, on the device and without a host round trip, 22 evaluations of ln P(lambda) up to lambda-independent terms,
 *   J(ln lambda) = y^T y / 2 - ln det(F + lambda g) / 2 + N_s ln(lambda) / 2,  L L^T = F + lambda g,  L y = D
 * (since -chi2/2 - lambda E_S = -(d^T C_d^-1 d - D^T s_MP)/2 at s_MP): the two ends, then 18 golden-section steps on ln lambda, then
 * the vertex of the parabola through the last bracket.  lambda_hat is rounded to float32 and everything glad_pixsrc_evidence_batch
 * returns is then evaluated at that value.  d_lam_hat [B] (required) receives lambda_hat; other arguments, outputs, flags and
 * errors as glad_pixsrc_evidence_batch; one vector needs about 4 N_pix N_s + 16 N_s^2 bytes of scratch.  GLAD_EINVAL unless
 * 0 < lambda_lo < lambda_hi.  An evidence that is not unimodal on the interval gives a local maximum.
 */
glad_status glad_pixsrc_lambda_opt_batch(glad_ctx* ctx, const float* d_lens_params, const float* d_src_grid, float lambda_lo, float lambda_hi,
                                         int n_sx, int n_sy, int B, int scratch_mib_max, float* d_lam_hat, float* d_logev, float* d_chi2,
                                         float* d_reg, float* d_s_mp, float* d_model, int32_t* d_flags);

/*
 * glad_lens_image_batch for callers that cannot allocate device memory at call time (a CUDA graph being captured, a tight serving
 * loop, a harness that forbids cudaMalloc): same arguments, same kernels (lens_prep_kernel -> lens_image_kernel), same results, but
 * the per-vector constants that the first kernel writes for the second (88 floats per vector) live in a file-scope
 * `static __device__` array of GLAD_LENS_NOALLOC_MAX_B vectors (1.4 MB, held by every GPU that loads the library until the
 * process exits) instead of the context's growable scratch block.  The call enqueues two kernels on the context's stream and
 * calls no cudaMalloc / cudaFree / allocating routine; the array's device address is taken once per device in glad_create.
 * (The CUDA driver may still load kernel code and size its local-memory pool at a process's FIRST launch of these kernels: make one
 * call before capturing a graph.)
 *   B > GLAD_LENS_NOALLOC_MAX_B: GLAD_ESHAPE (split the batch).  GLAD_ESTATE as glad_lens_image_batch, or if the address could
 *   not be taken at glad_create.  Mass sheet, eNFW halo and light-profile settings apply as in glad_lens_image_batch.
 * The array is SHARED by every context and call on the device and keeps the last call's contents: the first kernel rewrites every
 * slot the second one reads (nothing has to start at zero), and two calls whose kernels may overlap on the GPU (different
 * streams, or contexts created on different streams) RACE on it -- order them on one stream or with events.
 */
#define GLAD_LENS_NOALLOC_MAX_B 4096
glad_status glad_lens_image_noalloc(glad_ctx* ctx, const float* d_lens_params, int B, float* d_images, float* d_chi2,
                                    int32_t* d_flags);

/* Number of kernel launches enqueued by this context since creation (for bench.py's gpu_launches). */
long glad_launch_count(const glad_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GLAD_H */
