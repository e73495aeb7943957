// Internal declarations shared by the .cu files of libglad (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "glad.h"

// ---------------------------------------------------------------------------------------------
// Lens half: per-vector constants prepared in fp64 by lens_prep_kernel (row a0), read by
// lens_image_kernel.  Indices into a float[LC_SIZE] block.
// ---------------------------------------------------------------------------------------------
#define GLAD_EPL_MAX_TERMS 40     // series coefficients stored per vector (enough for q >= 0.2 at 2e-8)
#define GLAD_EPL_TERMS_CAP 500    // terms summed at most (DESIGN.md R-L3): coefficients past the table are formed on the fly
enum LensConstIdx {
    LC_XL = 0, LC_YL, LC_COSPA, LC_SINPA, LC_Q, LC_NEGF,  // -f = -(1-q)/(1+q)
    LC_PREF,      // 2 b_TM^t / (1+q)   (0 if theta_E = 0)
    LC_HEXP,      // -(t-1)/2 : alpha magnitude = PREF * (R_TM^2)^HEXP
    LC_NTERMS,    // number of series terms (int stored as float)
    LC_SH_C, LC_SH_S,  // gamma_ext cos 2phi_ext, gamma_ext sin 2phi_ext
    LC_BH,        // theta_E,BH^2
    LC_VALID,     // 1 valid / 0 invalid
    LC_MS_AMP,    // internal mass sheet: (1 - lambda) 2 r_core r_tr (0 = no sheet); LC_PREF then carries lambda
    LC_MS_RC, LC_MS_RT,
    LC_SERSIC0 = 16,   // 3 components x 8 floats: xc, yc, cos, sin, 1/q^2, amp = Ie e^bn, k1 = bn log2e Re^(-1/n), h = 1/(2n)
    LC_SERIES = 40,    // c_n, n = 1..GLAD_EPL_MAX_TERMS : (2n-(2-t))/(2n+(2-t))
    LC_NF_AMP = 80,    // eNFW halo (glad_set_enfw): rho_s r_s / sqrt(q), 0 = no halo
    LC_NF_SC,          // sqrt(q) / r_s
    LC_NF_Q, LC_NF_COS, LC_NF_SIN,
    LC_SIZE = 88
};
#define LC_SERSIC_STRIDE 8

// ---------------------------------------------------------------------------------------------
// Dynamics half: per-vector table block prepared in fp64 by jam_prep_kernel (rows a0/a5).
// Layout (floats): header[JT_HDR] | 8 x nl (per luminous Gaussian) | 3 x nmx (per mass Gaussian,
// nmx = n_mass+1 slots, the last for the BH) | 2 x nmx*nl (per pair), padded to a multiple of 4.
// ---------------------------------------------------------------------------------------------
#define JT_HDR 8
enum JamHdrIdx { JH_SCALE = 0, JH_COS2I, JH_SIN2I, JH_NM, JH_VALID };
enum JamLumIdx { JL_INVS2 = 0, JL_BKQ, JL_S0, JL_D0, JL_NKS, JL_I0, JL_E1, JL_E2, JL_COUNT };
enum JamMassIdx { JM_INVS2 = 0, JM_OMQ2, JM_MJ, JM_COUNT };

static inline __host__ __device__ int jam_table_floats(int nl, int nmx) {
    int n = JT_HDR + JL_COUNT * nl + JM_COUNT * nmx + 2 * nmx * nl;
    return (n + 3) & ~3;
}

// Thread tile of the quadrature contraction (outputs per thread = JQ_T x JQ_T) and rows of the
// contraction each thread group consumes per staged chunk.
#define JQ_T 8
#define JQ_MI 8

#define GLAD_PROF_MAX 2048
enum GladKernelId { GK_LENS_PREP = 0, GK_LENS_IMAGE, GK_JAM_PREP, GK_JAM_QUAD, GK_JAM_POST, GK_JOINT, GK_MGE, GK_QUASAR,
                    GK_PIX_MAP, GK_PIX_BLUR, GK_PIX_SYRK, GK_PIX_RHS, GK_PIX_CHOL, GK_PIX_MODEL, GK_JAM_SPH, GK_JAM_SPH_LOS };

// eNFW halo (glad_set_enfw), passed to the kernels by value: per-vector {rho_s, r_s, q, phi} rows and the CSE table (A_i, s_i)
struct HaloArgs {
    const float* nf;         // [B,4] or NULL = no halo
    const double2* cse64;    // [ncse] for the fp64 kernels
    const float2* cse32;     // [ncse] {A_i / s_i, s_i} for the fp32 ray-shoot
    int ncse;
};

// quasar data (glad_set_quasar_data), passed to quasar_kernel by value
struct glad_quasar_data {
    int n_img, ref;
    double theta[2 * GLAD_MAX_QIMG];     // observed image positions (x, y), arcsec
    double ivar_theta[GLAD_MAX_QIMG];    // 1 / sigma_theta^2
    double dt_obs[GLAD_MAX_QIMG];        // observed delays relative to image `ref`, days
    double ivar_dt[GLAD_MAX_QIMG];       // 1 / sigma_dt^2, 0 = no measurement
};

struct glad_ctx {
    int device;
    cudaStream_t stream;
    int sm_count;
    char err[512];
    long launches;
    int smem_optin; // cudaDevAttrMaxSharedMemoryPerBlockOptin of `device`
    // row a6 options (glad_set_jam_options): nothing in the library reads the environment
    int jam_simt;   // 1 = force the FP32 SIMT quadrature kernel; default tcgen05 where the grid fits
    int jam_terms;  // bf16 terms per operand value on the tcgen05 path: 2 (default) or 3
    int jam_flush;  // chunks per TMEM accumulator group, 0 = default (512 contraction rows, at least 2 * groups - 2 chunks)
    int jam_slices; // K-slices per vector, 0 = automatic
    // The two halves are independent until joint_kernel: glad_joint_loglike_batch forks the lens half onto a context-owned
    // side stream (event fork/join on the caller's stream, so the caller still sees plain stream order).  lens_stream is
    // the stream the lens launchers use: == stream except inside that fork.  glad_set_overlap(ctx, 0) keeps everything on `stream`.
    cudaStream_t lens_stream, side_stream;
    cudaEvent_t ev_fork, ev_join;
    int overlap, side_ok;

    // lensing static data
    int light_kinds;   // bit k set: light component k (0 source, 1-2 lens light) is a Chameleon (glad_set_light_profiles)
    bool have_image;
    glad_image_grid grid;
    const float* d_data;
    const float* d_ivar;
    float* d_psf;  // ctx-owned copy [kpsf*kpsf]
    const float* d_lens_params_cur;   // the lens vectors of the batch call in flight (launch_lens_prep -> launch_lens_image)
    int kpsf;

    // internal mass sheet (glad_set_mass_sheet): d_lambda borrowed, NULL = off
    const float* d_lambda;
    double ms_rc, ms_rt, ms_lo, ms_hi;
    int ms_n, n_lambda;

    // eNFW halo (glad_set_enfw): d_enfw borrowed, NULL = off; the CSE table is copied
    const float* d_enfw;
    int n_enfw, ncse, nf_n;
    double nf_lo, nf_hi;
    double2* d_cse64;
    float2* d_cse32;

    // quasar static data (copied)
    bool have_qso;
    glad_quasar_data qso;

    // kinematic static data
    bool have_kin;
    int nx, ny, nbins, kk, nu;
    int nxf, nyf;           // folded grid (== nx, ny if not mirror-symmetric)
    const float *d_xs, *d_ys, *d_kernel, *d_vobs, *d_vivar, *d_un, *d_uw;
    const int32_t* d_bin_id;
    float *d_xf2, *d_yf2;   // ctx-owned: squared coordinates of the folded grid [nxf], [nyf]
    float *d_xf, *d_yf;     // folded coordinates
    int *d_foldx, *d_foldy; // ctx-owned: full index -> folded index [nx], [ny]
    int *d_unfoldx, *d_unfoldy; // ctx-owned: folded index -> its (up to 2) full indices, -1 = none [2*nxf], [2*nyf]
    float* d_binw;          // ctx-owned: W_f[l][pf] = sum_{p in bin l} K(p - p') over the unfolded images p' of
                            // folded pixel pf  [nbins, nyf*nxf]  (static: bins and kernel are static data)
    int* d_bin_cnt;         // ctx-owned: spaxels per bin [nbins]
    int* d_binw_ptr;        // ctx-owned: the non-zero entries of W_f row by row (the kernel K is compact, so a bin touches a
    float2* d_binw_nz;      // fraction of the map): row l = entries [ptr[l], ptr[l+1]) of {folded pixel index as int bits, weight}

    // JAM_sph rules (glad_set_jam_sph_rules): borrowed device pointers
    bool have_sph;
    int sph_nr, sph_nth, sph_nt, sph_nu, sph_nz;
    const float *d_sph_r, *d_sph_th, *d_sph_tau, *d_sph_wtau, *d_sph_un, *d_sph_uw, *d_sph_zeta, *d_sph_wz;
    float* d_sph_tab;    size_t sph_tab_cap;    // per-vector JAM_sph tables
    float* d_sph_rat;    size_t sph_rat_cap;    // [B,3,nr,nth] moment ratios when the caller does not ask for them

    // grow-only scratch
    float* d_lens_const; size_t lens_const_cap;
    float* d_lens_const_static;       // device address of lens_kernels.cu's file-scope array (glad_lens_image_noalloc); NULL = not available
    float* d_jam_tab;    size_t jam_tab_cap;
    float* d_partial;    size_t partial_cap;
    float* d_tmp;        size_t tmp_cap;     // chi2_L, chi2_D [B] each
    int32_t* d_tmpflags; size_t tmpflags_cap; // flags_L, flags_D [B] each
    float* d_stage;      size_t stage_cap;   // device staging of glad_joint_loglike_host
    float* d_qtmp;       size_t qtmp_cap;    // chi2_img, chi2_tmd [B] each (full joint entry)
    char* d_pix;         size_t pix_cap;     // glad_pixsrc_evidence_batch: L, f, A, D, s of one chunk (bytes)
    float* d_model;      size_t model_cap;   // glad_joint_loglike_model_batch: lens', profile rows, derived MGE tables

    // optional per-kernel timing (glad_profile_*): CUDA events on the context stream around each launch
    bool prof_on;
    int prof_n;
    cudaEvent_t prof_ev[2 * GLAD_PROF_MAX];
    int prof_id[GLAD_PROF_MAX];
    double prof_ms[GLAD_NKERNELS];
    long prof_cnt[GLAD_NKERNELS];
};

// Records an event pair around one launch when profiling is on (RAII; the launch goes between ctor and dtor).
struct ProfScope {
    glad_ctx* c; int slot;
    cudaStream_t st;
    ProfScope(glad_ctx* ctx, int id, cudaStream_t stream = nullptr) : c(ctx), slot(-1), st(stream ? stream : ctx->stream) {
        c->launches++;
        if (!c->prof_on || c->prof_n >= GLAD_PROF_MAX) return;
        slot = c->prof_n++;
        c->prof_id[slot] = id;
        if (!c->prof_ev[2 * slot]) { cudaEventCreate(&c->prof_ev[2 * slot]); cudaEventCreate(&c->prof_ev[2 * slot + 1]); }
        cudaEventRecord(c->prof_ev[2 * slot], st);
    }
    ~ProfScope() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], st); }
};

// Opt a kernel in to the device's maximum dynamic shared memory.  The attribute is per function AND per device, so it is set
// (to the same value every time: the device limit minus the kernel's static shared memory) before each launch instead of being cached in a process-wide static: a second context on
// another GPU, or another host thread, sees the same state.  Cost: a few microseconds of host time per launch.
template <typename K>
static inline cudaError_t smem_optin(const glad_ctx* c, K kernel) {
    // the limit covers static + dynamic shared memory; a kernel's static size is a property of its code, not of the device
    static const int static_bytes = [kernel] {
        cudaFuncAttributes fa;
        return cudaFuncGetAttributes(&fa, kernel) == cudaSuccess ? (int)fa.sharedSizeBytes : 1024;
    }();
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_optin - static_bytes);
}
// Dynamic shared memory a launch may ask for: the device's opt-in limit minus 1 KB kept for the kernels' static shared memory
// (reduction scratch, barriers).  The shape checks made when static data is set use this number.
static inline int glad_smem_dynamic_max(const glad_ctx* c) { return c->smem_optin - 1024; }
// Every entry point makes the context's device current and restores the caller's on return.
struct DeviceScope {
    int prev;
    explicit DeviceScope(const glad_ctx* c) : prev(-1) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != c->device) cudaSetDevice(c->device); else prev = -1; }
    ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
};

static inline HaloArgs halo_args(const glad_ctx* c, size_t first_vector = 0) {
    HaloArgs a;
    a.nf = c->d_enfw ? c->d_enfw + 4 * first_vector : nullptr;
    a.cse64 = c->d_cse64; a.cse32 = c->d_cse32; a.ncse = c->ncse;
    return a;
}

// kernel launchers (return cudaGetLastError())
cudaError_t launch_lens_prep(glad_ctx* c, const float* d_params, int B);
cudaError_t launch_lens_image(glad_ctx* c, int B, float* d_images, float* d_chi2, int32_t* d_flags);
cudaError_t lens_noalloc_setup(glad_ctx* c);      // glad_create, device current: address of the static constants array
cudaError_t launch_lens_noalloc(glad_ctx* c, const float* d_params, int B, float* d_images, float* d_chi2, int32_t* d_flags);
cudaError_t launch_jam_prep(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                            const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian);
cudaError_t launch_jam_quad(glad_ctx* c, int B, int nl, int nmx, int S);
// unit_scale <= 0: the partial maps are in the cylindrical quadrature's units (scale from the table header)
cudaError_t launch_jam_post(glad_ctx* c, int B, int nl, int nmx, int S, float* d_vrms, float* d_chi2,
                            float* d_v2map, int32_t* d_flags, float unit_scale = 0.f);
// JAM_sph (jam_sph.cu): prep + intrinsic moments on the polar grid + LOS integral into c->d_partial (one slice, final units);
// needs c->d_jam_tab from launch_jam_prep (validity) and c->d_sph_tab sized jam_sph_table_floats() per vector
size_t jam_sph_table_floats(int nl, int nmx, int nu);
bool jam_sph_supported(const glad_ctx* c, int nl, int nmx);
cudaError_t launch_jam_sph(glad_ctx* c, const float* d_dyn, int B, const float* d_lum, int nl, long lum_stride,
                           const float* d_mass, int nm, long mass_stride, const float* d_beta, int per_gaussian,
                           float* d_ratios);
cudaError_t launch_joint(glad_ctx* c, int B, const float* d_c2l, const float* d_c2d, const float* d_c2img, const float* d_c2tmd,
                         const int32_t* d_fl, const int32_t* d_fd, float* d_loglike, int32_t* d_flags);
cudaError_t launch_quasar(glad_ctx* c, cudaStream_t st, const float* d_lens, const float* d_ddt, int B, float* d_chi2_img,
                          float* d_chi2_tmd, double* d_theta_pre, double* d_dt_pre, double* d_beta);
cudaError_t launch_kin_weights(glad_ctx* c);
cudaError_t launch_mge1d(glad_ctx* c, int kind, const float* d_prof, int B, int n_gauss, float sigma_lo, float sigma_hi,
                         int P, float* d_mge);
// d_mass has n_mass rows per vector, plus c->ms_n rows of the mass sheet when c->d_lambda is set
cudaError_t launch_model(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, double zd, int B, int tracer_kind, int n_lum,
                         float lum_lo, float lum_hi, int n_mass, float mass_lo, float mass_hi, int P, float* d_lens_out,
                         float* d_lum, float* d_mass);
// pixelated-source evidence (pixsrc_kernels.cu): bytes of scratch for a chunk of Bc vectors; the whole chain for one chunk
// search = the lambda_hat entry (a second N_s^2 matrix per vector + the search state)
size_t pixsrc_scratch_bytes(int npix, int ns, int Bc, bool search);
// d_lam != NULL: evidence at the given lambda; d_lam == NULL: lambda_hat searched on [lam_lo, lam_hi] (Eq. 43) and written to d_lam_hat
cudaError_t launch_pixsrc_chunk(glad_ctx* c, void* scratch, const float* d_lens, const float* d_src_grid, const float* d_lam,
                                const float* d_ms_lambda, int nsx, int nsy, int Bc, double logdet_g, float* d_logev, float* d_chi2,
                                float* d_reg, float* d_s_mp, float* d_model, int32_t* d_flags, double lam_lo, double lam_hi,
                                float* d_lam_hat);
// F = f^T C_d^-1 f (+ lambda g, lower triangle, fp64 out) and D = f^T C_d^-1 d on tcgen05 (pixsrc_syrk_tc.cu); d_lam NULL = plain F
cudaError_t launch_pixsrc_syrk_tc(glad_ctx* c, cudaStream_t st, const float* f, const int2* rng, const float* d_lam, int npix, int ns,
                                  int nsx, int nsy, int Bc, const double* stat, unsigned short* rowlist, double* A, double* D);
// batched Cholesky of the Bc matrices A [ns, ns] (lower triangle, in place; pixsrc_chol.cu); out[b*6+0] = ln det, out[b*6+3] = not-PD flag
size_t pixsrc_factor_scratch_bytes(int Bc);
cudaError_t launch_pixsrc_factor(glad_ctx* c, cudaStream_t st, double* A, int ns, int Bc, double* out, double* Winv);
// tensor-core (tcgen05) form of row a6; supported when the folded grid has ny_f <= 128, N = terms * nx_f <= 256
// and two operand stages fit in shared memory
bool jam_quad_tc_supported(const glad_ctx* c, int nl, int nmx);
cudaError_t launch_jam_quad_tc(glad_ctx* c, int B, int nl, int nmx, int S);
// dynamic shared memory of lens_image_kernel / jam_post_kernel for given sizes (checked when the static data is set)
size_t lens_image_smem_bytes(int nx, int ny, int kpsf);
size_t jam_post_smem_bytes(int nxf, int nyf, int nl);
// launch geometry of the quadrature kernel for the current sky grid: threads per CTA, thread groups
int jam_quad_geometry(const glad_ctx* c, int* groups);
