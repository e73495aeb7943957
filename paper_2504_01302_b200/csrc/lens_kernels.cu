// Lensing half of libglad for sm_100a: rows a0-a4 of SURVEY.md 8(a).
//   lens_prep_kernel  : per-vector constants in fp64 -> fp32 (EPL normalisation Eq. B.3, series
//                       coefficients, Sersic b_n root, rotations); validity flag.
//   lens_image_kernel : one CTA per parameter vector.  Ray-shoot every sub-pixel (Eq. 33), evaluate
//                       source at beta and lens light at theta, bin down into a whole-image shared-memory
//                       tile, convolve with the PSF from shared memory (Eq. 38), reduce chi2 with
//                       warp shuffles (Eq. 48).  No intermediate ever touches HBM.
#include <math.h>

#include "glad_internal.h"
#include "glad_special.cuh"
#include "glad_mass_fp64.cuh"

// 4 warps per 32 parameter vectors (lane = vector): warp role 0 = EPL / shear / point mass / validity, roles 1..3 =
// one Sersic component each (the b_n root is the only long serial chain of the kernel; a warp never mixes roles).
#define LENS_PREP_ROLES 4
__global__ void __launch_bounds__(32 * LENS_PREP_ROLES) lens_prep_kernel(const float* __restrict__ params, int B, int kinds,
                                                                         const float* __restrict__ lambda, double ms_rc, double ms_rt,
                                                                         const float* __restrict__ enfw, float* __restrict__ consts) {
    const int b = blockIdx.x * 32 + (threadIdx.x & 31), role = threadIdx.x >> 5;
    if (b >= B) return;
    const float* p = params + (size_t)b * GLAD_NLENS;
    float* c = consts + (size_t)b * LC_SIZE;
    double xl = p[0], yl = p[1], thE = p[2], gam = p[3], q = p[4], pa = p[5];
    bool valid = (thE >= 0.0) && (gam > 1.0 && gam < 3.0) && (q > 0.0 && q <= 1.0) && (p[8] >= 0.f);
    // internal mass sheet (Eq. 6 P:85 with the dPIE profile of Eq. 50; R-S1..3): kappa_int = (1-lam) S(R) + lam kappa_epl
    const double lam = lambda ? (double)lambda[b] : 1.0;
    if (!isfinite(lam)) valid = false;
    // eNFW halo {rho_s, r_s, q, phi} (Appendix A; R-N1..3): rho_s = 0 disables it
    const float* nf = enfw ? enfw + (size_t)b * 4 : nullptr;
    if (nf && !((nf[0] >= 0.f) && (nf[0] == 0.f || (nf[1] > 0.f && nf[2] > 0.f && nf[2] <= 1.f)))) valid = false;
    for (int k = 0; k < 3; ++k) {
        const float* s = p + (k == 0 ? 11 : (k == 1 ? 16 : 21));
        const bool cham = (kinds >> k) & 1;                            // Chameleon (Eq. 47): 0 < w_c < w_t
        if (s[0] != 0.f && !(s[1] > 0.f && (cham ? s[2] > s[1] : s[2] > 0.f) && s[3] > 0.f && s[3] <= 1.f)) valid = false;
    }
    if (role > 0) {
        const int k = role - 1;
        const float* s = p + (k == 0 ? 11 : (k == 1 ? 16 : 21));
        float* o = c + LC_SERSIC0 + k * LC_SERSIC_STRIDE;
        for (int i = 0; i < LC_SERSIC_STRIDE; ++i) o[i] = 0.f;
        if (!valid) return;
        double Ie = s[0], Re = s[1], n = s[2], qs = s[3], phi = s[4];
        o[0] = (k == 0) ? p[9] : (float)xl;
        o[1] = (k == 0) ? p[10] : (float)yl;
        if (Ie == 0.0) return;
        if ((kinds >> k) & 1) {
            // Chameleon, Eq. 47: slot = {I_0, w_c, w_t, q, phi}; I = amp (1/sqrt(R^2 + a_c) - 1/sqrt(R^2 + a_t)), a = 4 w^2/(1+q)^2
            const double opq = 1.0 + qs;
            o[2] = (float)cos(phi); o[3] = (float)sin(phi);
            o[4] = (float)(1.0 / (qs * qs));
            o[5] = (float)(Ie / opq);
            o[6] = (float)(4.0 * Re * Re / (opq * opq));                   // a_c
            o[7] = (float)(4.0 * (n * n - Re * Re) / (opq * opq));         // a_t - a_c, formed in fp64
            return;
        }
        double bn = sersic_bn(n);
        o[2] = (float)cos(phi); o[3] = (float)sin(phi);
        o[4] = (float)(1.0 / (qs * qs));
        o[5] = (float)(Ie * exp(bn));                                  // I(0)
        o[6] = (float)(bn * 1.4426950408889634 * pow(Re, -1.0 / n));   // I = amp 2^(-k1 (R^2)^h)
        o[7] = (float)(0.5 / n);
        return;
    }
    for (int i = 0; i < LC_SERSIC0; ++i) c[i] = 0.f;
    for (int i = LC_SERIES; i < LC_SIZE; ++i) c[i] = 0.f;
    c[LC_VALID] = valid ? 1.f : 0.f;
    if (!valid) return;
    if (nf && nf[0] > 0.f) {
        const double rho = nf[0], rs = nf[1], qh = nf[2];
        c[LC_NF_AMP] = (float)(rho * rs / sqrt(qh));
        c[LC_NF_SC] = (float)(sqrt(qh) / rs);
        c[LC_NF_Q] = (float)qh;
        c[LC_NF_COS] = (float)cos((double)nf[3]);
        c[LC_NF_SIN] = (float)sin((double)nf[3]);
    }
    double tt = gam - 1.0;
    double f = (1.0 - q) / (1.0 + q);
    double bTM = q * pow(2.0 / (1.0 + q), 1.0 / tt) * thE;  // b_TM = q b, b from Eq. B.3
    c[LC_XL] = (float)xl; c[LC_YL] = (float)yl;
    c[LC_COSPA] = (float)cos(pa); c[LC_SINPA] = (float)sin(pa);
    c[LC_Q] = (float)q; c[LC_NEGF] = (float)(-f);
    c[LC_PREF] = (thE > 0.0) ? (float)(lam * 2.0 * pow(bTM, tt) / (1.0 + q)) : 0.f;
    if (lambda) {
        c[LC_MS_AMP] = (float)((1.0 - lam) * 2.0 * ms_rc * ms_rt);
        c[LC_MS_RC] = (float)ms_rc;
        c[LC_MS_RT] = (float)ms_rt;
    }
    c[LC_HEXP] = (float)(-0.5 * (tt - 1.0));
    int nt = 0;
    if (f > 1e-12) {
        nt = (int)ceil(log(2e-8) / log(f)) + 1;
        if (nt < 1) nt = 1;
        if (nt > GLAD_EPL_TERMS_CAP) nt = GLAD_EPL_TERMS_CAP;
    }
    c[LC_NTERMS] = (float)nt;
    for (int n = 1; n <= GLAD_EPL_MAX_TERMS; ++n)
        c[LC_SERIES + n - 1] = (float)((2.0 * n - (2.0 - tt)) / (2.0 * n + (2.0 - tt)));
    c[LC_SH_C] = (float)((double)p[6] * cos(2.0 * (double)p[7]));
    c[LC_SH_S] = (float)((double)p[6] * sin(2.0 * (double)p[7]));
    c[LC_BH] = p[8];
}

// ------------------------------------------------------------------------------------------------
// main kernel
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2f(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ __forceinline__ float sersic_eval(const float* __restrict__ o, float px, float py) {
    float dx = px - o[0], dy = py - o[1];
    float x = dx * o[2] + dy * o[3];
    float y = dy * o[2] - dx * o[3];
    float R2 = fmaf(y * y, o[4], x * x);
    float pw = ex2f(o[7] * lg2f(R2));      // (R^2)^(1/2n); R2 = 0 -> 0
    return o[5] * ex2f(-o[6] * pw);
}

// Cusp guard: an fp32 ray carries ~5e-7" of absolute error in beta (|alpha| ~ 1.7").  Where the source
// profile is steep, |grad ln I| <= ln2 k1 2h (R^2)^h / R x max(1, 1/q_s) (the elliptical radius R stretches the minor axis by 1/q_s: a
// q_s = 0.15, n = 3.8 source of the C2 batch was 1.4e-4 off at its peak with the bound in R alone), that error is amplified: above
// LENS_CUSP_SLOPE per arcsec (2e-5 per ray) the
// pixel is recomputed with fp64 rays (src_pixel_fp64).  Happens within ~0.05" of the centre of an n ~ 4 source: a few hundred of the
// 40 000 rays of a C2 vector; one C2 vector in 1024 had a peak pixel 1.09e-4 off without it.
#define LENS_CUSP_SLOPE 30.f
__device__ __forceinline__ float sersic_at(const float* __restrict__ o, float dx, float dy, bool& cusp) {
    float x = dx * o[2] + dy * o[3];
    float y = dy * o[2] - dx * o[3];
    float R2 = fmaf(y * y, o[4], x * x);
    float pw = ex2f(o[7] * lg2f(R2));      // (R^2)^(1/2n); R2 = 0 -> 0
    const float gl = 1.3862944f * o[6] * o[7] * pw;                  // |d ln I / d ln R| = ln2 k1 2h pw
    cusp = gl * gl * fmaxf(o[4], 1.f) > (LENS_CUSP_SLOPE * LENS_CUSP_SLOPE) * R2;   // |grad ln I| <= (gl / R) max(1, 1/q_s): o[4] = 1/q_s^2
    return o[5] * ex2f(-o[6] * pw);
}

__device__ __forceinline__ float chameleon_eval(const float* __restrict__ o, float px, float py) {
    float dx = px - o[0], dy = py - o[1];
    float x = dx * o[2] + dy * o[3];
    float y = dy * o[2] - dx * o[3];
    float R2 = fmaf(y * y, o[4], x * x);
    // 1/s_c - 1/s_t = (a_t - a_c) / (s_c s_t (s_c + s_t)): no cancellation at large R or for close core radii
    float uc = R2 + o[6], ut = uc + o[7];
    float rc = rsqrtf(uc), rt = rsqrtf(ut);
    return o[5] * o[7] * rc * rt * __fdividef(1.f, fmaf(uc, rc, ut * rt));
}
// CH = some component is a Chameleon (kinds bit k set) or the internal mass sheet is on; the <false> instantiation is the code of
// rows a1-a2 as before
template <bool CH>
__device__ __forceinline__ float light_eval(int kinds, int k, const float* __restrict__ o, float px, float py) {
    if (CH && ((kinds >> k) & 1)) return chameleon_eval(o, px, py);
    return sersic_eval(o, px, py);
}

// One ray: returns source(beta) + lens light(theta).
// LONG = the vector needs more series terms than the stored table holds (q < 0.2): a separate instantiation, so that the
// code of the common case is exactly the table-driven loop
template <bool CH, bool LONG>
__device__ __forceinline__ float shoot(const float* __restrict__ c, float thx, float thy, int nterms,
                                       bool has_src, bool has_l1, bool has_l2, int kinds, const float2* __restrict__ cse, int ncse,
                                       float& src, bool& cusp) {
    float dx = thx - c[LC_XL], dy = thy - c[LC_YL];
    float cs = c[LC_COSPA], sn = c[LC_SINPA];
    float x = dx * cs + dy * sn, y = dy * cs - dx * sn;
    float qx = c[LC_Q] * x;
    float R2 = fmaxf(fmaf(qx, qx, y * y), 1e-12f);
    float rinv = rsqrtf(R2);
    float wr = qx * rinv, wi = y * rinv;
    float negf = c[LC_NEGF];
    float zr = negf * (wr * wr - wi * wi), zi = negf * (2.f * wr * wi);
    // Horner: h_n = 1 + c_n z h_{n+1}, sum = h_1
    float hr = 1.f, hi = 0.f;
    if (LONG) {
        // very flat mass (q < 0.2): the terms past the stored table take c_n = (2n - a)/(2n + a), a = 2 - t = 1 + 2 HEXP, on the fly
        const float a2t = fmaf(2.f, c[LC_HEXP], 1.f);
        for (int n = nterms; n > GLAD_EPL_MAX_TERMS; --n) {
            const float tn = 2.f * (float)n;
            const float cn = __fdividef(tn - a2t, tn + a2t);
            float tr = fmaf(zr, hr, -zi * hi), ti = fmaf(zr, hi, zi * hr);
            hr = fmaf(cn, tr, 1.f);
            hi = cn * ti;
        }
        nterms = GLAD_EPL_MAX_TERMS;
    }
    for (int n = nterms; n >= 1; --n) {
        float cn = c[LC_SERIES + n - 1];
        float tr = fmaf(zr, hr, -zi * hi), ti = fmaf(zr, hi, zi * hr);
        hr = fmaf(cn, tr, 1.f);
        hi = cn * ti;
    }
    float mag = c[LC_PREF] * ex2f(c[LC_HEXP] * lg2f(R2));
    float ar = mag * (wr * hr - wi * hi), ai = mag * (wr * hi + wi * hr);
    float ax = ar * cs - ai * sn, ay = ar * sn + ai * cs;
    ax = fmaf(c[LC_SH_C], dx, fmaf(c[LC_SH_S], dy, ax));
    ay = fmaf(c[LC_SH_S], dx, fmaf(-c[LC_SH_C], dy, ay));
    float r2 = fmaxf(fmaf(dx, dx, dy * dy), 1e-12f);
    float bh = __fdividef(c[LC_BH], r2);
    ax = fmaf(bh, dx, ax);
    ay = fmaf(bh, dy, ay);
    if (CH && c[LC_MS_AMP] != 0.f) {
        // mass sheet: alpha = g (dx, dy), g = (1-lam) 2 rc rt [1 + (rt+rc)/(ht+hc)] / ((hc+rc)(ht+rt)), h = sqrt(R^2 + r^2):
        // the closed form 2A[(hc-rc) - (ht-rt)]/R^2 with the common factor (rt - rc) divided out (no cancellation in fp32)
        const float rc = c[LC_MS_RC], rt = c[LC_MS_RT];
        const float rr = fmaf(dx, dx, dy * dy);
        const float hc = sqrtf(fmaf(rc, rc, rr)), ht = sqrtf(fmaf(rt, rt, rr));
        const float gs = c[LC_MS_AMP] * (1.f + (rt + rc) / (ht + hc)) / ((hc + rc) * (ht + rt));   // IEEE divisions: this path is optional
        ax = fmaf(gs, dx, ax);
        ay = fmaf(gs, dy, ay);
    }
    if (CH && c[LC_NF_AMP] != 0.f) {
        // eNFW halo = sum of core-steep ellipsoids (Eq. A.3-A.7): alpha_X = (q X / s) [a q^2/psi_s + 1 - q^2] / Psi,
        // alpha_Y = (q Y / s) a / (psi_s Psi), a = psi_s + s, in the halo frame scaled by sqrt(q)/r_s; every term positive
        const float q = c[LC_NF_Q], q2 = q * q, omq2 = 1.f - q2, hc = c[LC_NF_COS], hs = c[LC_NF_SIN];
        const float X = c[LC_NF_SC] * (dx * hc + dy * hs), Y = c[LC_NF_SC] * (dy * hc - dx * hs);
        const float X2 = X * X, Y2 = Y * Y;
        float sx = 0.f, sy = 0.f;
        for (int i = 0; i < ncse; ++i) {
            const float2 t = __ldg(cse + i);                          // {A_i / s_i, s_i}
            const float s2 = t.y * t.y;
            const float pss = sqrtf(fmaf(q2, s2 + X2, Y2));
            const float a = pss + t.y;
            const float iden = __fdividef(t.x, pss * fmaf(a, a, omq2 * X2));
            sx = fmaf(iden, fmaf(a, q2, omq2 * pss), sx);
            sy = fmaf(iden, a, sy);
        }
        const float hx = c[LC_NF_AMP] * q * X * sx, hy = c[LC_NF_AMP] * q * Y * sy;
        ax += hx * hc - hy * hs;
        ay += hx * hs + hy * hc;
    }
    float v = 0.f;
    src = 0.f;
    cusp = false;
    if (has_src) {
        const float* o = c + LC_SERSIC0;
        if (CH && (kinds & 1)) src = chameleon_eval(o, thx - ax, thy - ay);          // cored: no cusp
        else src = sersic_at(o, (thx - ax) - o[0], (thy - ay) - o[1], cusp);
    }
    if (has_l1) v += light_eval<CH>(kinds, 1, c + LC_SERSIC0 + LC_SERSIC_STRIDE, thx, thy);
    if (has_l2) v += light_eval<CH>(kinds, 2, c + LC_SERSIC0 + 2 * LC_SERSIC_STRIDE, thx, thy);
    return v;
}

// PSF convolution geometry: a thread owns LENS_STRIP consecutive output pixels of one row; taps are consumed
// LENS_TAPS at a time with every register index static, so the inner block is LENS_STRIP*LENS_TAPS FFMAs on
// LENS_STRIP+LENS_TAPS-1 source pixels and LENS_TAPS taps held in registers.  The binned image sits in shared memory
// with a zero halo (left cc+LENS_TAPS, right cc+LENS_STRIP-1) and one zero row, so the loop has no bounds tests;
// the row pitch is odd and consecutive lanes own consecutive rows, so source loads are bank-conflict free and
// tap loads are broadcasts.
#define LENS_STRIP 16
#define LENS_TAPS 8
static inline __host__ __device__ int lens_tap_pitch(int kpsf) { return (kpsf + LENS_TAPS - 1) & ~(LENS_TAPS - 1); }
static inline __host__ __device__ int lens_halo_left(int kpsf) { return kpsf / 2 + LENS_TAPS; }
static inline __host__ __device__ int lens_img_pitch(int nx, int kpsf) { return (nx + 2 * (kpsf / 2) + LENS_TAPS + LENS_STRIP - 1) | 1; }

#define LENS_CUSP_LIST 2048
__device__ __noinline__ void cusp_mass_const(const float* __restrict__ p, double lam, double rc, double rt, bool sheet, const float* nf,
                                             const double2* cse, int ncse, MassConst& m) {
    mass_const(p, lam, rc, rt, sheet, m);
    mass_const_halo(nf, cse, ncse, m);
}
// rows a1-a3 for one vector: every sub-pixel ray, averaged into the binned image in shared memory.  A pixel one of whose rays trips
// the cusp guard keeps only its lens light here and is put on the list for src_pixel_fp64 (or, if the list is full, done at once).
template <bool CH>
__device__ __noinline__ float src_pixel_fp64(const float* __restrict__ c, const glad_image_grid& g, const MassConst& m, int ix, int iy);
template <bool CH>
__device__ __noinline__ float src_ray_fp64(const float* __restrict__ c, const glad_image_grid& g, const MassConst& m, int ix, int iy, int r);

template <bool CH, bool LONG>
__device__ __forceinline__ void ray_pass(const float* __restrict__ c, const glad_image_grid& g, float* __restrict__ img, int pitch,
                                         int HL, int nterms, int kinds, const float2* __restrict__ cse, int ncse,
                                         unsigned short* __restrict__ cusp_list, int* __restrict__ cusp_count, const MassConst& m) {
    const int tid = threadIdx.x, nthr = blockDim.x, nx = g.nx, npx = g.nx * g.ny, ss = g.supersample;
    const bool has_src = c[LC_SERSIC0 + 5] != 0.f;
    const bool has_l1 = c[LC_SERSIC0 + LC_SERSIC_STRIDE + 5] != 0.f;
    const bool has_l2 = c[LC_SERSIC0 + 2 * LC_SERSIC_STRIDE + 5] != 0.f;
    const float inv_s = 1.f / (float)ss, inv_s2 = 1.f / (float)(ss * ss);
    for (int p = tid; p < npx; p += nthr) {
        int iy = p / nx, ix = p - iy * nx;
        float acc = 0.f, acc_s = 0.f;
        bool any = false;
        for (int sb = 0; sb < ss; ++sb) {
            float thy = fmaf(g.pix, (float)iy + (((float)sb + 0.5f) * inv_s - 0.5f), g.y0);
            for (int sa = 0; sa < ss; ++sa) {
                float thx = fmaf(g.pix, (float)ix + (((float)sa + 0.5f) * inv_s - 0.5f), g.x0);
                float src;
                bool cusp;
                acc += shoot<CH, LONG>(c, thx, thy, nterms, has_src, has_l1, has_l2, kinds, cse, ncse, src, cusp);
                acc_s += src;
                any |= cusp;
            }
        }
        if (any) {
            const int slot = atomicAdd(cusp_count, 1);
            if (slot < LENS_CUSP_LIST) { cusp_list[slot] = (unsigned short)p; acc_s = 0.f; }
            else acc_s = src_pixel_fp64<CH>(c, g, m, ix, iy);
        }
        img[iy * pitch + HL + ix] = (acc + acc_s) * inv_s2;
    }
}

// out of line: the rare long-series loop must not raise the register count of the kernel (2 CTAs of 512 threads per SM)
template <bool CH>
__device__ __noinline__ void ray_pass_long(const float* __restrict__ c, const glad_image_grid& g, float* __restrict__ img, int pitch,
                                           int HL, int nterms, int kinds, const float2* __restrict__ cse, int ncse,
                                           unsigned short* __restrict__ cusp_list, int* __restrict__ cusp_count, const MassConst& m) {
    ray_pass<CH, true>(c, g, img, pitch, HL, nterms, kinds, cse, ncse, cusp_list, cusp_count, m);
}

// Sum over the s x s rays of pixel (ix, iy) of the SOURCE brightness with the deflection in fp64 (the mass model of the quasar terms,
// glad_mass_fp64.cuh, from the raw parameters: the same arithmetic type as the definition), beta - source centre formed in fp64, the
// profile itself in fp32.  Only the Sersic source reaches this (a Chameleon source has a core).
template <bool CH>
__device__ __noinline__ float src_pixel_fp64(const float* __restrict__ c, const glad_image_grid& g, const MassConst& m, int ix, int iy) {
    const int ss = g.supersample;
    float sum = 0.f;
    for (int r = 0; r < ss * ss; ++r) sum += src_ray_fp64<CH>(c, g, m, ix, iy, r);
    return sum;
}
// one of the s x s rays of the pixel: r = sb * s + sa
template <bool CH>
__device__ __noinline__ float src_ray_fp64(const float* __restrict__ c, const glad_image_grid& g, const MassConst& m, int ix, int iy, int r) {
    const float* o = c + LC_SERSIC0;
    const int ss = g.supersample, sb = r / ss, sa = r - sb * ss;
    const double thx = (double)g.x0 + (double)g.pix * ((double)ix + (((double)sa + 0.5) / ss - 0.5));
    const double thy = (double)g.y0 + (double)g.pix * ((double)iy + (((double)sb + 0.5) / ss - 0.5));
    MassEval e;
    mass_eval(m, thx, thy, e);
    bool dummy;
    return sersic_at(o, (float)(thx - e.ax - (double)o[0]), (float)(thy - e.ay - (double)o[1]), dummy);
}

template <bool CH>
__global__ void __launch_bounds__(512, 2) lens_image_kernel(const float* __restrict__ consts, int kinds, glad_image_grid g,
                                                         const float* __restrict__ psf, int kpsf,
                                                         const float* __restrict__ data,
                                                         const float* __restrict__ ivar, float* __restrict__ images,
                                                         float* __restrict__ chi2, int32_t* __restrict__ flags,
                                                         const float2* __restrict__ cse, int ncse, const float* __restrict__ params,
                                                         const float* __restrict__ lambda, double ms_rc, double ms_rt, const HaloArgs halo) {
    extern __shared__ __align__(16) float smem[];
    __shared__ MassConst s_mc;                           // fp64 mass model of this vector, for the cusp guard's rays
    __shared__ unsigned short s_cusp[LENS_CUSP_LIST];
    __shared__ int s_ncusp;
    const int b = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x;
    const int nx = g.nx, ny = g.ny, npx = nx * ny;
    const int KP = lens_tap_pitch(kpsf), HL = lens_halo_left(kpsf), pitch = lens_img_pitch(nx, kpsf);
    float* c = smem;                       // LC_SIZE
    float* spsf = smem + LC_SIZE;          // kpsf rows x KP taps, zero padded
    float* img = spsf + kpsf * KP;         // (ny + 1) rows x pitch, zero halo, last row zero
    __shared__ float red[32];

    for (int i = tid; i < LC_SIZE; i += nthr) c[i] = consts[(size_t)b * LC_SIZE + i];
    for (int i = tid; i < kpsf * KP; i += nthr) {
        int r = i / KP, k = i - r * KP;
        spsf[i] = k < kpsf ? psf[r * kpsf + k] : 0.f;
    }
    for (int i = tid; i < (ny + 1) * pitch; i += nthr) img[i] = 0.f;
    if (tid == nthr - 1) {
        s_ncusp = 0;
        cusp_mass_const(params + (size_t)b * GLAD_NLENS, (CH && lambda) ? (double)lambda[b] : 1.0, ms_rc, ms_rt, CH && lambda != nullptr,
                        (CH && halo.nf) ? halo.nf + 4 * (size_t)b : nullptr, halo.cse64, halo.ncse, s_mc);
    }
    __syncthreads();
    const bool valid = c[LC_VALID] != 0.f;
    if (!valid) {
        if (images) for (int i = tid; i < npx; i += nthr) images[(size_t)b * npx + i] = __int_as_float(0x7fc00000);
        if (tid == 0) {
            if (chi2) chi2[b] = __int_as_float(0x7f800000);
            if (flags) flags[b] = GLAD_FLAG_LENS_INVALID;
        }
        return;
    }
    const int nterms = (int)c[LC_NTERMS];

    // rows a1-a3: rays -> binned pixel in shared memory
    if (nterms > GLAD_EPL_MAX_TERMS) ray_pass_long<CH>(c, g, img, pitch, HL, nterms, kinds, cse, ncse, s_cusp, &s_ncusp, s_mc);   // CTA-uniform
    else ray_pass<CH, false>(c, g, img, pitch, HL, nterms, kinds, cse, ncse, s_cusp, &s_ncusp, s_mc);
    __syncthreads();
    {
        // cusp guard: the listed pixels get their source light from fp64 rays.  LP = 4 or 8 neighbouring lanes share a pixel, one
        // ray (or two) each, and add up by shuffles: no atomics, a result that does not depend on the order of the list, and the
        // few hundred listed pixels keep the whole CTA busy (one thread per pixel left most of it idle behind a chain of s^2 fp64
        // ray evaluations: a tenth of the kernel)
        const int nc = min(s_ncusp, LENS_CUSP_LIST);
        const int R = g.supersample * g.supersample, LP = R <= 4 ? 4 : 8;
        const float inv_s2 = 1.f / (float)R;
        const int lr = tid & (LP - 1), per_pass = nthr / LP;
        for (int base = 0; base < nc; base += per_pass) {                   // trip count is CTA-uniform
            const int e = base + tid / LP;
            float sum = 0.f;
            int iy = 0, ix = 0;
            if (e < nc) {
                const int p = s_cusp[e];
                iy = p / nx; ix = p - iy * nx;
                for (int r = lr; r < R; r += LP) sum += src_ray_fp64<CH>(c, g, s_mc, ix, iy, r);
            }
            for (int o = LP >> 1; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
            if (e < nc && lr == 0) img[iy * pitch + HL + ix] += sum * inv_s2;
        }
        __syncthreads();
    }

    // row a4: PSF convolution from shared memory + chi2.  out[x] = sum_dy sum_dx psf[dy][dx] img[y+cc-dy][x+cc-dx]
    const int cc = kpsf / 2;
    const int nstrip_x = (nx + LENS_STRIP - 1) / LENS_STRIP;
    const int nitems = ny * nstrip_x;
    float part = 0.f;
    for (int t = tid; t < nitems; t += nthr) {
        const int sx = t / ny, y = t - sx * ny, x0 = sx * LENS_STRIP;
        float out[LENS_STRIP];
#pragma unroll
        for (int j = 0; j < LENS_STRIP; ++j) out[j] = 0.f;
        for (int dy = 0; dy < kpsf; ++dy) {
            int sy = y + cc - dy;
            sy = ((unsigned)sy < (unsigned)ny) ? sy : ny;                   // out of range -> the zero row
            // source column of (output j, tap dx = c8 + d) in halo coordinates: x0 + HL + cc - c8 + (j - d)
            const float* row = img + sy * pitch + x0 + HL + cc - (LENS_TAPS - 1);
            const float* prow = spsf + dy * KP;
            for (int c8 = 0; c8 < KP; c8 += LENS_TAPS) {
                const float4 pa = *reinterpret_cast<const float4*>(prow + c8);
                const float4 pb = *reinterpret_cast<const float4*>(prow + c8 + 4);
                const float p[LENS_TAPS] = {pa.x, pa.y, pa.z, pa.w, pb.x, pb.y, pb.z, pb.w};
                const float* r = row - c8;
                float s[LENS_STRIP + LENS_TAPS - 1];
#pragma unroll
                for (int i = 0; i < LENS_STRIP + LENS_TAPS - 1; ++i) s[i] = r[i];
#pragma unroll
                for (int d = 0; d < LENS_TAPS; ++d)
#pragma unroll
                    for (int j = 0; j < LENS_STRIP; ++j) out[j] = fmaf(p[d], s[j - d + LENS_TAPS - 1], out[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < LENS_STRIP; ++j) {
            int x = x0 + j;
            if (x < nx) {
                int p = y * nx + x;
                if (images) images[(size_t)b * npx + p] = out[j];
                if (chi2) {
                    float r = data[p] - out[j];
                    part = fmaf(ivar[p] * r, r, part);
                }
            }
        }
    }
    if (chi2) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        if ((tid & 31) == 0) red[tid >> 5] = part;
        __syncthreads();
        if (tid < 32) {
            float v = (tid < (nthr >> 5)) ? red[tid] : 0.f;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (tid == 0) chi2[b] = v;
        }
    }
    if (flags && tid == 0) flags[b] = 0;
}

cudaError_t launch_lens_prep(glad_ctx* c, const float* d_params, int B) {
    c->d_lens_params_cur = d_params;                 // lens_image_kernel's cusp guard re-reads the raw vectors (launched right after this)
    ProfScope ps(c, GK_LENS_PREP, c->lens_stream);
    lens_prep_kernel<<<(B + 31) / 32, 32 * LENS_PREP_ROLES, 0, c->lens_stream>>>(d_params, B, c->light_kinds, c->d_lambda, c->ms_rc,
                                                                                 c->ms_rt, c->d_enfw, c->d_lens_const);
    return cudaGetLastError();
}

size_t lens_image_smem_bytes(int nx, int ny, int kpsf) {
    return sizeof(float) * (LC_SIZE + (size_t)kpsf * lens_tap_pitch(kpsf) + (size_t)(ny + 1) * lens_img_pitch(nx, kpsf));
}

cudaError_t launch_lens_image(glad_ctx* c, int B, float* d_images, float* d_chi2, int32_t* d_flags) {
    const size_t smem = lens_image_smem_bytes(c->grid.nx, c->grid.ny, c->kpsf);
    if (smem > (size_t)glad_smem_dynamic_max(c)) return cudaErrorInvalidConfiguration;   // glad_set_image_data checks this up front
    const int ch = c->light_kinds != 0 || c->d_lambda != nullptr || c->d_enfw != nullptr;
    cudaError_t e = ch ? smem_optin(c, lens_image_kernel<true>) : smem_optin(c, lens_image_kernel<false>);
    if (e != cudaSuccess) return e;
    ProfScope ps(c, GK_LENS_IMAGE, c->lens_stream);
    if (ch)
        lens_image_kernel<true><<<B, 512, smem, c->lens_stream>>>(c->d_lens_const, c->light_kinds, c->grid, c->d_psf, c->kpsf,
                                                                 c->d_data, c->d_ivar, d_images, d_chi2, d_flags, c->d_cse32, c->ncse, c->d_lens_params_cur,
                                                                 c->d_lambda, c->ms_rc, c->ms_rt, halo_args(c));
    else
        lens_image_kernel<false><<<B, 512, smem, c->lens_stream>>>(c->d_lens_const, 0, c->grid, c->d_psf, c->kpsf, c->d_data,
                                                                  c->d_ivar, d_images, d_chi2, d_flags, nullptr, 0, c->d_lens_params_cur, nullptr, 0.0, 0.0, HaloArgs{nullptr, nullptr, nullptr, 0});
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// glad_lens_image_noalloc: the same two kernels with the per-vector constants in a file-scope device array, for callers that
// cannot allocate at call time.  In host code the array's NAME is a host-side stand-in, not a device address: the address the
// kernels get is the one cudaGetSymbolAddress returns, taken once per device with that device current.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) float g_lens_const_noalloc[(size_t)GLAD_LENS_NOALLOC_MAX_B * LC_SIZE];

#define LENS_NOALLOC_MAX_DEV 64
static float* s_noalloc_addr[LENS_NOALLOC_MAX_DEV];      // per device; 0 = not taken yet

cudaError_t lens_noalloc_setup(glad_ctx* c) {
    c->d_lens_const_static = nullptr;
    if (c->device < 0 || c->device >= LENS_NOALLOC_MAX_DEV) return cudaErrorInvalidDevice;
    float* p = s_noalloc_addr[c->device];
    if (!p) {
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_lens_const_noalloc);
        if (e != cudaSuccess) return e;
        // the shared-memory opt-in of the image kernel is per function and per device: set here so that the call itself only launches
        e = smem_optin(c, lens_image_kernel<true>);
        if (e == cudaSuccess) e = smem_optin(c, lens_image_kernel<false>);
        cudaFuncAttributes fa;                              // loads the first kernel's code now rather than at its first launch
        if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, lens_prep_kernel);
        if (e != cudaSuccess) return e;
        s_noalloc_addr[c->device] = p;
    }
    c->d_lens_const_static = p;
    return cudaSuccess;
}

cudaError_t launch_lens_noalloc(glad_ctx* c, const float* d_params, int B, float* d_images, float* d_chi2, int32_t* d_flags) {
    float* consts = c->d_lens_const_static;
    if (!consts || B > GLAD_LENS_NOALLOC_MAX_B) return cudaErrorInvalidValue;
    const size_t smem = lens_image_smem_bytes(c->grid.nx, c->grid.ny, c->kpsf);
    if (smem > (size_t)glad_smem_dynamic_max(c)) return cudaErrorInvalidConfiguration;
    cudaStream_t st = c->stream;
    const int ch = c->light_kinds != 0 || c->d_lambda != nullptr || c->d_enfw != nullptr;
    lens_prep_kernel<<<(B + 31) / 32, 32 * LENS_PREP_ROLES, 0, st>>>(d_params, B, c->light_kinds, c->d_lambda, c->ms_rc, c->ms_rt,
                                                                     c->d_enfw, consts);
    if (ch)
        lens_image_kernel<true><<<B, 512, smem, st>>>(consts, c->light_kinds, c->grid, c->d_psf, c->kpsf, c->d_data, c->d_ivar, d_images,
                                                      d_chi2, d_flags, c->d_cse32, c->ncse, d_params, c->d_lambda, c->ms_rc, c->ms_rt,
                                                      halo_args(c));
    else
        lens_image_kernel<false><<<B, 512, smem, st>>>(consts, 0, c->grid, c->d_psf, c->kpsf, c->d_data, c->d_ivar, d_images, d_chi2,
                                                       d_flags, nullptr, 0, d_params, nullptr, 0.0, 0.0, HaloArgs{nullptr, nullptr, nullptr, 0});
    c->launches += 2;
    return cudaGetLastError();
}
