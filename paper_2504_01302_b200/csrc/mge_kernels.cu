// the step between the two halves of the joint model (Fig. 2) on the device.
//   mge1d_kernel      : 1-D multi-Gaussian expansion of a radial profile, Eq. 44-46 ("following
//                       Shajib (2019)"):  f(sigma) ~ sum_{n=0}^{2P} eta_n Re F(sigma chi_n)   (Eq. 45)
//                       A_n = w_n f(sigma_n) dln(sigma) / sqrt(2 pi), sigma_n log-spaced        (Eq. 46)
//                       The paper prints neither eta_n nor chi_n; reading R-M1 states the Euler-algorithm
//                       constants used (chi_n = sqrt(2 P ln10/3 + 2 pi i n), eta_n = (-1)^n 2 sqrt(2 pi) 10^(P/3) xi_n),
//                       R-M2 the trapezoid weights w_n.  fp64 throughout (the sum cancels 10^(P/3)-fold), fp32 rows out.
//   model_kernel      : R-M3 in one launch: from one lens vector + distances expand the luminous tracer (lens-light Sersic #1)
//                       and Sigma_crit * kappa_epl (Eq. 13, Eq. B.1-B.3), and write a copy of the lens
//                       vector whose lens[8] = theta_E,BH^2 follows M_BH and D_dt (Eq. 4).
// One CTA per parameter vector, one warp per Gaussian in turn, lane n = term n of the Euler sum (2P+1 <= 32).
#include <math.h>

#include "glad_internal.h"
#include "glad_special.cuh"

struct cplx { double re, im; };
// principal-branch z^a for real a
__device__ static cplx cpow_real(cplx z, double a) {
    const double r = hypot(z.re, z.im), th = atan2(z.im, z.re);
    const double m = exp(a * log(r));
    double s, c;
    sincos(a * th, &s, &c);
    return {m * c, m * s};
}
__device__ static cplx cexp_d(cplx z) {
    const double m = exp(z.re);
    double s, c;
    sincos(z.im, &s, &c);
    return {m * c, m * s};
}
#define MGE_PI 3.14159265358979323846

// Eq. 45's constants ("can be precomputed at the start"): built once per launch on the host, passed by value.
struct EulerConsts { double eta[31], chi_re[31], chi_im[31]; int P; };
static EulerConsts euler_consts(int P) {
    EulerConsts e;
    e.P = P;
    // xi_0 = 1/2, xi_n = 1 (1..P), xi_2P = 2^-P, xi_{2P-n} = xi_{2P-n+1} + 2^-P binom(P, n)
    double xi[31];
    const double tp = ldexp(1.0, -P);
    xi[0] = 0.5;
    for (int n = 1; n <= P; ++n) xi[n] = 1.0;
    xi[2 * P] = tp;
    double binom = 1.0;
    for (int n = 1; n < P; ++n) {
        binom = binom * (double)(P - n + 1) / (double)n;
        xi[2 * P - n] = xi[2 * P - n + 1] + tp * binom;
    }
    const double amp = 2.0 * sqrt(2.0 * MGE_PI) * pow(10.0, P / 3.0);
    for (int n = 0; n <= 2 * P; ++n) {
        e.eta[n] = ((n & 1) ? -amp : amp) * xi[n];
        // principal sqrt of a + i b with a > 0
        const double a = 2.0 * P * log(10.0) / 3.0, b = 2.0 * MGE_PI * n;
        const double r = hypot(a, b), re = sqrt(0.5 * (r + a));
        e.chi_re[n] = re; e.chi_im[n] = 0.5 * b / re;
    }
    return e;
}

// One profile of one vector: the n_gauss rows {A_n, sigma_n, q'} (Eq. 46).  Called by all warps of the CTA; warp w takes
// Gaussians w, w + nwarps, ..; lane n = term n of the Euler sum.  bn = Sersic b_n (unused for the EPL).
__device__ static void mge_rows(int kind, double p0, double p1, double p2, double qp, double bn, const EulerConsts& ec,
                                int n_gauss, double sigma_lo, double dln, float* __restrict__ out_rows, double scale = 1.0,
                                const double2* __restrict__ cse = nullptr, int ncse = 0) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int nterm = 2 * ec.P + 1;
    const double t = p2 - 1.0;
    const double bepl = kind == GLAD_PROFILE_EPL ? pow(2.0 / (1.0 + qp), 1.0 / t) * p1 : 0.0;   // Eq. B.3
    const double eta = lane < nterm ? ec.eta[lane] : 0.0, cre = lane < nterm ? ec.chi_re[lane] : 1.0,
                 cim = lane < nterm ? ec.chi_im[lane] : 0.0;
    for (int g = warp; g < n_gauss; g += nwarps) {
        const double sigma = sigma_lo * exp(dln * g);
        double term = 0.0;
        if (lane < nterm) {
            const cplx z = {sigma * cre, sigma * cim};
            double re;
            if (kind == GLAD_PROFILE_SERSIC) {
                const cplx w = cpow_real({z.re / p1, z.im / p1}, 1.0 / p2);
                re = p0 * cexp_d({-bn * (w.re - 1.0), -bn * w.im}).re;
            } else if (kind == GLAD_PROFILE_NFW_CSE) {
                // Eq. A.2-A.4 at complex radius: p0 sum A_i / (2 (s_i^2 + u^2)^(3/2)), u = z sqrt(q) / r_s
                const double k2 = qp / (p1 * p1);
                const cplx u2 = {k2 * (z.re * z.re - z.im * z.im), k2 * 2.0 * z.re * z.im};
                double acc = 0.0;
                for (int i = 0; i < ncse; ++i) {
                    const double2 t = cse[i];
                    acc += t.x * 0.5 * cpow_real({t.y * t.y + u2.re, u2.im}, -1.5).re;
                }
                re = p0 * acc;
            } else if (kind == GLAD_PROFILE_CHAMELEON) {
                // Eq. 47 at complex radius: p0/(1+q) [ (z^2 + a_c)^(-1/2) - (z^2 + a_t)^(-1/2) ], a = 4 w^2/(1+q)^2
                const double opq = 1.0 + qp, ac = 4.0 * p1 * p1 / (opq * opq), at = 4.0 * p2 * p2 / (opq * opq);
                const cplx z2 = {z.re * z.re - z.im * z.im, 2.0 * z.re * z.im};
                const cplx ic = cpow_real({z2.re + ac, z2.im}, -0.5), it = cpow_real({z2.re + at, z2.im}, -0.5);
                re = p0 / opq * (ic.re - it.re);
            } else {
                const double n2 = z.re * z.re + z.im * z.im;               // b/z = b conj(z)/|z|^2
                re = p0 * 0.5 * (3.0 - p2) * cpow_real({bepl * z.re / n2, -bepl * z.im / n2}, t).re;   // Eq. B.1
            }
            term = eta * re;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) term += __shfl_xor_sync(0xffffffffu, term, o);
        if (lane == 0) {
            const double w = (g == 0 || g == n_gauss - 1) ? 0.5 : 1.0;
            float* o3 = out_rows + (size_t)g * 3;
            o3[0] = (float)(scale * (w * term * dln / sqrt(2.0 * MGE_PI)));
            o3[1] = (float)sigma;
            o3[2] = (float)qp;
        }
    }
}

__global__ void __launch_bounds__(256) mge1d_kernel(int kind, const float* __restrict__ prof, int B, int n_gauss,
                                                    double sigma_lo, double dln, const __grid_constant__ EulerConsts ec,
                                                    const double2* __restrict__ cse, int ncse, float* __restrict__ mge) {
    __shared__ double s_bn;
    const int b = blockIdx.x;
    const float* p = prof + (size_t)b * GLAD_NPROF;
    const double p0 = p[0], p1 = p[1], p2 = p[2], qp = p[3];
    if (kind == GLAD_PROFILE_SERSIC) {
        if (threadIdx.x == 0) s_bn = sersic_bn(p2);
        __syncthreads();
    }
    mge_rows(kind, p0, p1, p2, qp, kind == GLAD_PROFILE_SERSIC ? s_bn : 0.0, ec, n_gauss, sigma_lo, dln,
             mge + (size_t)b * n_gauss * 3, 1.0, cse, ncse);
}

cudaError_t launch_mge1d(glad_ctx* c, int kind, const float* d_prof, int B, int n_gauss, float sigma_lo, float sigma_hi,
                         int P, float* d_mge) {
    ProfScope ps(c, GK_MGE);
    const double dln = log((double)sigma_hi / (double)sigma_lo) / (n_gauss - 1);
    const int warps = n_gauss < 8 ? n_gauss : 8;
    mge1d_kernel<<<B, 32 * warps, 0, c->stream>>>(kind, d_prof, B, n_gauss, (double)sigma_lo, dln, euler_consts(P), c->d_cse64, c->ncse, d_mge);
    return cudaGetLastError();
}

// G in (km/s)^2 pc / Msun (R-D1), c in km/s
#define MGE_G_NEWTON 0.004301
#define MGE_C_KMS 299792.458

// R-M3 in one launch: CTA per vector.  Thread 0 derives theta_E,BH^2 (Eq. 4), Sigma_crit (Eq. 13) and the Sersic b_n, the
// whole CTA copies the lens vector, then all warps expand the lens-light Sersic and Sigma_crit kappa_epl (Eq. 46).
__global__ void __launch_bounds__(256) model_kernel(const float* __restrict__ lens, const float* __restrict__ dyn,
                                                    const float* __restrict__ ddt, double zd, int B, int tracer_kind, int n_lum, double lum_lo,
                                                    double lum_dln, int n_mass, double mass_lo, double mass_dln,
                                                    const float* __restrict__ lambda, double ms_rc, double ms_rt, int ms_n, double ms_lo,
                                                    double ms_dln, const HaloArgs halo, int nf_n, double nf_lo, double nf_dln,
                                                    const __grid_constant__ EulerConsts ec, float* __restrict__ lens_out,
                                                    float* __restrict__ lum, float* __restrict__ mass) {
    __shared__ double s_bn, s_sc;
    const int b = blockIdx.x;
    const float* L = lens + (size_t)b * GLAD_NLENS;
    float* Lo = lens_out + (size_t)b * GLAD_NLENS;
    const double Ddt = ddt[b], Dd = dyn[(size_t)b * GLAD_NDYN + 1], Mbh = dyn[(size_t)b * GLAD_NDYN + 2];
    if (threadIdx.x < GLAD_NLENS && threadIdx.x != 8) Lo[threadIdx.x] = L[threadIdx.x];
    if (threadIdx.x == 0) {
        // Eq. 4: theta_E,BH^2 = 4 G M (1+z_d) / (c^2 D_dt), radians^2 -> arcsec^2
        const double asr = 648000.0 / MGE_PI;
        Lo[8] = (float)(4.0 * MGE_G_NEWTON * Mbh * (1.0 + zd) / (MGE_C_KMS * MGE_C_KMS * Ddt * 1e6) * asr * asr);
        // Eq. 13: Sigma_crit = c^2/(4 pi G) D_dt / ((1+z_d) D_d^2)  [Msun/pc^2, distances Mpc -> pc]; rounded to fp32 like a
        // profile row of glad_mge1d_batch
        s_sc = (double)(float)(MGE_C_KMS * MGE_C_KMS / (4.0 * MGE_PI * MGE_G_NEWTON) * (Ddt * 1e6) / ((1.0 + zd) * (Dd * 1e6) * (Dd * 1e6)));
        s_bn = tracer_kind == GLAD_PROFILE_SERSIC ? sersic_bn((double)L[18]) : 0.0;
    }
    __syncthreads();
    mge_rows(tracer_kind, L[16], L[17], L[18], L[19], s_bn, ec, n_lum, lum_lo, lum_dln, lum + (size_t)b * n_lum * 3);
    // internal mass sheet (Eq. 6, 12, 50; R-S1..3): Sigma_int = Sigma_crit [lam kappa_epl + (1 - lam) S(R)].  The EPL rows carry lam;
    // the round sheet (q' = 1) gets ms_n rows of its own after them: it is Eq. 47's shape at q = 1 with I_0/2 = Sigma_crit (1-lam)/(1/rc - 1/rt)
    const int nm_tot = n_mass + (lambda ? ms_n : 0) + (halo.nf ? nf_n : 0);
    const double lam = lambda ? (double)lambda[b] : 1.0;
    float* M = mass + (size_t)b * nm_tot * 3;
    mge_rows(GLAD_PROFILE_EPL, s_sc, L[2], L[3], L[4], 0.0, ec, n_mass, mass_lo, mass_dln, M, lam);
    if (lambda)
        mge_rows(GLAD_PROFILE_CHAMELEON, 2.0 * s_sc * (1.0 - lam) / (1.0 / ms_rc - 1.0 / ms_rt), ms_rc, ms_rt, 1.0, 0.0, ec, ms_n, ms_lo,
                 ms_dln, M + (size_t)n_mass * 3);
    // eNFW halo (Appendix A): Sigma_crit lam kappa_enfw, nf_n rows with q' = the halo's q after the EPL (and sheet) rows;
    // the halo is part of the lens mass, so it carries lam like the EPL (kappa_int,comp of P:380)
    if (halo.nf) {
        const float* nf = halo.nf + 4 * (size_t)b;
        mge_rows(GLAD_PROFILE_NFW_CSE, s_sc * (double)nf[0], (double)nf[1], 0.0, (double)nf[2], 0.0, ec, nf_n, nf_lo, nf_dln,
                 M + (size_t)(n_mass + (lambda ? ms_n : 0)) * 3, lam, halo.cse64, halo.ncse);
    }
}

cudaError_t launch_model(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, double zd, int B, int tracer_kind, int n_lum,
                         float lum_lo, float lum_hi, int n_mass, float mass_lo, float mass_hi, int P, float* d_lens_out,
                         float* d_lum, float* d_mass) {
    ProfScope ps(c, GK_MGE);
    const double ldln = log((double)lum_hi / (double)lum_lo) / (n_lum - 1), mdln = log((double)mass_hi / (double)mass_lo) / (n_mass - 1);
    const double sdln = (c->d_lambda && c->ms_n > 1) ? log(c->ms_hi / c->ms_lo) / (c->ms_n - 1) : 0.0;
    model_kernel<<<B, 256, 0, c->stream>>>(d_lens, d_dyn, d_ddt, zd, B, tracer_kind, n_lum, (double)lum_lo, ldln, n_mass, (double)mass_lo, mdln,
                                           c->d_lambda, c->ms_rc, c->ms_rt, c->ms_n, c->ms_lo, sdln, halo_args(c), c->nf_n, c->nf_lo,
                                           (c->d_enfw && c->nf_n > 1) ? log(c->nf_hi / c->nf_lo) / (c->nf_n - 1) : 0.0, euler_consts(P), d_lens_out, d_lum, d_mass);
    return cudaGetLastError();
}
