// the step between the two halves of the joint model (Fig. 2) on the device.
//   mge1d_kernel      : 1-D multi-Gaussian expansion of a radial profile, Eq. 44-46 ("following
//                       Shajib (2019)"):  f(sigma) ~ sum_{n=0}^{2P} eta_n Re F(sigma chi_n)   (Eq. 45)
//                       A_n = w_n f(sigma_n) dln(sigma) / sqrt(2 pi), sigma_n log-spaced        (Eq. 46)
//                       The paper prints neither eta_n nor chi_n; reading R-M1 states the Euler-algorithm
//                       constants used (chi_n = sqrt(2 P ln10/3 + 2 pi i n), eta_n = (-1)^n 2 sqrt(2 pi) 10^(P/3) xi_n),
//                       R-M2 the trapezoid weights w_n.  fp64 throughout (the sum cancels 10^(P/3)-fold), fp32 rows out.
//   model_prep_kernel : from one lens vector + distances build the profile rows of the luminous tracer (lens-light
//                       Sersic #1) and of Sigma_crit * kappa_epl (Eq. 13, Eq. B.1-B.3), and a copy of the
//                       lens vector whose lens[8] = theta_E,BH^2 follows M_BH and D_dt (Eq. 4)   (R-M3).
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
__device__ static cplx csqrt_d(cplx z) {                    // principal square root, Re >= 0
    const double r = hypot(z.re, z.im);
    const double a = sqrt(0.5 * (r + fabs(z.re)));
    const double b = 0.5 * z.im / a;
    return z.re >= 0.0 ? cplx{a, b} : cplx{fabs(b), copysign(a, z.im)};
}

#define MGE_PI 3.14159265358979323846

__global__ void __launch_bounds__(256) mge1d_kernel(int kind, const float* __restrict__ prof, int B, int n_gauss,
                                                    double sigma_lo, double dln, int P, float* __restrict__ mge) {
    __shared__ double s_eta[32];
    __shared__ double s_chi[64];
    __shared__ double s_bn;
    const int b = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nwarps = blockDim.x >> 5;
    const float* p = prof + (size_t)b * GLAD_NPROF;
    const double p0 = p[0], p1 = p[1], p2 = p[2], qp = p[3];
    if (tid == 0) {
        // xi_0 = 1/2, xi_n = 1 (1..P), xi_2P = 2^-P, xi_{2P-n} = xi_{2P-n+1} + 2^-P binom(P, n)
        double xi[32];
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
            s_eta[n] = ((n & 1) ? -amp : amp) * xi[n];
            const cplx chi = csqrt_d({2.0 * P * log(10.0) / 3.0, 2.0 * MGE_PI * n});
            s_chi[2 * n] = chi.re; s_chi[2 * n + 1] = chi.im;
        }
        s_bn = kind == GLAD_PROFILE_SERSIC ? sersic_bn(p2) : 0.0;
    }
    __syncthreads();
    const int nterm = 2 * P + 1;
    // EPL: b of Eq. B.3 and the amplitude of Eq. B.1
    const double t = p2 - 1.0;
    const double bepl = kind == GLAD_PROFILE_EPL ? pow(2.0 / (1.0 + qp), 1.0 / t) * p1 : 0.0;
    for (int g = warp; g < n_gauss; g += nwarps) {
        const double sigma = sigma_lo * exp(dln * g);
        double term = 0.0;
        if (lane < nterm) {
            const cplx z = {sigma * s_chi[2 * lane], sigma * s_chi[2 * lane + 1]};
            double re;
            if (kind == GLAD_PROFILE_SERSIC) {
                const cplx w = cpow_real({z.re / p1, z.im / p1}, 1.0 / p2);
                re = p0 * cexp_d({-s_bn * (w.re - 1.0), -s_bn * w.im}).re;
            } else {
                // (b/z)^t = conj-free form: b/z = b conj(z)/|z|^2
                const double n2 = z.re * z.re + z.im * z.im;
                re = p0 * 0.5 * (3.0 - p2) * cpow_real({bepl * z.re / n2, -bepl * z.im / n2}, t).re;
            }
            term = s_eta[lane] * re;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) term += __shfl_xor_sync(0xffffffffu, term, o);
        if (lane == 0) {
            const double w = (g == 0 || g == n_gauss - 1) ? 0.5 : 1.0;
            float* out = mge + ((size_t)b * n_gauss + g) * 3;
            out[0] = (float)(w * term * dln / sqrt(2.0 * MGE_PI));
            out[1] = (float)sigma;
            out[2] = (float)qp;
        }
    }
}

cudaError_t launch_mge1d(glad_ctx* c, int kind, const float* d_prof, int B, int n_gauss, float sigma_lo, float sigma_hi,
                         int P, float* d_mge) {
    ProfScope ps(c, GK_MGE);
    const double dln = log((double)sigma_hi / (double)sigma_lo) / (n_gauss - 1);
    const int warps = n_gauss < 8 ? n_gauss : 8;
    mge1d_kernel<<<B, 32 * warps, 0, c->stream>>>(kind, d_prof, B, n_gauss, (double)sigma_lo, dln, P, d_mge);
    return cudaGetLastError();
}

// G in (km/s)^2 pc / Msun (R-D1), c in km/s
#define MGE_G_NEWTON 0.004301
#define MGE_C_KMS 299792.458

__global__ void model_prep_kernel(const float* __restrict__ lens, const float* __restrict__ dyn, const float* __restrict__ ddt,
                                  double zd, int B, float* __restrict__ lens_out, float* __restrict__ prof_lum,
                                  float* __restrict__ prof_mass) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const float* L = lens + (size_t)b * GLAD_NLENS;
    float* Lo = lens_out + (size_t)b * GLAD_NLENS;
    for (int i = 0; i < GLAD_NLENS; ++i) Lo[i] = L[i];
    const double Ddt = ddt[b], Dd = dyn[(size_t)b * GLAD_NDYN + 1], Mbh = dyn[(size_t)b * GLAD_NDYN + 2];
    // Eq. 4: theta_E,BH^2 = 4 G M (1+z_d) / (c^2 D_dt), radians^2 -> arcsec^2
    const double asr = 648000.0 / MGE_PI;
    Lo[8] = (float)(4.0 * MGE_G_NEWTON * Mbh * (1.0 + zd) / (MGE_C_KMS * MGE_C_KMS * Ddt * 1e6) * asr * asr);
    // Eq. 13: Sigma_crit = c^2/(4 pi G) D_dt / ((1+z_d) D_d^2)  [Msun/pc^2, distances Mpc -> pc]
    const double sc = MGE_C_KMS * MGE_C_KMS / (4.0 * MGE_PI * MGE_G_NEWTON) * (Ddt * 1e6) / ((1.0 + zd) * (Dd * 1e6) * (Dd * 1e6));
    float* pl = prof_lum + (size_t)b * GLAD_NPROF;
    float* pm = prof_mass + (size_t)b * GLAD_NPROF;
    pl[0] = L[16]; pl[1] = L[17]; pl[2] = L[18]; pl[3] = L[19];          // lens-light Sersic #1: I_e, R_e, n, q
    pm[0] = (float)sc; pm[1] = L[2]; pm[2] = L[3]; pm[3] = L[4];          // Sigma_crit, theta_E, gamma, q
}

cudaError_t launch_model_prep(glad_ctx* c, const float* d_lens, const float* d_dyn, const float* d_ddt, double zd, int B,
                              float* d_lens_out, float* d_prof_lum, float* d_prof_mass) {
    ProfScope ps(c, GK_MGE);
    model_prep_kernel<<<(B + 127) / 128, 128, 0, c->stream>>>(d_lens, d_dyn, d_ddt, zd, B, d_lens_out, d_prof_lum, d_prof_mass);
    return cudaGetLastError();
}
