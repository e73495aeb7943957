// Quasar terms of libglad for sm_100a (quasar part): chi^2_img (Eq. 35) and chi^2_tmd (Eq. 36)
// of the lensed point source, from the Fermat potential of Eq. 1-4.  The paper keeps these two terms on the CPU (P:265-267:
// 4 images, < 0.1 s); in a batched sampler they are one more per-vector reduction, so they run here beside the lens half.
//   quasar_kernel : 8 lanes per parameter vector, lane = image.  All arithmetic fp64 (a few thousand instructions per lane; the
//                   Newton steps amplify rounding near critical curves, and nothing here is throughput-bound).
//     1. beta_i = theta_i - alpha(theta_i) (Eq. 33), mu_i = 1/det(I - Hessian psi), beta_bar = sum |mu_i| beta_i / sum |mu_i|   (R-Q1)
//     2. theta_i^pre: QSO_NEWTON Newton steps on theta - alpha(theta) = beta_bar from theta_i                                  (R-Q2)
//     3. chi2_img = sum |theta_i - theta_i^pre|^2 / sigma_i^2 ; phi_i = |theta_i^pre - beta_bar|^2/2 - psi(theta_i^pre) (Eq. 2);
//        dt_i = K D_dt (phi_i - phi_ref) (Eq. 3-4, R-Q3/R-Q5) ; chi2_tmd = sum (dt_obs,i - dt_i)^2 / sigma_dt,i^2
//   psi and its Hessian for the EPL follow from the homogeneity of kappa (Eq. B.1) -- DESIGN.md R-Q4:
//     psi = (x alpha_x + y alpha_y)/(2-t);  gamma_1 + i gamma_2 = [(1-t) alpha z - kappa z^2]/|z|^2 (z = x + iy, lens frame).
#include <math.h>

#include "glad_internal.h"
#include "glad_mass_fp64.cuh"

#define QSO_LANES 8            // == GLAD_MAX_QIMG
#define QSO_NEWTON 12
// days per (Mpc arcsec^2): (1 Mpc / c) / 86400 s * (pi/648000)^2
#define QSO_TDELAY_K (3.0856775814913673e22 / 299792458.0 / 86400.0 * (3.14159265358979323846 / 648000.0) * (3.14159265358979323846 / 648000.0))

__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = QSO_LANES / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, QSO_LANES);
    return v;
}

__global__ void __launch_bounds__(64) quasar_kernel(const float* __restrict__ lens, const float* __restrict__ ddt,
                                                    const float* __restrict__ lambda, double ms_rc, double ms_rt, const HaloArgs halo,
                                                    int B, const glad_quasar_data qd, float* __restrict__ chi2_img,
                                                    float* __restrict__ chi2_tmd, double* __restrict__ theta_pre,
                                                    double* __restrict__ dt_pre, double* __restrict__ beta_out) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    int b = gid / QSO_LANES;
    const int i = gid % QSO_LANES;
    const bool vec = b < B;          // whole 8-lane groups are in or out; keep every lane for the shuffles
    if (!vec) b = B - 1;
    const float* p = lens + (size_t)b * GLAD_NLENS;
    const double lam = lambda ? (double)lambda[b] : 1.0;
    bool valid = (p[2] >= 0.f) && (p[3] > 1.f && p[3] < 3.f) && (p[4] > 0.f && p[4] <= 1.f) && (p[8] >= 0.f) && isfinite(lam);
    const bool img = i < qd.n_img;
    const double inf = __longlong_as_double(0x7ff0000000000000LL), nan = __longlong_as_double(0x7ff8000000000000LL);
    MassConst m;
    mass_const(p, lam, ms_rc, ms_rt, lambda != nullptr, m);
    mass_const_halo(halo.nf ? halo.nf + 4 * (size_t)b : nullptr, halo.cse64, halo.ncse, m);
    valid = valid && m.halo_ok;
    const int ii = img ? i : 0;
    const double ox = qd.theta[2 * ii], oy = qd.theta[2 * ii + 1];
    MassEval e;
    // 1. source-plane positions and magnification weights
    mass_eval(m, ox, oy, e);
    double w = fabs(1.0 / ((1.0 - e.hxx) * (1.0 - e.hyy) - e.hxy * e.hxy));
    if (!img) w = 0.0;
    const double wsum = group_sum(w);
    const double bx = group_sum(w * (ox - e.ax)) / wsum, by = group_sum(w * (oy - e.ay)) / wsum;
    // 2. back to the image plane
    double tx = ox, ty = oy;
    for (int it = 0; it < QSO_NEWTON; ++it) {
        if (it > 0) mass_eval(m, tx, ty, e);
        const double fx = tx - e.ax - bx, fy = ty - e.ay - by;
        const double a11 = 1.0 - e.hxx, a12 = -e.hxy, a22 = 1.0 - e.hyy;
        const double idet = 1.0 / (a11 * a22 - a12 * a12);
        tx -= (a22 * fx - a12 * fy) * idet;
        ty -= (a11 * fy - a12 * fx) * idet;
    }
    mass_eval(m, tx, ty, e);
    // 3. chi^2 terms
    const double ex = ox - tx, ey = oy - ty;
    const double c2i = group_sum(img ? (ex * ex + ey * ey) * qd.ivar_theta[ii] : 0.0);
    const double phi = 0.5 * ((tx - bx) * (tx - bx) + (ty - by) * (ty - by)) - e.psi;
    const double phi_ref = __shfl_sync(0xffffffffu, phi, qd.ref, QSO_LANES);
    const double dt = QSO_TDELAY_K * (double)ddt[b] * (phi - phi_ref);
    const double r = qd.dt_obs[ii] - dt;
    const double c2t = group_sum((img && i != qd.ref) ? r * r * qd.ivar_dt[ii] : 0.0);
    if (!vec) return;              // after the last shuffle: no lane leaves a warp early
    // an invalid mass model (same test as lens_prep_kernel) went through the arithmetic with whatever it produced
    // (every loop is bounded); its outputs are chi2 = +inf, NaN positions and delays
    if (img) {
        if (theta_pre) { theta_pre[((size_t)b * qd.n_img + i) * 2] = valid ? tx : nan; theta_pre[((size_t)b * qd.n_img + i) * 2 + 1] = valid ? ty : nan; }
        if (dt_pre) dt_pre[(size_t)b * qd.n_img + i] = valid ? dt : nan;
    }
    if (i == 0) {
        if (chi2_img) chi2_img[b] = valid ? (float)c2i : (float)inf;
        if (chi2_tmd) chi2_tmd[b] = valid ? (float)c2t : (float)inf;
        if (beta_out) { beta_out[2 * b] = valid ? bx : nan; beta_out[2 * b + 1] = valid ? by : nan; }
    }
}

cudaError_t launch_quasar(glad_ctx* c, cudaStream_t st, const float* d_lens, const float* d_ddt, int B, float* d_chi2_img,
                          float* d_chi2_tmd, double* d_theta_pre, double* d_dt_pre, double* d_beta) {
    ProfScope ps(c, GK_QUASAR, st);
    const int threads = 64, total = B * QSO_LANES;
    quasar_kernel<<<(total + threads - 1) / threads, threads, 0, st>>>(d_lens, d_ddt, c->d_lambda, c->ms_rc, c->ms_rt, halo_args(c), B, c->qso, d_chi2_img, d_chi2_tmd,
                                                                      d_theta_pre, d_dt_pre, d_beta);
    return cudaGetLastError();
}
