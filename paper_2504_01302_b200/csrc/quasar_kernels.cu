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

#define QSO_LANES 8            // == GLAD_MAX_QIMG
#define QSO_NEWTON 12
#define QSO_MAX_TERMS 400
// days per (Mpc arcsec^2): (1 Mpc / c) / 86400 s * (pi/648000)^2
#define QSO_TDELAY_K (3.0856775814913673e22 / 299792458.0 / 86400.0 * (3.14159265358979323846 / 648000.0) * (3.14159265358979323846 / 648000.0))

struct MassConst {
    double xl, yl, c, s, q, t, negf, bTM, pref0, sh_c, sh_s, bh;
    double lam, ms_rc, ms_rt, ms_a;     // internal mass sheet (R-S1..3): ms_a = (1 - lam) rc rt, 0 = none
    int nterms;
    bool epl, sheet;
};

struct MassEval { double ax, ay, hxx, hxy, hyy, psi; };

__device__ static void mass_const(const float* __restrict__ p, double lam, double rc, double rt, bool sheet, MassConst& m) {
    m.lam = lam; m.sheet = sheet; m.ms_rc = rc; m.ms_rt = rt;
    m.ms_a = (1.0 - lam) * rc * rt;
    m.xl = p[0]; m.yl = p[1];
    const double thE = p[2], gam = p[3], q = p[4];
    sincos((double)p[5], &m.s, &m.c);
    m.q = q;
    m.t = gam - 1.0;
    const double f = (1.0 - q) / (1.0 + q);
    m.negf = -f;
    m.epl = thE > 0.0;
    m.bTM = q * pow(2.0 / (1.0 + q), 1.0 / m.t) * thE;        // b_TM = q b, b of Eq. B.3
    m.pref0 = lam * 2.0 * m.bTM / (1.0 + q);        // lam kappa_epl: alpha, Hessian and psi of the EPL all carry lam
    int nt = 0;
    if (f > 1e-17) {                                          // |a_n| <= f^n: terms until f^n < 1e-17
        const double est = ceil(log(1e-17) / log(f)) + 1.0;
        nt = (est > 0.0 && est < (double)QSO_MAX_TERMS) ? (int)est : QSO_MAX_TERMS;   // also for an invalid q (NaN)
    }
    m.nterms = nt;
    double s2, c2;
    sincos(2.0 * (double)p[7], &s2, &c2);
    m.sh_c = (double)p[6] * c2;
    m.sh_s = (double)p[6] * s2;
    m.bh = p[8];
}

// deflection, Hessian and potential of EPL + shear + point mass at the sky position (thx, thy)
__device__ static void mass_eval(const MassConst& m, double thx, double thy, MassEval& e) {
    const double dx = thx - m.xl, dy = thy - m.yl;
    double ax = 0.0, ay = 0.0, hxx = 0.0, hxy = 0.0, hyy = 0.0, psi = 0.0;
    if (m.epl) {
        const double x = dx * m.c + dy * m.s, y = dy * m.c - dx * m.s;
        double R2 = m.q * m.q * x * x + y * y;
        if (R2 < 1e-12) R2 = 1e-12;
        const double R = sqrt(R2), iR = 1.0 / R;
        const double wr = m.q * x * iR, wi = y * iR;
        const double zr = m.negf * (wr * wr - wi * wi), zi = m.negf * 2.0 * wr * wi;
        double ar = 1.0, ai = 0.0, sr = 1.0, si = 0.0;
        const double tt = 2.0 - m.t;
        for (int n = 1; n <= m.nterms; ++n) {
            const double cn = (2.0 * n - tt) / (2.0 * n + tt);
            const double nr = (ar * zr - ai * zi) * cn, ni = (ar * zi + ai * zr) * cn;
            ar = nr; ai = ni;
            sr += ar; si += ai;
        }
        const double u = m.bTM * iR;                       // b_TM / R_TM = b / R
        const double um = exp((m.t - 1.0) * log(u));       // (b/R)^(t-1)
        const double mag = m.pref0 * um;
        const double alr = mag * (wr * sr - wi * si), ali = mag * (wr * si + wi * sr);
        const double kap = m.lam * 0.5 * tt * um * u;      // lam x Eq. B.1: (2-t)/2 (b/R)^t
        double r2 = x * x + y * y;
        if (r2 < 1e-12) r2 = 1e-12;
        const double ir2 = 1.0 / r2;
        // gamma_c = [(1-t) alpha z - kappa z^2] / |z|^2
        const double azr = alr * x - ali * y, azi = alr * y + ali * x;
        const double z2r = x * x - y * y, z2i = 2.0 * x * y;
        const double g1 = ((1.0 - m.t) * azr - kap * z2r) * ir2, g2 = ((1.0 - m.t) * azi - kap * z2i) * ir2;
        const double lxx = kap + g1, lyy = kap - g1, lxy = g2;
        const double cc = m.c * m.c, ss = m.s * m.s, cs = m.c * m.s;
        hxx = cc * lxx - 2.0 * cs * lxy + ss * lyy;
        hyy = ss * lxx + 2.0 * cs * lxy + cc * lyy;
        hxy = cs * (lxx - lyy) + (cc - ss) * lxy;
        ax = alr * m.c - ali * m.s;
        ay = alr * m.s + ali * m.c;
        psi = (x * alr + y * ali) / tt;
    }
    // external shear, Eq. 49, origin at the lens centre (R-L5)
    ax += m.sh_c * dx + m.sh_s * dy;
    ay += m.sh_s * dx - m.sh_c * dy;
    hxx += m.sh_c; hyy -= m.sh_c; hxy += m.sh_s;
    psi += 0.5 * (m.sh_c * (dx * dx - dy * dy) + 2.0 * m.sh_s * dx * dy);
    // point mass (R-L6)
    double r2 = dx * dx + dy * dy;
    if (r2 < 1e-12) r2 = 1e-12;
    const double ir2 = 1.0 / r2;
    ax += m.bh * dx * ir2;
    ay += m.bh * dy * ir2;
    const double hb = m.bh * (dy * dy - dx * dx) * ir2 * ir2;
    hxx += hb; hyy -= hb;
    hxy -= 2.0 * m.bh * dx * dy * ir2 * ir2;
    psi += 0.5 * m.bh * log(r2);
    if (m.sheet) {
        // (1 - lam) S(R), S = dPIE of Eq. 50 normalised to S(0) = 1, every difference with (rt - rc) divided out:
        //   g = alpha_R/R = 2 a [1 + (rt+rc)/(ht+hc)] / ((hc+rc)(ht+rt)),  kappa = a (rt+rc) / ((ht+hc) hc ht),  a = (1-lam) rc rt
        //   Hessian = g I + 2 (kappa - g) x x^T / R^2 ;  psi = 2 a/(rt-rc) {[dc - rc log1p(dc/2rc)] - [dt - rt log1p(dt/2rt)]}, d = h - r
        const double rc = m.ms_rc, rt = m.ms_rt, R2 = dx * dx + dy * dy;
        const double hc = sqrt(R2 + rc * rc), ht = sqrt(R2 + rt * rt);
        const double g = 2.0 * m.ms_a * (1.0 + (rt + rc) / (ht + hc)) / ((hc + rc) * (ht + rt));
        const double kp = m.ms_a * (rt + rc) / ((ht + hc) * hc * ht);
        const double ee = R2 > 0.0 ? 2.0 * (kp - g) / R2 : 0.0;
        ax += g * dx; ay += g * dy;
        hxx += g + ee * dx * dx; hyy += g + ee * dy * dy; hxy += ee * dx * dy;
        const double dc = R2 / (hc + rc), dt = R2 / (ht + rt);
        psi += 2.0 * m.ms_a / (rt - rc) * ((dc - rc * log1p(dc / (2.0 * rc))) - (dt - rt * log1p(dt / (2.0 * rt))));
    }
    e.ax = ax; e.ay = ay; e.hxx = hxx; e.hxy = hxy; e.hyy = hyy; e.psi = psi;
}

__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = QSO_LANES / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, QSO_LANES);
    return v;
}

__global__ void __launch_bounds__(64) quasar_kernel(const float* __restrict__ lens, const float* __restrict__ ddt,
                                                    const float* __restrict__ lambda, double ms_rc, double ms_rt, int B,
                                                    const glad_quasar_data qd, float* __restrict__ chi2_img,
                                                    float* __restrict__ chi2_tmd, double* __restrict__ theta_pre,
                                                    double* __restrict__ dt_pre, double* __restrict__ beta_out) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    int b = gid / QSO_LANES;
    const int i = gid % QSO_LANES;
    const bool vec = b < B;          // whole 8-lane groups are in or out; keep every lane for the shuffles
    if (!vec) b = B - 1;
    const float* p = lens + (size_t)b * GLAD_NLENS;
    const double lam = lambda ? (double)lambda[b] : 1.0;
    const bool valid = (p[2] >= 0.f) && (p[3] > 1.f && p[3] < 3.f) && (p[4] > 0.f && p[4] <= 1.f) && (p[8] >= 0.f) && isfinite(lam);
    const bool img = i < qd.n_img;
    const double inf = __longlong_as_double(0x7ff0000000000000LL), nan = __longlong_as_double(0x7ff8000000000000LL);
    MassConst m;
    mass_const(p, lam, ms_rc, ms_rt, lambda != nullptr, m);
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
    quasar_kernel<<<(total + threads - 1) / threads, threads, 0, st>>>(d_lens, d_ddt, c->d_lambda, c->ms_rc, c->ms_rt, B, c->qso, d_chi2_img, d_chi2_tmd,
                                                                      d_theta_pre, d_dt_pre, d_beta);
    return cudaGetLastError();
}
