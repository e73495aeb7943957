// fp64 mass model shared by quasar_kernel and the pixelated-source mapping kernel: per-vector constants and the deflection,
// Hessian and potential of (lambda x) EPL + external shear + point mass (+ dPIE sheet) at one sky position.
// Conventions: Eq. B.1-B.3, Eq. 49, Eq. 50-51 (DESIGN.md R-L3..6, R-Q4, R-S1..3).
#pragma once
#include <math.h>

#define QSO_MAX_TERMS 400

struct MassConst {
    double xl, yl, c, s, q, t, negf, bTM, pref0, sh_c, sh_s, bh;
    double lam, ms_rc, ms_rt, ms_a;     // internal mass sheet (R-S1..3): ms_a = (1 - lam) rc rt, 0 = none
    int nterms;
    bool epl, sheet;
};

struct MassEval { double ax, ay, hxx, hxy, hyy, psi; };

__device__ static inline void mass_const(const float* __restrict__ p, double lam, double rc, double rt, bool sheet, MassConst& m) {
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
__device__ static inline void mass_eval(const MassConst& m, double thx, double thy, MassEval& e) {
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

