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
    // eNFW halo through core-steep ellipsoids (Appendix A; DESIGN.md R-N1..3): amp = rho_s r_s / sqrt(q), sc = sqrt(q) / r_s
    bool halo, halo_ok;
    double nf_rho, nf_amp, nf_sc, nf_q, nf_c, nf_s, nf_psi;
    const double2* cse;
    int ncse;
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

// per-vector halo constants; nf = {rho_s, r_s, q, phi} (NULL = none).  halo_ok = the vector's halo parameters are valid.
__device__ static inline void mass_const_halo(const float* __restrict__ nf, const double2* cse, int ncse, MassConst& m) {
    m.halo = false; m.halo_ok = true; m.cse = cse; m.ncse = ncse;
    if (!nf) return;
    const double rho = nf[0], rs = nf[1], q = nf[2];
    m.halo_ok = (rho >= 0.0) && (rho == 0.0 || (rs > 0.0 && q > 0.0 && q <= 1.0));
    if (!(rho > 0.0) || !m.halo_ok) return;
    m.halo = true;
    m.nf_rho = rho; m.nf_q = q;
    m.nf_amp = rho * rs / sqrt(q);
    m.nf_sc = sqrt(q) / rs;
    m.nf_psi = rho * rs * rs / q;
    sincos((double)nf[3], &m.nf_s, &m.nf_c);
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
    if (m.halo) {
        // kappa = rho_s sum A_i / (2 (s_i^2 + u^2)^(3/2)) (Eq. A.3-A.4); psi_CSE = q/(2s) ln Psi - q/s ln((1+q)s) (Eq. A.6),
        // Psi = (psi_s + s)^2 + (1-q^2) X^2, psi_s = sqrt(q^2 (s^2 + X^2) + Y^2), (X, Y) = sc x (halo-frame offset)
        const double q = m.nf_q, q2 = q * q;
        const double xh = dx * m.nf_c + dy * m.nf_s, yh = dy * m.nf_c - dx * m.nf_s;
        const double X = m.nf_sc * xh, Y = m.nf_sc * yh;
        double aX = 0.0, aY = 0.0, hXX = 0.0, hXY = 0.0, hYY = 0.0, ps = 0.0;
        for (int i = 0; i < m.ncse; ++i) {
            const double2 t = m.cse[i];
            const double A = t.x, si = t.y;
            const double pss = sqrt(q2 * (si * si + X * X) + Y * Y), ip = 1.0 / pss, a = pss + si;
            const double Psi = a * a + (1.0 - q2) * X * X, iP = 1.0 / Psi;
            const double sX = q2 * X * ip, sY = Y * ip;
            const double sXX = q2 * ip - sX * sX * ip, sYY = ip - sY * sY * ip, sXY = -sX * sY * ip;
            const double PX = 2.0 * a * sX + 2.0 * (1.0 - q2) * X, PY = 2.0 * a * sY;
            const double PXX = 2.0 * sX * sX + 2.0 * a * sXX + 2.0 * (1.0 - q2), PYY = 2.0 * sY * sY + 2.0 * a * sYY,
                         PXY = 2.0 * sX * sY + 2.0 * a * sXY;
            const double f = A * q / (2.0 * si);
            aX += f * PX * iP; aY += f * PY * iP;
            hXX += f * (PXX * iP - PX * PX * iP * iP);
            hYY += f * (PYY * iP - PY * PY * iP * iP);
            hXY += f * (PXY * iP - PX * PY * iP * iP);
            ps += A * (q / (2.0 * si) * log(Psi) - q / si * log((1.0 + q) * si));
        }
        const double c = m.nf_c, s = m.nf_s;
        ax += m.nf_amp * (aX * c - aY * s);
        ay += m.nf_amp * (aX * s + aY * c);
        hxx += m.nf_rho * (c * c * hXX - 2.0 * c * s * hXY + s * s * hYY);
        hyy += m.nf_rho * (s * s * hXX + 2.0 * c * s * hXY + c * c * hYY);
        hxy += m.nf_rho * (c * s * (hXX - hYY) + (c * c - s * s) * hXY);
        psi += m.nf_psi * ps;
    }
    e.ax = ax; e.ay = ay; e.hxx = hxx; e.hxy = hxy; e.hyy = hyy; e.psi = psi;
}

