/*
 * glad_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU statement of what the batched joint
 * lensing + dynamics log-likelihood computes (arXiv 2504.01302, "GLaD").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path in paper_2504_01302_b200/csrc.
 *
 * Citations: "P:n" = /root/reference/PAPER.md line n.  Where the paper prints
 * no formula the reading taken is listed in DESIGN.md ("Readings").
 *
 * No blocking, fusion, symmetry or separability is used anywhere: every ray,
 * every PSF tap and every (node, mass Gaussian, luminous Gaussian, pixel)
 * quadrature term is evaluated exactly as the formulas are written, in fp64.
 * The only parallelism is an OpenMP `parallel for` over batch elements.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   EPL deflection ........ SIE closed form, kappa = div(alpha)/2 by finite
 *                           differences vs Eq. B.1-B.3, curl = 0, alpha(theta_E)
 *                           = theta_E at q = 1
 *   shear, point mass ..... analytic; kappa = 0 by finite differences
 *   Sersic ................ b_n vs scipy.special.gammaincinv, n = 1/2 Gaussian,
 *                           total flux closed form
 *   image / PSF / chi2 .... SIS ring, delta image, flux conservation, chi2 = k^2 N
 *   JAM second moment ..... brute-force spherical Jeans, brute-force axisymmetric
 *                           Jeans (anisotropic, inclined), Keplerian point mass,
 *                           inclination independence, evenness, linearity
 *   PSF / bins (kin) ...... constant-field invariance, delta kernel
 *   joint ................. additivity, -inf propagation
 *   Chameleon light ....... total flux closed form, w_t -> inf cored isothermal,
 *                           Eq. 47 on the axes, = Sersic-free image pipeline
 *   1-D MGE (8(f) rank 1) . power-law closed form, Gaussian profile, profiles
 *                           summed back to the paper's ~0.5 %, linearity
 * Overall numbers: PARITY UNPINNED against any published value -- the paper
 * prints no model image, v_rms map or likelihood value for any parameter
 * vector.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_NLENS 26
#define ORACLE_NDYN 4

/* flag bits (same meaning as include/glad.h, restated, not included) */
#define FLAG_LENS_INVALID 1
#define FLAG_DYN_INVALID 2
#define FLAG_BIN_INVALID 4

static const double PI = 3.14159265358979323846;
/* G in (km/s)^2 pc / Msun -- paper silent; reading R-D1 */
static const double G_NEWTON = 0.004301;
/* BH Gaussian width in arcsec = the paper's central softening scale */
static const double SIGMA_BH_ARCSEC = 0.01;

int glad_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------ */
/* Sersic b_n: exact root of P(2n, b) = 1/2 (regularised lower incomplete    */
/* gamma).  DESIGN.md reading R-L7 (paper names Sersic only).         */
/* ------------------------------------------------------------------------ */
static double gammainc_P(double a, double x) {
    if (x <= 0.0) return 0.0;
    if (x < a + 1.0) { /* series: P = x^a e^-x / Gamma(a+1) * sum x^n / (a+1)...(a+n) */
        double term = 1.0 / a, sum = term, ap = a;
        for (int n = 0; n < 100000; ++n) {
            ap += 1.0;
            term *= x / ap;
            sum += term;
            if (fabs(term) < fabs(sum) * 1e-17) break;
        }
        return sum * exp(-x + a * log(x) - lgamma(a));
    }
    /* continued fraction for Q = 1 - P (modified Lentz) */
    double tiny = 1e-300, b = x + 1.0 - a, c = 1.0 / tiny, d = 1.0 / b, h = d;
    for (int i = 1; i < 100000; ++i) {
        double an = -i * (i - a);
        b += 2.0;
        d = an * d + b; if (fabs(d) < tiny) d = tiny;
        c = b + an / c; if (fabs(c) < tiny) c = tiny;
        d = 1.0 / d;
        double del = d * c;
        h *= del;
        if (fabs(del - 1.0) < 1e-16) break;
    }
    return 1.0 - exp(-x + a * log(x) - lgamma(a)) * h;
}

double glad_oracle_sersic_bn(double n) {
    double a = 2.0 * n, lo = 0.0, hi = 2.0 * n + 20.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (gammainc_P(a, mid) < 0.5) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* Elliptical Sersic, paper's elliptical radius R = sqrt(x^2 + y^2/q^2)
 * (footnote P:234, Eq. B.2); (dx,dy) already relative to the centre. */
double glad_oracle_sersic(double dx, double dy, double Ie, double Re, double n, double q,
                          double phi, double bn) {
    double c = cos(phi), s = sin(phi);
    double x = dx * c + dy * s, y = -dx * s + dy * c;
    double R = sqrt(x * x + y * y / (q * q));
    return Ie * exp(-bn * (pow(R / Re, 1.0 / n) - 1.0));
}

/* ------------------------------------------------------------------------ */
/* EPL deflection in the lens frame (major axis on x).  Paper convention      */
/* App. B Eq. B.1-B.3; deflection "following Tessore & Metcalf    */
/* (2015)", formula restated in DESIGN.md reading R-L3:               */
/*   R_TM = sqrt(q^2 x^2 + y^2), b_TM = q b, b = (2/(1+q))^(1/(gamma-1)) th_E */
/*   w = (q x + i y)/R_TM, t = gamma-1, f = (1-q)/(1+q)                       */
/*   alpha = 2 b_TM/(1+q) (b_TM/R_TM)^(t-1) w sum_n a_n,                      */
/*   a_0 = 1, a_n = a_{n-1} (-f w^2) (2n-(2-t))/(2n+(2-t))                    */
/* Singular (r_soft = 0), R_TM^2 clamped below at (1e-6)^2.                   */
/* ------------------------------------------------------------------------ */
void glad_oracle_epl_alpha(double x, double y, double thetaE, double gamma, double q,
                           double* ax, double* ay) {
    double t = gamma - 1.0;
    if (thetaE == 0.0) { *ax = 0.0; *ay = 0.0; return; } /* no mass: kappa = 0 everywhere */
    double b = pow(2.0 / (1.0 + q), 1.0 / t) * thetaE;
    double bTM = q * b;
    double R2 = q * q * x * x + y * y;
    if (R2 < 1e-12) R2 = 1e-12;
    double R = sqrt(R2);
    double complex w = (q * x + I * y) / R;
    double f = (1.0 - q) / (1.0 + q);
    double complex z = -f * w * w, an = 1.0, sum = 1.0;
    for (int n = 1; n <= 500; ++n) {
        an *= z * (2.0 * n - (2.0 - t)) / (2.0 * n + (2.0 - t));
        sum += an;
        if (cabs(an) < 1e-16) break;
    }
    double complex alpha = 2.0 * bTM / (1.0 + q) * pow(bTM / R, t - 1.0) * w * sum;
    *ax = creal(alpha);
    *ay = cimag(alpha);
}

/* ------------------------------------------------------------------------ */
/* Internal mass sheet, Eq. 6 with the dPIE profile of Eq. 50-51       */
/* in place of the constant sheet -- DESIGN.md readings R-S1..3:  */
/*   kappa_int = (1 - lam) S(R) + lam kappa_epl + kappa_BH   (shear outside)  */
/*   S(R) = [1/sqrt(R^2+rc^2) - 1/sqrt(R^2+rt^2)] / (1/rc - 1/rt),  S(0) = 1,  */
/*   R^2 = x^2 + y^2 about the lens centre; lam = the constant of Eq. 51.     */
/* For kappa = A/sqrt(R^2+s^2) (circular): alpha_R = 2A (h - s)/R, h = sqrt(R^2+s^2)*/
/* (mean convergence inside R), psi = 2A [(h - s) - s ln((s+h)/2s)] (psi(0)=0),*/
/* Hessian = g I + 2 (kappa - g) x x^T / R^2 with g = alpha_R/R.              */
/* long double: rc = 45", rt = 45.09" make every term a small difference.     */
/* ------------------------------------------------------------------------ */
static void sheet_terms(double lam, double rc, double rt, double dx, double dy, double* ax, double* ay,
                        double* h, double* psi, double* kap) {
    /* every term is a difference of two nearly equal numbers (rt - rc << rc): written with h - s = R^2/(h + s),
     * 1/hc - 1/ht = (rt^2 - rc^2)/((ht + hc) hc ht) and log1p so that nothing is lost for any rc, rt */
    long double c = rc, t = rt, A = (1.0L - (long double)lam) * c * t / (t - c);      /* (1-lam)/(1/rc - 1/rt) */
    long double x = dx, y = dy, R2 = x * x + y * y;
    long double hc = sqrtl(R2 + c * c), ht = sqrtl(R2 + t * t);
    long double k = A * (t * t - c * c) / ((ht + hc) * hc * ht);                      /* Eq. 50 */
    long double g = 2.0L * A * (1.0L / (hc + c) - 1.0L / (ht + t));                   /* alpha_R / R */
    if (ax) *ax = (double)(g * x);
    if (ay) *ay = (double)(g * y);
    if (kap) *kap = (double)k;
    if (h) {
        long double e = (R2 > 0.0L) ? 2.0L * (k - g) / R2 : 0.0L;
        h[0] = (double)(g + e * x * x);
        h[1] = (double)(e * x * y);
        h[2] = (double)(g + e * y * y);
    }
    if (psi) {
        long double dc = R2 / (hc + c), dt = R2 / (ht + t);                           /* h - s */
        *psi = (double)(2.0L * A * ((dc - c * log1pl(dc / (2.0L * c))) - (dt - t * log1pl(dt / (2.0L * t)))));
    }
}

double glad_oracle_sheet_kappa(double lam, double rc, double rt, double dx, double dy) {
    double k;
    sheet_terms(lam, rc, rt, dx, dy, NULL, NULL, NULL, NULL, &k);
    return k;
}

/* ------------------------------------------------------------------------ */
/* SURVEY.md 8(f) rank 4, mass part: elliptical NFW halo through core-steep    */
/* ellipsoids (Appendix A, Eq. A.1-A.7).                            */
/*   kappa_enfw(x,y) = rho_s sum_i A_i kappa_CSE(u; s_i)              (Eq. A.3) */
/*   kappa_CSE(u; s) = 1 / (2 (s^2 + u^2)^(3/2))                      (Eq. A.4) */
/*   u^2 = X^2 + Y^2/q^2, (X, Y) = (sqrt(q)/r_s) (x, y) in the halo frame (A.2) */
/*   psi_CSE(X,Y) = q/(2s) ln Psi - q/s ln[(1+q) s]                   (Eq. A.6) */
/*   Psi = (psi_s + s)^2 + (1-q^2) X^2, psi_s = sqrt(q^2 (s^2 + X^2) + Y^2)     */
/*   (Psi: Oguri 2021, not printed in the paper; pinned here by Poisson's       */
/*   equation, Eq. 7: Laplacian psi_CSE = 2 kappa_CSE by finite differences).   */
/* Amplitudes follow from Eq. 7 and the scaling of Eq. A.2 (reading R-N2: the   */
/* prefactor printed in Eq. A.7 is not consistent with Eq. A.3 by one power of  */
/* r_s): psi = (rho_s r_s^2 / q) sum A_i psi_CSE, alpha = (rho_s r_s/sqrt q)    */
/* sum A_i grad psi_CSE, Hessian = rho_s sum A_i Hess psi_CSE.                  */
/* The table (A_i, s_i) is an INPUT of the method ("predetermined";      */
/* reading R-N1): set once with glad_oracle_set_cse_table.                      */
/* Halo vector nf = {rho_s, r_s [arcsec], q, phi}; centre = lens centre;        */
/* rho_s = 0 switches the halo off.                                             */
/* ------------------------------------------------------------------------ */
#define ORACLE_MAX_CSE 128
static int g_ncse = 0;
static double g_cse_A[ORACLE_MAX_CSE], g_cse_s[ORACLE_MAX_CSE];
int glad_oracle_set_cse_table(int n, const double* A, const double* s) {
    if (n < 0 || n > ORACLE_MAX_CSE) return -1;
    g_ncse = n;
    for (int i = 0; i < n; ++i) { g_cse_A[i] = A[i]; g_cse_s[i] = s[i]; }
    return 0;
}
/* Eq. A.1 with rho_s = 1 */
double glad_oracle_nfw_kappa(double u) {
    if (u < 1.0) { double t = sqrt(1.0 - u * u); return 0.5 / (u * u - 1.0) * (1.0 - atanh(t) / t); }
    if (u > 1.0) { double t = sqrt(u * u - 1.0); return 0.5 / (u * u - 1.0) * (1.0 - atan(t) / t); }
    return 1.0 / 6.0;
}
/* kappa, alpha, Hessian (h[0..2] = xx, xy, yy) and psi of the halo at offset (dx, dy) from its centre, sky frame;
 * any output may be NULL */
void glad_oracle_enfw(const double* nf, double dx, double dy, double* kappa, double* ax, double* ay, double* h, double* psi) {
    double rho = nf[0], rs = nf[1], q = nf[2], c = cos(nf[3]), s = sin(nf[3]);
    double xh = dx * c + dy * s, yh = -dx * s + dy * c;          /* halo frame */
    double sc = sqrt(q) / rs, X = sc * xh, Y = sc * yh;
    double k = 0.0, aX = 0.0, aY = 0.0, hXX = 0.0, hXY = 0.0, hYY = 0.0, ps = 0.0;
    for (int i = 0; i < g_ncse; ++i) {
        double A = g_cse_A[i], si = g_cse_s[i];
        double u2 = X * X + Y * Y / (q * q);
        k += A * 0.5 / pow(si * si + u2, 1.5);
        double pss = sqrt(q * q * (si * si + X * X) + Y * Y), a = pss + si;
        double Psi = a * a + (1.0 - q * q) * X * X;
        double sX = q * q * X / pss, sY = Y / pss;               /* d psi_s */
        double sXX = q * q / pss - q * q * q * q * X * X / (pss * pss * pss), sYY = 1.0 / pss - Y * Y / (pss * pss * pss),
               sXY = -q * q * X * Y / (pss * pss * pss);
        double PX = 2.0 * a * sX + 2.0 * (1.0 - q * q) * X, PY = 2.0 * a * sY;
        double PXX = 2.0 * sX * sX + 2.0 * a * sXX + 2.0 * (1.0 - q * q), PYY = 2.0 * sY * sY + 2.0 * a * sYY,
               PXY = 2.0 * sX * sY + 2.0 * a * sXY;
        double f = A * q / (2.0 * si);
        aX += f * PX / Psi;
        aY += f * PY / Psi;
        hXX += f * (PXX / Psi - PX * PX / (Psi * Psi));
        hYY += f * (PYY / Psi - PY * PY / (Psi * Psi));
        hXY += f * (PXY / Psi - PX * PY / (Psi * Psi));
        ps += A * (q / (2.0 * si) * log(Psi) - q / si * log((1.0 + q) * si));
    }
    double amp = rho * rs / sqrt(q);
    if (kappa) *kappa = rho * k;
    if (ax) *ax = amp * (aX * c - aY * s);
    if (ay) *ay = amp * (aX * s + aY * c);
    if (h) {
        h[0] = rho * (c * c * hXX - 2.0 * c * s * hXY + s * s * hYY);
        h[2] = rho * (s * s * hXX + 2.0 * c * s * hXY + c * c * hYY);
        h[1] = rho * (c * s * (hXX - hYY) + (c * c - s * s) * hXY);
    }
    if (psi) *psi = rho * rs * rs / q * ps;
}
static int enfw_valid(const double* nf) {
    if (!(nf[0] >= 0.0)) return 0;
    if (nf[0] == 0.0) return 1;
    return (nf[1] > 0.0) && (nf[2] > 0.0) && (nf[2] <= 1.0);
}

/* Total deflection at image-plane position (thx, thy): lam * EPL (rotated by phi_PA
 * about the lens centre) + external shear (Eq. 49, origin = lens centre,
 * reading R-L5) + point mass alpha = thE2 * D/|D|^2 (reading R-L6) + the mass
 * sheet (rc > 0; rc <= 0 = no sheet, lam must then be 1). */
void glad_oracle_deflection_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy,
                                 double* ax, double* ay);
void glad_oracle_deflection_sheet(const double* p, double lam, double rc, double rt, double thx, double thy,
                                  double* ax, double* ay) {
    glad_oracle_deflection_halo(p, lam, rc, rt, NULL, thx, thy, ax, ay);
}
/* ... + the eNFW halo nf = {rho_s, r_s, q, phi} about the lens centre (NULL or rho_s = 0: none) */
void glad_oracle_deflection_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy,
                                 double* ax, double* ay) {
    double dx = thx - p[0], dy = thy - p[1];
    double c = cos(p[5]), s = sin(p[5]);
    double xl = dx * c + dy * s, yl = -dx * s + dy * c;
    double axl, ayl;
    glad_oracle_epl_alpha(xl, yl, p[2], p[3], p[4], &axl, &ayl);
    double a_x = lam * (axl * c - ayl * s), a_y = lam * (axl * s + ayl * c);
    double c2 = cos(2.0 * p[7]), s2 = sin(2.0 * p[7]);
    a_x += p[6] * (dx * c2 + dy * s2);
    a_y += p[6] * (dx * s2 - dy * c2);
    double r2 = dx * dx + dy * dy;
    if (r2 < 1e-12) r2 = 1e-12;
    a_x += p[8] * dx / r2;
    a_y += p[8] * dy / r2;
    if (rc > 0.0) {
        double sx, sy;
        sheet_terms(lam, rc, rt, dx, dy, &sx, &sy, NULL, NULL, NULL);
        a_x += sx;
        a_y += sy;
    }
    if (nf && nf[0] != 0.0) {
        double hx, hy;
        glad_oracle_enfw(nf, dx, dy, NULL, &hx, &hy, NULL, NULL);
        a_x += hx;
        a_y += hy;
    }
    *ax = a_x;
    *ay = a_y;
}
void glad_oracle_deflection(const double* p, double thx, double thy, double* ax, double* ay) {
    glad_oracle_deflection_sheet(p, 1.0, 0.0, 0.0, thx, thy, ax, ay);
}

/* Chameleon light profile, Eq. 47: the paper's lens-light model (two of them), a difference of two cored
 * isothermal profiles with core radii w_c < w_t; R^2 = x^2 + y^2/q^2 in the component frame.
 * SURVEY.md 8(f) rank 4 (light part).  Slot layout when a component is of this kind: {I_0, w_c, w_t, q, phi}. */
double glad_oracle_chameleon(double dx, double dy, double I0, double wc, double wt, double q, double phi) {
    double c = cos(phi), s = sin(phi);
    double x = dx * c + dy * s, y = -dx * s + dy * c;
    double R2 = x * x + y * y / (q * q);
    double opq = 1.0 + q;
    return I0 / opq * (1.0 / sqrt(R2 + 4.0 * wc * wc / (opq * opq)) - 1.0 / sqrt(R2 + 4.0 * wt * wt / (opq * opq)));
}

/* kinds[c] (c = source, lens light 1, lens light 2): 0 = Sersic (R-L7), 1 = Chameleon (Eq. 47); NULL = all Sersic */
static int lens_params_valid_kinds(const double* p, const int* kinds);
static int lens_params_valid(const double* p) { return lens_params_valid_kinds(p, NULL); }
static int lens_params_valid_kinds(const double* p, const int* kinds) {
    if (!(p[2] >= 0.0)) return 0;                       /* theta_E */
    if (!(p[3] > 1.0 && p[3] < 3.0)) return 0;          /* gamma in (1,3) */
    if (!(p[4] > 0.0 && p[4] <= 1.0)) return 0;         /* q */
    if (!(p[8] >= 0.0)) return 0;                       /* theta_E,BH^2 */
    const int off[3] = {11, 16, 21};                    /* Ie,Re,n,q,phi of the 3 Sersics */
    for (int c = 0; c < 3; ++c) {
        const double* s = p + off[c];
        if (s[0] == 0.0) continue;                      /* disabled component */
        if (kinds && kinds[c] == 1) {                   /* Chameleon: 0 < w_c < w_t (positive profile), q in (0,1] */
            if (!(s[1] > 0.0 && s[2] > s[1] && s[3] > 0.0 && s[3] <= 1.0)) return 0;
            continue;
        }
        if (!(s[1] > 0.0 && s[2] > 0.0 && s[3] > 0.0 && s[3] <= 1.0)) return 0;
    }
    return 1;
}

/*
 * Lensing half, for B parameter vectors.
 *   lens   [B,26] float32 parameter vectors (layout in include/glad.h, restated in DESIGN.md)
 *   grid   nx, ny, supersample s, pixel size pix, (x0,y0) = centre of pixel (0,0)   (reading R-L1)
 *   psf    [kpsf,kpsf] float32, odd kpsf, NOT renormalised                         (reading R-L8)
 *   data, ivar [ny,nx] float32
 * Outputs (either may be NULL): images [B,ny,nx] fp64 PSF-convolved model; chi2 [B] fp64;
 * flags [B] int32 (FLAG_LENS_INVALID -> image NaN, chi2 +inf).
 */
int glad_oracle_lens_image_batch_kinds(const float* lens, int B, int nx, int ny, int s, double pix,
                                       double x0, double y0, const float* psf, int kpsf,
                                       const float* data, const float* ivar, const int* kinds,
                                       double* images, double* chi2, int32_t* flags);
int glad_oracle_lens_image_batch(const float* lens, int B, int nx, int ny, int s, double pix,
                                 double x0, double y0, const float* psf, int kpsf,
                                 const float* data, const float* ivar, double* images,
                                 double* chi2, int32_t* flags) {
    return glad_oracle_lens_image_batch_kinds(lens, B, nx, ny, s, pix, x0, y0, psf, kpsf, data, ivar, NULL, images, chi2, flags);
}
int glad_oracle_lens_image_batch_sheet(const float* lens, int B, int nx, int ny, int s, double pix,
                                       double x0, double y0, const float* psf, int kpsf,
                                       const float* data, const float* ivar, const int* kinds,
                                       const float* lambda, double rc, double rt,
                                       double* images, double* chi2, int32_t* flags);
/* same, with the light profile kind of each component (see lens_params_valid_kinds) */
int glad_oracle_lens_image_batch_kinds(const float* lens, int B, int nx, int ny, int s, double pix,
                                       double x0, double y0, const float* psf, int kpsf,
                                       const float* data, const float* ivar, const int* kinds,
                                       double* images, double* chi2, int32_t* flags) {
    return glad_oracle_lens_image_batch_sheet(lens, B, nx, ny, s, pix, x0, y0, psf, kpsf, data, ivar, kinds, NULL, 0.0, 0.0,
                                              images, chi2, flags);
}
/* same, with the internal mass sheet: lambda [B] float32 (NULL = none), rt > rc > 0 arcsec (R-S1..3);
 * a non-finite lambda invalidates the vector */
int glad_oracle_lens_image_batch_halo(const float* lens, int B, int nx, int ny, int s, double pix,
                                      double x0, double y0, const float* psf, int kpsf,
                                      const float* data, const float* ivar, const int* kinds,
                                      const float* lambda, double rc, double rt, const float* enfw,
                                      double* images, double* chi2, int32_t* flags);
int glad_oracle_lens_image_batch_sheet(const float* lens, int B, int nx, int ny, int s, double pix,
                                       double x0, double y0, const float* psf, int kpsf,
                                       const float* data, const float* ivar, const int* kinds,
                                       const float* lambda, double rc, double rt,
                                       double* images, double* chi2, int32_t* flags) {
    return glad_oracle_lens_image_batch_halo(lens, B, nx, ny, s, pix, x0, y0, psf, kpsf, data, ivar, kinds, lambda, rc, rt, NULL,
                                             images, chi2, flags);
}
/* same, with an eNFW halo per vector: enfw [B,4] float32 {rho_s, r_s, q, phi} or NULL (mass part) */
int glad_oracle_lens_image_batch_halo(const float* lens, int B, int nx, int ny, int s, double pix,
                                      double x0, double y0, const float* psf, int kpsf,
                                      const float* data, const float* ivar, const int* kinds,
                                      const float* lambda, double rc, double rt, const float* enfw,
                                      double* images, double* chi2, int32_t* flags) {
    if (lambda && !(rc > 0.0 && rt > rc)) return -1;
    if (B < 0 || nx <= 0 || ny <= 0 || s <= 0 || kpsf <= 0 || (kpsf % 2) == 0) return -1;
    if (kinds) for (int c = 0; c < 3; ++c) if (kinds[c] != 0 && kinds[c] != 1) return -1;
    const int ks = kinds ? kinds[0] : 0, k1 = kinds ? kinds[1] : 0, k2 = kinds ? kinds[2] : 0;
    int npx = nx * ny, c = kpsf / 2;
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < B; ++b) {
        double p[ORACLE_NLENS];
        for (int i = 0; i < ORACLE_NLENS; ++i) p[i] = (double)lens[(size_t)b * ORACLE_NLENS + i];
        if (flags) flags[b] = 0;
        const double lam = lambda ? (double)lambda[b] : 1.0, src = lambda ? rc : 0.0;
        double nfv[4] = {0.0, 1.0, 1.0, 0.0};
        if (enfw) for (int i = 0; i < 4; ++i) nfv[i] = (double)enfw[(size_t)b * 4 + i];
        const double* nf = enfw ? nfv : NULL;
        if (!lens_params_valid_kinds(p, kinds) || !isfinite(lam) || !enfw_valid(nfv)) {
            if (flags) flags[b] |= FLAG_LENS_INVALID;
            if (images) for (int i = 0; i < npx; ++i) images[(size_t)b * npx + i] = NAN;
            if (chi2) chi2[b] = INFINITY;
            continue;
        }
        double bn_s = (p[11] != 0.0 && !ks) ? glad_oracle_sersic_bn(p[13]) : 0.0;
        double bn_1 = (p[16] != 0.0 && !k1) ? glad_oracle_sersic_bn(p[18]) : 0.0;
        double bn_2 = (p[21] != 0.0 && !k2) ? glad_oracle_sersic_bn(p[23]) : 0.0;
        double* binned = (double*)malloc(sizeof(double) * npx);
        /* a1-a3: ray-shoot every sub-pixel centre (Eq. 33), evaluate light, mean (R-L2) */
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                double acc = 0.0;
                for (int sb = 0; sb < s; ++sb)
                    for (int sa = 0; sa < s; ++sa) {
                        double thx = x0 + ix * pix + ((sa + 0.5) / s - 0.5) * pix;
                        double thy = y0 + iy * pix + ((sb + 0.5) / s - 0.5) * pix;
                        double ax, ay;
                        glad_oracle_deflection_halo(p, lam, src, rt, nf, thx, thy, &ax, &ay);
                        double bx = thx - ax, by = thy - ay; /* beta = theta - alpha */
                        double v = 0.0;
                        if (p[11] != 0.0)
                            v += ks ? glad_oracle_chameleon(bx - p[9], by - p[10], p[11], p[12], p[13], p[14], p[15])
                                    : glad_oracle_sersic(bx - p[9], by - p[10], p[11], p[12], p[13], p[14], p[15], bn_s);
                        if (p[16] != 0.0)
                            v += k1 ? glad_oracle_chameleon(thx - p[0], thy - p[1], p[16], p[17], p[18], p[19], p[20])
                                    : glad_oracle_sersic(thx - p[0], thy - p[1], p[16], p[17], p[18], p[19], p[20], bn_1);
                        if (p[21] != 0.0)
                            v += k2 ? glad_oracle_chameleon(thx - p[0], thy - p[1], p[21], p[22], p[23], p[24], p[25])
                                    : glad_oracle_sersic(thx - p[0], thy - p[1], p[21], p[22], p[23], p[24], p[25], bn_2);
                        acc += v;
                    }
                binned[iy * nx + ix] = acc / (double)(s * s);
            }
        /* a4: m = binned (*) PSF, "same", zero outside (Eq. 38, R-L8); chi2 (Eq. 48) */
        double x2 = 0.0;
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                double m = 0.0;
                for (int dy = 0; dy < kpsf; ++dy)
                    for (int dx = 0; dx < kpsf; ++dx) {
                        int sy = iy - (dy - c), sx = ix - (dx - c);
                        if (sy < 0 || sy >= ny || sx < 0 || sx >= nx) continue;
                        m += (double)psf[dy * kpsf + dx] * binned[sy * nx + sx];
                    }
                if (images) images[(size_t)b * npx + iy * nx + ix] = m;
                if (data && ivar) {
                    double r = (double)data[iy * nx + ix] - m;
                    x2 += (double)ivar[iy * nx + ix] * r * r;
                }
            }
        if (chi2) chi2[b] = x2;
        free(binned);
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Dynamics half.                                                             */
/* ------------------------------------------------------------------------ */

/*
 * Integrand-summed second moment at ONE sky position, lengths in pc:
 * cylindrically-aligned axisymmetric JAM, single quadrature over u in (0,1)
 * (paper defers to Cappellari at P:228; reading R-D1 states it):
 *
 *  [Sigma v2_los](x',y') = 4 pi^{3/2} G  sum_u w_u sum_k sum_j nu0_k q_j rho0_j u^2
 *        [ s_k^2 q_k^2 (cos^2 i + b_k sin^2 i) + D x'^2 sin^2 i ]
 *        / [ (1 - C u^2) sqrt( (A + B cos^2 i) [1 - (1-q_j^2) u^2] ) ]
 *        exp{ -A [ x'^2 + y'^2 (A+B)/(A + B cos^2 i) ] }
 *  A = (u^2/s_j^2 + 1/s_k^2)/2
 *  B = { (1-q_k^2)/(s_k^2 q_k^2) + (1-q_j^2) u^4 / (s_j^2 [1-(1-q_j^2)u^2]) } / 2
 *  C = 1 - q_j^2 - s_k^2 q_k^2 / s_j^2
 *  D = 1 - b_k q_k^2 - [ (1-b_k) C + (1-q_j^2) b_k ] u^2
 *
 * k = luminous Gaussian (sigma_k, intrinsic q_k, nu0_k, b_k = 1/(1-beta_z,k)),
 * j = mass Gaussian (sigma_j, q_j, rho0_j).
 */
double glad_oracle_jam_sigv2_point(double xp, double yp, double inc, int nl, const double* sig_k,
                                   const double* q_k, const double* nu0_k, const double* b_k,
                                   int nm, const double* sig_j, const double* q_j,
                                   const double* rho0_j, int nu, const double* u_nodes,
                                   const double* u_weights) {
    double ci = cos(inc), si = sin(inc), ci2 = ci * ci, si2 = si * si;
    double total = 0.0;
    for (int iu = 0; iu < nu; ++iu) {
        double u = u_nodes[iu], u2 = u * u, node = 0.0;
        for (int k = 0; k < nl; ++k)
            for (int j = 0; j < nm; ++j) {
                double sk2 = sig_k[k] * sig_k[k], sj2 = sig_j[j] * sig_j[j];
                double qk2 = q_k[k] * q_k[k], qj2 = q_j[j] * q_j[j];
                double g = 1.0 - (1.0 - qj2) * u2;
                double A = 0.5 * (u2 / sj2 + 1.0 / sk2);
                double Bc = 0.5 * ((1.0 - qk2) / (sk2 * qk2) + (1.0 - qj2) * u2 * u2 / (sj2 * g));
                double C = 1.0 - qj2 - sk2 * qk2 / sj2;
                double D = 1.0 - b_k[k] * qk2 - ((1.0 - b_k[k]) * C + (1.0 - qj2) * b_k[k]) * u2;
                double E = A + Bc * ci2;
                double numer = sk2 * qk2 * (ci2 + b_k[k] * si2) + D * xp * xp * si2;
                double denom = (1.0 - C * u2) * sqrt(E * g);
                double ex = exp(-A * (xp * xp + yp * yp * (A + Bc) / E));
                node += nu0_k[k] * q_j[j] * rho0_j[j] * u2 * numer / denom * ex;
            }
        total += u_weights[iu] * node;
    }
    return 4.0 * pow(PI, 1.5) * G_NEWTON * total;
}

/* Deprojection of one Gaussian (Eq. 22, Eq. 23/25 P:176,186):
 * q = sqrt(q'^2 - cos^2 i)/sin i ; dens0 = surf0 q' / (q sigma sqrt(2 pi)).
 * Returns 0 if not deprojectable. */
static int deproject(double surf0, double sigma_pc, double qp, double inc, double* q,
                     double* dens0) {
    double ci = cos(inc), si = sin(inc);
    double d = qp * qp - ci * ci;
    if (!(d > 0.0) || !(si > 0.0) || !(qp > 0.0) || !(sigma_pc > 0.0)) return 0;
    *q = sqrt(d) / si;
    *dens0 = surf0 * qp / (*q * sigma_pc * sqrt(2.0 * PI));
    return 1;
}

/*
 * a7 + a8 on given maps: num = Sv2 (*) K, den = S (*) K, true convolution,
 * "same" size, zero outside (Eq. 27, reading R-D6); V2_l = sum_{p in l} num / sum_{p in l} den;
 * v_l = sqrt(V2_l) (Eq. 28); chi2_D = sum_l ivar_l (obs_l - v_l)^2 (Eq. 32, diagonal
 * covariance, reading R-D7).  Returns 1 if any bin is empty or has V2 < 0 (v = NaN there).
 */
int glad_oracle_kin_bins(const double* sv2, const double* sb, int nx, int ny, const int32_t* bin_id,
                         int nbins, const float* kern, int kk, const float* vrms_obs,
                         const float* vrms_ivar, double* vrms, double* chi2) {
    int c = kk / 2, bad = 0;
    double* bnum = calloc(nbins, sizeof(double));
    double* bden = calloc(nbins, sizeof(double));
    int* bcnt = calloc(nbins, sizeof(int));
    for (int iy = 0; iy < ny; ++iy)
        for (int ix = 0; ix < nx; ++ix) {
            int l = bin_id[iy * nx + ix];
            if (l < 0 || l >= nbins) continue;
            double num = 0.0, den = 0.0;
            for (int dy = 0; dy < kk; ++dy)
                for (int dx = 0; dx < kk; ++dx) {
                    int sy = iy - (dy - c), sx = ix - (dx - c);
                    if (sy < 0 || sy >= ny || sx < 0 || sx >= nx) continue;
                    double w = kern[dy * kk + dx];
                    num += w * sv2[sy * nx + sx];
                    den += w * sb[sy * nx + sx];
                }
            bnum[l] += num;
            bden[l] += den;
            bcnt[l] += 1;
        }
    double x2 = 0.0;
    for (int l = 0; l < nbins; ++l) {
        double v2 = (bcnt[l] > 0 && bden[l] > 0.0) ? bnum[l] / bden[l] : NAN;
        double v = (v2 >= 0.0) ? sqrt(v2) : NAN;
        if (!(v == v)) bad = 1;
        if (vrms) vrms[l] = v;
        if (vrms_obs && vrms_ivar) {
            double r = (double)vrms_obs[l] - v;
            x2 += (double)vrms_ivar[l] * r * r;
        }
    }
    if (chi2) *chi2 = x2;
    free(bnum); free(bden); free(bcnt);
    return bad;
}

/*
 * Dynamics half, for B parameter vectors.
 *   dyn      [B,4] float32 {inclination rad, D_d Mpc, M_BH Msun, Upsilon}
 *   lum_mge  [.,n_lum,3] float32 rows {I0 Lsun/pc^2, sigma' arcsec, q'}; lum_stride floats
 *            between vectors (0 = one table shared by all)
 *   mass_mge [.,n_mass,3] likewise {Sigma0 Msun/pc^2, sigma' arcsec, q'}
 *   beta     [B,n_lum] (beta_per_gaussian) or [B] : beta_z,k  (reading R-D2)
 *   sky grid xs[nx], ys[ny] arcsec, galaxy-aligned tensor grid (reading R-D5)
 *   bin_id   [ny,nx] int32 in [0,nbins) or -1; kern [kk,kk] float32 odd kk
 *   vrms_obs, vrms_ivar [nbins]; u_nodes, u_weights [nu]  (reading R-D4)
 * Outputs (may be NULL): vrms [B,nbins], chi2 [B], v2map [B,ny,nx] = raw Sigma*v2_los map,
 * sbmap [B,ny,nx] = Sigma map, flags [B].
 */
int glad_oracle_jam_vrms_batch(const float* dyn, int B, const float* lum_mge, int n_lum,
                               long lum_stride, const float* mass_mge, int n_mass,
                               long mass_stride, const float* beta, int beta_per_gaussian, int nx,
                               int ny, const float* xs, const float* ys, const int32_t* bin_id,
                               int nbins, const float* kern, int kk, const float* vrms_obs,
                               const float* vrms_ivar, const float* u_nodes,
                               const float* u_weights, int nu, double* vrms, double* chi2,
                               double* v2map, double* sbmap, int32_t* flags) {
    if (B < 0 || n_lum <= 0 || n_mass < 0 || nx <= 0 || ny <= 0 || nbins <= 0 || kk <= 0 ||
        (kk % 2) == 0 || nu <= 0)
        return -1;
    int npx = nx * ny;
    double* un = (double*)malloc(sizeof(double) * nu);
    double* uw = (double*)malloc(sizeof(double) * nu);
    for (int i = 0; i < nu; ++i) { un[i] = u_nodes[i]; uw[i] = u_weights[i]; }
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < B; ++b) {
        double inc = dyn[b * ORACLE_NDYN + 0], Dd = dyn[b * ORACLE_NDYN + 1];
        double Mbh = dyn[b * ORACLE_NDYN + 2], ups = dyn[b * ORACLE_NDYN + 3];
        double pc_per_arcsec = Dd * PI / 0.648; /* D_d[Mpc] 1e6 pi/648000 */
        const float* lt = lum_mge + (size_t)b * lum_stride;
        const float* mt = mass_mge + (size_t)b * mass_stride;
        int nm = n_mass + (Mbh > 0.0 ? 1 : 0);
        double *sk = malloc(sizeof(double) * n_lum), *qk = malloc(sizeof(double) * n_lum),
               *nu0 = malloc(sizeof(double) * n_lum), *bk = malloc(sizeof(double) * n_lum),
               *sj = malloc(sizeof(double) * (nm + 1)), *qj = malloc(sizeof(double) * (nm + 1)),
               *rho0 = malloc(sizeof(double) * (nm + 1));
        double* sv2 = malloc(sizeof(double) * npx);
        double* sb = malloc(sizeof(double) * npx);
        int ok = (Dd > 0.0) && (Mbh >= 0.0);
        for (int k = 0; k < n_lum && ok; ++k) {
            sk[k] = (double)lt[3 * k + 1] * pc_per_arcsec;
            ok = deproject((double)lt[3 * k + 0], sk[k], (double)lt[3 * k + 2], inc, &qk[k], &nu0[k]);
            double bz = beta_per_gaussian ? (double)beta[(size_t)b * n_lum + k] : (double)beta[b];
            if (!(bz < 1.0)) ok = 0;
            bk[k] = 1.0 / (1.0 - bz);
        }
        for (int j = 0; j < n_mass && ok; ++j) {
            sj[j] = (double)mt[3 * j + 1] * pc_per_arcsec;
            ok = deproject(ups * (double)mt[3 * j + 0], sj[j], (double)mt[3 * j + 2], inc, &qj[j],
                           &rho0[j]);
        }
        if (ok && Mbh > 0.0) { /* reading R-D3: BH = one round Gaussian of sigma 0.01" */
            sj[n_mass] = SIGMA_BH_ARCSEC * pc_per_arcsec;
            double surf0 = Mbh / (2.0 * PI * sj[n_mass] * sj[n_mass]);
            ok = deproject(surf0, sj[n_mass], 1.0, inc, &qj[n_mass], &rho0[n_mass]);
        }
        int32_t fl = 0;
        if (!ok) {
            fl |= FLAG_DYN_INVALID;
            if (vrms) for (int l = 0; l < nbins; ++l) vrms[(size_t)b * nbins + l] = NAN;
            if (chi2) chi2[b] = INFINITY;
            if (v2map) for (int i = 0; i < npx; ++i) v2map[(size_t)b * npx + i] = NAN;
            if (sbmap) for (int i = 0; i < npx; ++i) sbmap[(size_t)b * npx + i] = NAN;
        } else {
            /* a6: quadrature at every pixel centre; Sigma map (Eq. 21) */
            for (int iy = 0; iy < ny; ++iy)
                for (int ix = 0; ix < nx; ++ix) {
                    double xa = xs[ix], ya = ys[iy]; /* arcsec */
                    sv2[iy * nx + ix] = glad_oracle_jam_sigv2_point(
                        xa * pc_per_arcsec, ya * pc_per_arcsec, inc, n_lum, sk, qk, nu0, bk, nm, sj,
                        qj, rho0, nu, un, uw);
                    double sbv = 0.0;
                    for (int k = 0; k < n_lum; ++k) {
                        double s = lt[3 * k + 1], qp = lt[3 * k + 2];
                        sbv += (double)lt[3 * k + 0] *
                               exp(-(xa * xa + ya * ya / (qp * qp)) / (2.0 * s * s));
                    }
                    sb[iy * nx + ix] = sbv;
                }
            if (v2map) memcpy(v2map + (size_t)b * npx, sv2, sizeof(double) * npx);
            if (sbmap) memcpy(sbmap + (size_t)b * npx, sb, sizeof(double) * npx);
            /* a7 + a8 */
            double* vout = malloc(sizeof(double) * nbins);
            double x2 = 0.0;
            int bad = glad_oracle_kin_bins(sv2, sb, nx, ny, bin_id, nbins, kern, kk, vrms_obs, vrms_ivar,
                                           vout, &x2);
            if (bad) fl |= FLAG_BIN_INVALID;
            if (vrms) memcpy(vrms + (size_t)b * nbins, vout, sizeof(double) * nbins);
            if (chi2) chi2[b] = bad ? INFINITY : x2;
            free(vout);
        }
        if (flags) flags[b] = fl;
        free(sk); free(qk); free(nu0); free(bk); free(sj); free(qj); free(rho0);
        free(sv2); free(sb);
    }
    free(un); free(uw);
    return 0;
}

/* Joint: lnL = -(chi2_L + chi2_D)/2, no normalisation constant (Eq. 52-53
 * restricted to the pixel term and chi2_dyn; R-J1); -inf where either half is invalid. */
void glad_oracle_joint(const double* chi2_lens, const double* chi2_dyn, int B, double* loglike) {
    for (int b = 0; b < B; ++b) {
        double s = chi2_lens[b] + chi2_dyn[b];
        loglike[b] = (isfinite(s)) ? -0.5 * s : -INFINITY;
    }
}

/* theta_E,BH^2 [arcsec^2] = 4 G M (1+z_d) / (c^2 D_dt), from Eq. 4 P:75 (host helper). */
double glad_oracle_bh_theta2(double Mbh_msun, double Ddt_mpc, double zd) {
    const double c_kms = 299792.458;
    double rad2 = 4.0 * G_NEWTON * Mbh_msun * (1.0 + zd) / (c_kms * c_kms * Ddt_mpc * 1e6);
    double arcsec_per_rad = 648000.0 / PI;
    return rad2 * arcsec_per_rad * arcsec_per_rad;
}

/* ------------------------------------------------------------------------ */
/* SURVEY.md 8(f) rank 4 (quasar part): image-position and time-delay chi^2,  */
/* Eq. 35-36, built on the Fermat potential of Eq. 1-4. */
/* The paper prints neither psi nor the Jacobian of the models; both follow   */
/* from its convergence (App. B) -- DESIGN.md readings R-Q1..R-Q5:            */
/*   EPL: kappa = (3-gamma)/2 (b/R)^(gamma-1) is homogeneous of degree -t      */
/*        (t = gamma-1), hence psi of degree 2-t and alpha of degree 1-t, so   */
/*        (Euler's theorem)  psi = (x alpha_x + y alpha_y)/(2-t)               */
/*        and, with z = x+iy, alpha = alpha_x + i alpha_y, kappa = d(alpha)/dz,*/
/*        gamma_c = d(alpha)/d(conj z):  z kappa + conj(z) gamma_c = (1-t) alpha*/
/*        => gamma_1 + i gamma_2 = [(1-t) alpha z - kappa z^2]/|z|^2 ;         */
/*        psi_xx = kappa+gamma_1, psi_yy = kappa-gamma_1, psi_xy = gamma_2.    */
/*   shear (Eq. 49): psi = gamma_ext/2 r^2 cos 2(phi - phi_ext).         */
/*   point mass: psi = theta_E,BH^2 ln r.                              */
/* ------------------------------------------------------------------------ */

/* psi(theta) of EPL + shear + point mass; p = lens vector (first 9 entries used) */
double glad_oracle_potential_sheet(const double* p, double lam, double rc, double rt, double thx, double thy);
double glad_oracle_potential(const double* p, double thx, double thy) {
    return glad_oracle_potential_sheet(p, 1.0, 0.0, 0.0, thx, thy);
}
/* with the internal mass sheet: lam psi_epl + psi_sheet (+ shear, point mass), Eq. 8 with the dPIE sheet */
double glad_oracle_potential_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy);
double glad_oracle_potential_sheet(const double* p, double lam, double rc, double rt, double thx, double thy) {
    return glad_oracle_potential_halo(p, lam, rc, rt, NULL, thx, thy);
}
double glad_oracle_potential_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy) {
    double dx = thx - p[0], dy = thy - p[1];
    double c = cos(p[5]), s = sin(p[5]);
    double xl = dx * c + dy * s, yl = -dx * s + dy * c;
    double axl, ayl;
    glad_oracle_epl_alpha(xl, yl, p[2], p[3], p[4], &axl, &ayl);
    double psi = lam * (xl * axl + yl * ayl) / (3.0 - p[3]);
    double c2 = cos(2.0 * p[7]), s2 = sin(2.0 * p[7]);
    psi += 0.5 * p[6] * ((dx * dx - dy * dy) * c2 + 2.0 * dx * dy * s2);
    double r2 = dx * dx + dy * dy;
    if (r2 < 1e-12) r2 = 1e-12;
    psi += 0.5 * p[8] * log(r2);
    if (rc > 0.0) {
        double ps;
        sheet_terms(lam, rc, rt, dx, dy, NULL, NULL, NULL, &ps, NULL);
        psi += ps;
    }
    if (nf && nf[0] != 0.0) {
        double ph;
        glad_oracle_enfw(nf, dx, dy, NULL, NULL, NULL, NULL, &ph);
        psi += ph;
    }
    return psi;
}

/* Hessian of psi: h[0] = psi_xx, h[1] = psi_xy, h[2] = psi_yy (sky frame) */
void glad_oracle_hessian_sheet(const double* p, double lam, double rc, double rt, double thx, double thy, double* h);
void glad_oracle_hessian(const double* p, double thx, double thy, double* h) {
    glad_oracle_hessian_sheet(p, 1.0, 0.0, 0.0, thx, thy, h);
}
void glad_oracle_hessian_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy, double* h);
void glad_oracle_hessian_sheet(const double* p, double lam, double rc, double rt, double thx, double thy, double* h) {
    glad_oracle_hessian_halo(p, lam, rc, rt, NULL, thx, thy, h);
}
void glad_oracle_hessian_halo(const double* p, double lam, double rc, double rt, const double* nf, double thx, double thy, double* h) {
    double dx = thx - p[0], dy = thy - p[1];
    double c = cos(p[5]), s = sin(p[5]);
    double xl = dx * c + dy * s, yl = -dx * s + dy * c;
    double hxx = 0.0, hxy = 0.0, hyy = 0.0;
    if (p[2] != 0.0) {
        double t = p[3] - 1.0, q = p[4];
        double axl, ayl;
        glad_oracle_epl_alpha(xl, yl, p[2], p[3], q, &axl, &ayl);
        double b = pow(2.0 / (1.0 + q), 1.0 / t) * p[2];          /* Eq. B.3 */
        double R2 = xl * xl + yl * yl / (q * q);                   /* Eq. B.2 */
        if (q * q * R2 < 1e-12) R2 = 1e-12 / (q * q);
        double kappa = 0.5 * (2.0 - t) * pow(b * b / R2, 0.5 * t); /* Eq. B.1 */
        double complex z = xl + I * yl;
        double r2 = xl * xl + yl * yl;
        if (r2 < 1e-12) r2 = 1e-12;
        double complex g = ((1.0 - t) * (axl + I * ayl) * z - kappa * z * z) / r2;
        double lxx = kappa + creal(g), lyy = kappa - creal(g), lxy = cimag(g);
        /* rotate the lens-frame tensor back by +phi_PA: H = R L R^T */
        hxx = lam * (c * c * lxx - 2.0 * c * s * lxy + s * s * lyy);
        hyy = lam * (s * s * lxx + 2.0 * c * s * lxy + c * c * lyy);
        hxy = lam * (c * s * (lxx - lyy) + (c * c - s * s) * lxy);
    }
    if (rc > 0.0) {
        double hs[3];
        sheet_terms(lam, rc, rt, dx, dy, NULL, NULL, hs, NULL, NULL);
        hxx += hs[0]; hxy += hs[1]; hyy += hs[2];
    }
    if (nf && nf[0] != 0.0) {
        double hh[3];
        glad_oracle_enfw(nf, dx, dy, NULL, NULL, NULL, hh, NULL);
        hxx += hh[0]; hxy += hh[1]; hyy += hh[2];
    }
    double c2 = cos(2.0 * p[7]), s2 = sin(2.0 * p[7]);
    hxx += p[6] * c2;
    hyy -= p[6] * c2;
    hxy += p[6] * s2;
    double r2 = dx * dx + dy * dy;
    if (r2 < 1e-12) r2 = 1e-12;
    hxx += p[8] * (dy * dy - dx * dx) / (r2 * r2);
    hyy -= p[8] * (dy * dy - dx * dx) / (r2 * r2);
    hxy -= 2.0 * p[8] * dx * dy / (r2 * r2);
    h[0] = hxx; h[1] = hxy; h[2] = hyy;
}

/* days per (Mpc arcsec^2): D_dt/c of Eq. 3-4 with theta in arcsec and Delta t in days (R-Q5) */
double glad_oracle_tdelay_const(void) {
    const double mpc_m = 3.0856775814913673e22, c_ms = 299792458.0, day_s = 86400.0;
    double arcsec = PI / 648000.0;
    return mpc_m / c_ms / day_s * arcsec * arcsec;
}

#define ORACLE_MAX_QIMG 8
/*
 * chi^2_img (Eq. 35) and chi^2_tmd (Eq. 36) for B lens vectors, following P:253 step by step:
 *   1. beta_i = theta_i - alpha(theta_i)                                     (Eq. 33)
 *   2. mu_i = 1/det(I - Hessian psi(theta_i));  beta_bar = sum |mu_i| beta_i / sum |mu_i|   (R-Q1)
 *   3. theta_i^pre = the solution of theta - alpha(theta) = beta_bar reached by Newton's method from
 *      theta_i with the Jacobian A = I - Hessian psi, NEWTON_STEPS full steps                (R-Q2)
 *   4. chi2_img = sum_i |theta_i - theta_i^pre|^2 / sigma_theta,i^2
 *   5. phi_i = |theta_i^pre - beta_bar|^2/2 - psi(theta_i^pre)  (Eq. 2);
 *      dt_i^pre = K D_dt (phi_i - phi_ref)  (Eq. 3-4; R-Q3: at the predicted positions);
 *      chi2_tmd = sum_{i != ref, sigma_dt,i > 0} (dt_obs,i - dt_i^pre)^2 / sigma_dt,i^2
 *   lens [B,26] float32 (entries 0..8 used); ddt [B] float32 Mpc; theta_obs [n_img,2], sigma_theta [n_img],
 *   dt_obs, sigma_dt [n_img] (entry ref ignored; sigma_dt <= 0 = no measurement) double.
 * Outputs (may be NULL): chi2_img, chi2_tmd [B]; theta_pre [B,n_img,2]; dt_pre [B,n_img]; beta_bar [B,2];
 * last_step [B,n_img] = length of the last Newton step (how converged step 3 is).
 * Invalid mass parameters (theta_E < 0, gamma outside (1,3), q outside (0,1]) -> chi2 = +inf, outputs NaN.
 */
#define NEWTON_STEPS 12
int glad_oracle_quasar_batch_sheet(const float* lens, const float* ddt, const float* lambda, double rc, double rt, int B,
                                   int n_img, const double* theta_obs, const double* sigma_theta, int ref,
                                   const double* dt_obs, const double* sigma_dt, double* chi2_img, double* chi2_tmd,
                                   double* theta_pre, double* dt_pre, double* beta_bar, double* last_step);
int glad_oracle_quasar_batch(const float* lens, const float* ddt, int B, int n_img, const double* theta_obs,
                             const double* sigma_theta, int ref, const double* dt_obs, const double* sigma_dt,
                             double* chi2_img, double* chi2_tmd, double* theta_pre, double* dt_pre,
                             double* beta_bar, double* last_step) {
    return glad_oracle_quasar_batch_sheet(lens, ddt, NULL, 0.0, 0.0, B, n_img, theta_obs, sigma_theta, ref, dt_obs, sigma_dt,
                                          chi2_img, chi2_tmd, theta_pre, dt_pre, beta_bar, last_step);
}
int glad_oracle_quasar_batch_halo(const float* lens, const float* ddt, const float* lambda, double rc, double rt, const float* enfw,
                                  int B, int n_img, const double* theta_obs, const double* sigma_theta, int ref,
                                  const double* dt_obs, const double* sigma_dt, double* chi2_img, double* chi2_tmd,
                                  double* theta_pre, double* dt_pre, double* beta_bar, double* last_step);
/* same with the internal mass sheet (lambda [B] float32 or NULL; rt > rc > 0) in alpha, the Hessian and psi */
int glad_oracle_quasar_batch_sheet(const float* lens, const float* ddt, const float* lambda, double rc, double rt, int B,
                                   int n_img, const double* theta_obs, const double* sigma_theta, int ref,
                                   const double* dt_obs, const double* sigma_dt, double* chi2_img, double* chi2_tmd,
                                   double* theta_pre, double* dt_pre, double* beta_bar, double* last_step) {
    return glad_oracle_quasar_batch_halo(lens, ddt, lambda, rc, rt, NULL, B, n_img, theta_obs, sigma_theta, ref, dt_obs, sigma_dt,
                                         chi2_img, chi2_tmd, theta_pre, dt_pre, beta_bar, last_step);
}
/* same with an eNFW halo per vector (enfw [B,4] float32 or NULL) */
int glad_oracle_quasar_batch_halo(const float* lens, const float* ddt, const float* lambda, double rc, double rt, const float* enfw,
                                  int B, int n_img, const double* theta_obs, const double* sigma_theta, int ref,
                                  const double* dt_obs, const double* sigma_dt, double* chi2_img, double* chi2_tmd,
                                  double* theta_pre, double* dt_pre, double* beta_bar, double* last_step) {
    if (lambda && !(rc > 0.0 && rt > rc)) return -1;
    if (n_img < 1 || n_img > ORACLE_MAX_QIMG || ref < 0 || ref >= n_img) return -1;
    const double K = glad_oracle_tdelay_const();
#pragma omp parallel for schedule(dynamic)
    for (int b = 0; b < B; ++b) {
        double p[ORACLE_NLENS];
        for (int k = 0; k < ORACLE_NLENS; ++k) p[k] = (double)lens[(size_t)b * ORACLE_NLENS + k];
        const double lam = lambda ? (double)lambda[b] : 1.0, src = lambda ? rc : 0.0;
        double nfv[4] = {0.0, 1.0, 1.0, 0.0};
        if (enfw) for (int i = 0; i < 4; ++i) nfv[i] = (double)enfw[(size_t)b * 4 + i];
        const double* nf = enfw ? nfv : NULL;
        int ok = (p[2] >= 0.0) && (p[3] > 1.0) && (p[3] < 3.0) && (p[4] > 0.0) && (p[4] <= 1.0) && (p[8] >= 0.0) && isfinite(lam) &&
                 enfw_valid(nfv);
        if (!ok) {
            if (chi2_img) chi2_img[b] = INFINITY;
            if (chi2_tmd) chi2_tmd[b] = INFINITY;
            for (int i = 0; i < n_img; ++i) {
                if (theta_pre) { theta_pre[((size_t)b * n_img + i) * 2] = NAN; theta_pre[((size_t)b * n_img + i) * 2 + 1] = NAN; }
                if (dt_pre) dt_pre[(size_t)b * n_img + i] = NAN;
                if (last_step) last_step[(size_t)b * n_img + i] = NAN;
            }
            if (beta_bar) { beta_bar[2 * b] = NAN; beta_bar[2 * b + 1] = NAN; }
            continue;
        }
        /* steps 1-2 */
        double bx = 0.0, by = 0.0, wsum = 0.0;
        for (int i = 0; i < n_img; ++i) {
            double tx = theta_obs[2 * i], ty = theta_obs[2 * i + 1], ax, ay, h[3];
            glad_oracle_deflection_halo(p, lam, src, rt, nf, tx, ty, &ax, &ay);
            glad_oracle_hessian_halo(p, lam, src, rt, nf, tx, ty, h);
            double det = (1.0 - h[0]) * (1.0 - h[2]) - h[1] * h[1];
            double w = fabs(1.0 / det);
            bx += w * (tx - ax);
            by += w * (ty - ay);
            wsum += w;
        }
        bx /= wsum;
        by /= wsum;
        if (beta_bar) { beta_bar[2 * b] = bx; beta_bar[2 * b + 1] = by; }
        /* steps 3-5 */
        double phi[ORACLE_MAX_QIMG], c2i = 0.0;
        for (int i = 0; i < n_img; ++i) {
            double tx = theta_obs[2 * i], ty = theta_obs[2 * i + 1], step = 0.0;
            for (int it = 0; it < NEWTON_STEPS; ++it) {
                double ax, ay, h[3];
                glad_oracle_deflection_halo(p, lam, src, rt, nf, tx, ty, &ax, &ay);
                glad_oracle_hessian_halo(p, lam, src, rt, nf, tx, ty, h);
                double fx = tx - ax - bx, fy = ty - ay - by;          /* lens equation residual */
                double a11 = 1.0 - h[0], a12 = -h[1], a22 = 1.0 - h[2];
                double det = a11 * a22 - a12 * a12;
                double sx = (a22 * fx - a12 * fy) / det, sy = (-a12 * fx + a11 * fy) / det;
                tx -= sx;
                ty -= sy;
                step = sqrt(sx * sx + sy * sy);
            }
            if (theta_pre) { theta_pre[((size_t)b * n_img + i) * 2] = tx; theta_pre[((size_t)b * n_img + i) * 2 + 1] = ty; }
            if (last_step) last_step[(size_t)b * n_img + i] = step;
            double ex = theta_obs[2 * i] - tx, ey = theta_obs[2 * i + 1] - ty;
            c2i += (ex * ex + ey * ey) / (sigma_theta[i] * sigma_theta[i]);
            phi[i] = 0.5 * ((tx - bx) * (tx - bx) + (ty - by) * (ty - by)) - glad_oracle_potential_halo(p, lam, src, rt, nf, tx, ty);
        }
        double c2t = 0.0;
        for (int i = 0; i < n_img; ++i) {
            double dt = K * (double)ddt[b] * (phi[i] - phi[ref]);
            if (dt_pre) dt_pre[(size_t)b * n_img + i] = dt;
            if (i != ref && sigma_dt[i] > 0.0) c2t += (dt_obs[i] - dt) * (dt_obs[i] - dt) / (sigma_dt[i] * sigma_dt[i]);
        }
        if (chi2_img) chi2_img[b] = c2i;
        if (chi2_tmd) chi2_tmd[b] = c2t;
    }
    return 0;
}

/* ------------------------------------------------------------------------ */
/* 1-D multi-Gaussian expansion of a radial profile    */
/* (Eq. 44-46, "following Shajib (2019)"), the step between the    */
/* two halves of the joint model ("we decompose I_light and Sigma_int  */
/* into multiple Gaussian components").                                       */
/*                                                                            */
/*   Eq. 44   f(sigma) = 1/(i sigma^2) sqrt(2/pi) int_C z F(z) e^{z^2/2s^2} dz */
/*   Eq. 45   f(sigma) ~ sum_{n=0}^{2P} eta_n Re F(sigma chi_n)                */
/*   Eq. 46   F(R) ~ sum_n A_n exp(-R^2 / 2 sigma_n^2)  (the printed exponent  */
/*            lost its minus sign), A_n = w_n f(sigma_n) dln(sigma)/sqrt(2pi), */
/*            sigma_n log-spaced, R = sqrt(x^2 + y^2/q^2) (footnote P:234)     */
/* The paper says eta_n, chi_n "can be precomputed" and prints neither; they   */
/* are the Euler-algorithm constants of the cited method (reading    */
/* R-M1):  chi_n = sqrt(2 P ln10 / 3 + 2 pi i n),                              */
/*         eta_n = (-1)^n 2 sqrt(2 pi) 10^{P/3} xi_n,  xi_0 = 1/2,             */
/*         xi_n = 1 (1 <= n <= P), xi_2P = 2^-P,                               */
/*         xi_{2P-n} = xi_{2P-n+1} + 2^-P binom(P, n)  (0 < n < P).            */
/* w_n ("fixed weighting factors") = trapezoid weights in ln(sigma): 1/2 at    */
/* both ends, 1 inside (R-M2).                                                 */
/* Profiles F(z), z complex, principal branches:                              */
/*   kind 0, Sersic (R-L7):  prof = {I_e, R_e, n, q'}                          */
/*           F = I_e exp(-b_n ((z/R_e)^{1/n} - 1))                             */
/*   kind 1, EPL convergence (Eq. B.1-B.3, r_soft = 0 as in R-L3):             */
/*           prof = {scale, theta_E, gamma, q},  F = scale (3-gamma)/2 (b/z)^{gamma-1} */
/*   kind 2, Chameleon (Eq. 47, the paper's I_light):  prof = {I_0, w_c, w_t, q'}          */
/*           F = I_0/(1+q) [ (z^2 + 4 w_c^2/(1+q)^2)^{-1/2} - (z^2 + 4 w_t^2/(1+q)^2)^{-1/2} ]  */
/*           exact transform: 1/sqrt(R^2+a) = sqrt(2/pi) int dln(s) s^-1 e^{-a/2s^2} e^{-R^2/2s^2}, */
/*           so f(sigma) = I_0/(1+q) (2/sigma) (e^{-a_c/2 sigma^2} - e^{-a_t/2 sigma^2})  (pin)    */
/* Output rows {A_n, sigma_n, q'}.  Returns 0, or -1 on bad arguments.         */
/* Pins (tests/test_oracle_mge.py): the power law has the closed form          */
/*   f(sigma) = sqrt(2pi) 2^{1-t/2}/Gamma(t/2) sigma^-t; F = Gaussian of width */
/*   s gives an expansion concentrated at sigma = s; the expansion summed back */
/*   reproduces Sersic and power-law profiles to the accuracy the paper prints */
/*   (~0.5 % with 21 Gaussians); amplitudes linear in the profile       */
/*   scale; sigma_n geometric.                                                 */
/* ------------------------------------------------------------------------ */
static double binom_d(int n, int k) {
    double r = 1.0;
    for (int i = 1; i <= k; ++i) r = r * (double)(n - k + i) / (double)i;
    return r;
}

static double complex mge_profile(int kind, const double* prof, double bn, double complex z) {
    if (kind == 0) {
        double complex w = cpow(z / prof[1], 1.0 / prof[2]);
        return prof[0] * cexp(-bn * (w - 1.0));
    }
    if (kind == 3) {   /* eNFW through CSEs, Eq. A.2-A.4: prof = {scale, r_s, -, q}; F = scale sum A_i / (2 (s_i^2 + u^2)^(3/2)), u = z sqrt(q)/r_s */
        double complex u2 = z * z * prof[3] / (prof[1] * prof[1]), acc = 0.0;
        for (int i = 0; i < g_ncse; ++i) acc += g_cse_A[i] * 0.5 / cpow(g_cse_s[i] * g_cse_s[i] + u2, 1.5);
        return prof[0] * acc;
    }
    if (kind == 2) {   /* Chameleon, Eq. 47: prof = {I_0, w_c, w_t, q} */
        double opq = 1.0 + prof[3];
        double ac = 4.0 * prof[1] * prof[1] / (opq * opq), at = 4.0 * prof[2] * prof[2] / (opq * opq);
        return prof[0] / opq * (1.0 / csqrt(z * z + ac) - 1.0 / csqrt(z * z + at));
    }
    double t = prof[2] - 1.0;
    double b = pow(2.0 / (1.0 + prof[3]), 1.0 / t) * prof[1];        /* Eq. B.3 */
    return prof[0] * 0.5 * (3.0 - prof[2]) * cpow(b / z, t);          /* Eq. B.1 */
}

/* Eq. 45 at one sigma */
double glad_oracle_mge_f_sigma(int kind, const double* prof, double sigma, int P) {
    if (P < 1 || P > 20) return NAN;
    double xi[41];
    xi[0] = 0.5;
    for (int n = 1; n <= P; ++n) xi[n] = 1.0;
    xi[2 * P] = ldexp(1.0, -P);
    for (int n = 1; n < P; ++n) xi[2 * P - n] = xi[2 * P - n + 1] + ldexp(1.0, -P) * binom_d(P, n);
    double bn = kind == 0 ? glad_oracle_sersic_bn(prof[2]) : 0.0;
    double sum = 0.0;
    for (int n = 0; n <= 2 * P; ++n) {
        double complex chi = csqrt(2.0 * P * log(10.0) / 3.0 + 2.0 * PI * n * I);
        double eta = ((n & 1) ? -1.0 : 1.0) * 2.0 * sqrt(2.0 * PI) * pow(10.0, P / 3.0) * xi[n];
        sum += eta * creal(mge_profile(kind, prof, bn, sigma * chi));
    }
    return sum;
}

int glad_oracle_mge1d(int kind, const double* prof, int n_gauss, double sigma_lo, double sigma_hi, int P,
                      double* mge /* [n_gauss,3] */) {
    if ((kind != 0 && kind != 1 && kind != 2 && kind != 3) || n_gauss < 2 || !(sigma_lo > 0.0) || !(sigma_hi > sigma_lo) || P < 1 || P > 20)
        return -1;
    double dln = log(sigma_hi / sigma_lo) / (n_gauss - 1);
    for (int n = 0; n < n_gauss; ++n) {
        double sigma = sigma_lo * exp(dln * n);
        double w = (n == 0 || n == n_gauss - 1) ? 0.5 : 1.0;
        mge[3 * n + 0] = w * glad_oracle_mge_f_sigma(kind, prof, sigma, P) * dln / sqrt(2.0 * PI);   /* Eq. 46 */
        mge[3 * n + 1] = sigma;
        mge[3 * n + 2] = prof[3];
    }
    return 0;
}

/* Eq. 13: Sigma_crit = c^2/(4 pi G) D_dt / ((1+z_d) D_d^2), in Msun/pc^2 for distances in Mpc. */
double glad_oracle_sigma_crit(double Ddt_mpc, double Dd_mpc, double zd) {
    const double c_kms = 299792.458;
    return c_kms * c_kms / (4.0 * PI * G_NEWTON) * (Ddt_mpc * 1e6) / ((1.0 + zd) * (Dd_mpc * 1e6) * (Dd_mpc * 1e6));
}
