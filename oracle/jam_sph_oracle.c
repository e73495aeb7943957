/*
 * jam_sph_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rules as glad_oracle.c).
 *
 * the dynamics the paper actually runs -- axisymmetric Jeans model with a
 * SPHERICALLY-aligned velocity ellipsoid (JAM_sph; Eq. 17-20, Eq. 26, fixed
 * integration mesh P:358-362), plain C, fp64, no blocking / fusion / symmetry / reordering.
 * "P:n" = /root/reference/PAPER.md line n; "R-SPHn" = a reading listed in DESIGN.md.
 *
 * What the paper prints: the two Jeans equations (Eq. 17-18), beta_ani = 1 - v_th^2/v_r^2 (Eq. 20),
 * the MGE densities (Eq. 23, 25), the LOS average (Eq. 26), and the order of the computation:
 * intrinsic moments v_r^2, v_th^2, v_phi^2 "at the required positions ... points in polar
 * coordinates" by a non-adaptive 2-D quadrature, then the projection.  Everything else
 * it defers to Cappellari (2020).  The solution used here is DERIVED from Eq. 17-18 (not
 * taken from any code), so that it can be checked by eye:
 *
 *  (i)  eliminate nu v_phi^2 between Eq. 17 and Eq. 18.  With F = nu v_r^2,
 *          r dF/dr - (1-beta) tan(th) dF/dth + 2 beta F = -Psi,
 *          Psi = nu (r dPhi/dr - tan(th) dPhi/dth) = nu (r^2/z) dPhi/dz     (R = r sin th, z = r cos th).
 *       Its characteristics are sin th' = sin th (r/r')^(1-beta); with F -> 0 at infinity
 *          F(r,th) = int_r^inf (r'/r)^(2 beta) Psi(r',th') dr'/r'.
 *  (ii) nu v_th^2 = (1-beta) F (Eq. 20) and, from Eq. 18,
 *          nu v_phi^2 = (1-beta) [F + tan(th) dF/dth] + nu tan(th) dPhi/dth ;
 *       d th'/d th = tan th'/tan th along a characteristic and Psi depends on th' through sin^2 th' only, so
 *       tan(th) dF/dth = int (r'/r)^(2 beta) [2 s'^2 dPsi/d(s'^2)] dr'/r'  is one more integral of the same kind.
 *  (iii) MGE potential (Emsellem et al. 1994; the one behind Eq. 25):
 *          Phi = -sqrt(2/pi) G sum_j M_j/sigma_j int_0^1 H_j(u) du,
 *          H_j = exp{-u^2/(2 sigma_j^2) [R^2 + z^2/(1 - e_j u^2)]} / sqrt(1 - e_j u^2),  e_j = 1 - q_j^2,
 *          M_j = (2 pi)^(3/2) rho_0j sigma_j^3 q_j.
 *       Hence (r^2/z) dPhi_j/dz = C_j r^2 int_0^1 u^2 / (sigma_j^2 (1-e_j u^2)^(3/2)) E_j du,
 *             tan(th) dPhi_j/dth = -C_j r^2 s^2 int_0^1 e_j u^4 / (sigma_j^2 (1-e_j u^2)^(3/2)) E_j du,
 *             E_j = exp{-(u^2 r^2 / 2 sigma_j^2) [s^2 + (1-s^2)/(1-e_j u^2)]},  C_j = sqrt(2/pi) G M_j / sigma_j.
 *  (iv) anisotropy per luminous Gaussian k (beta_k; the paper samples ONE beta_ani, P:576 -- then all are equal):
 *       the equations are linear in nu, so each Gaussian is transported along its own characteristics and summed.
 *
 * Readings (paper silent; DESIGN.md R-SPH1..6):
 *   R-SPH1  the radial integral uses r' = r exp(W tau), tau in (0,1), W = ln(r_cut/r), r_cut = 6 max_k sigma_k
 *           (nu_k <= exp(-18) beyond it); a point with r >= r_cut has zero moments.  The rule (tau_n, w_n) and
 *           the rule (u_m, w_m) on (0,1) are INPUTS (the paper's mesh: 64 sub-regions x 4 rectangles of Gauss-
 *           Kronrod nodes, is what the default generator builds), so both sides use the same nodes.
 *   R-SPH2  the polar grid r_a (ascending, arcsec), th_b in [0, pi/2] (ascending) is an INPUT ("over 200 points in
 *           polar coordinates").
 *   R-SPH3  LOS integral of Eq. 26: the three ratios v_r^2, v_th^2, v_phi^2 = (nu v^2)/nu at the grid points are
 *           interpolated bilinearly in (ln r, th), clamped to the grid's edges, th folded to [0, pi/2]; nu itself is
 *           evaluated exactly at every LOS point.
 *   R-SPH4  z' = rho_0 sinh(a zeta), zeta in (-1,1) with an INPUT rule, rho_0 = max(sqrt(x'^2+y'^2), r_0),
 *           a = asinh(r_cut/rho_0).
 *   R-SPH5  frames: x = x', y = -y' cos i + z' sin i, z = y' sin i + z' cos i; the LOS direction in the galaxy
 *           frame is (0, sin i, cos i); v_z'^2 = v_r^2 (z'/r)^2 + v_th^2 (cos th sin phi sin i - sin th cos i)^2
 *           + v_phi^2 (cos phi sin i)^2  (second moments: the velocity ellipsoid is diagonal in (r, th, phi)).
 *   R-SPH6  SMBH, Upsilon, units, deprojection, PSF / bins / chi2: exactly as the cylindrical path (R-D3, R-D6..8).
 *
 * Pins (tests/test_oracle_jam_sph.py): Poisson's equation for (iii); Eq. 17 and Eq. 18 themselves by finite
 * differences of the computed moments (flattened, anisotropic); brute-force spherical Jeans with constant beta
 * (scipy.integrate.quad), intrinsic and projected; beta = 0 equals the independently pinned CYLINDRICAL oracle
 * for any flattening and inclination; evenness; linearity in mass.  Overall numbers: parity unpinned against any
 * published value (the paper prints none).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define SPH_NDYN 4
#define SPH_FLAG_DYN_INVALID 2
#define SPH_FLAG_BIN_INVALID 4
#define SPH_RCUT_SIGMAS 6.0

static const double SPH_PI = 3.14159265358979323846;
static const double SPH_G = 0.004301;          /* (km/s)^2 pc / Msun, reading R-D1 */
static const double SPH_SIGMA_BH_ARCSEC = 0.01; /* reading R-D3 */

/* defined in glad_oracle.c (rows a7 + a8 on given maps) */
int glad_oracle_kin_bins(const double* sv2, const double* sb, int nx, int ny, const int32_t* bin_id,
                         int nbins, const float* kern, int kk, const float* vrms_obs,
                         const float* vrms_ivar, double* vrms, double* chi2);

/* luminosity density of Gaussian k at (r, s2 = sin^2 theta), Eq. 23 */
static double nu_gauss(double nu0, double sig, double q, double r, double s2) {
    return nu0 * exp(-(r * r) / (2.0 * sig * sig) * (s2 + (1.0 - s2) / (q * q)));
}

/*
 * Intrinsic second moments at one point (r, theta), lengths in pc, masses in Msun:
 *   out[0] = nu v_r^2, out[1] = nu v_theta^2, out[2] = nu v_phi^2, out[3] = nu   (sums over luminous Gaussians)
 * sig_k, q_k, nu0_k, beta_k: deprojected luminous Gaussians; sig_j, q_j, mass_j: mass Gaussians.
 */
void glad_oracle_jam_sph_intrinsic(double r, double theta, int nl, const double* sig_k,
                                   const double* q_k, const double* nu0_k, const double* beta_k, int nm,
                                   const double* sig_j, const double* q_j, const double* mass_j,
                                   double rcut, int nt, const double* tau, const double* wtau, int nu,
                                   const double* un, const double* uw, double* out) {
    double s = sin(theta), s2 = s * s;
    double Tr = 0.0, Tth = 0.0, Tph = 0.0, nutot = 0.0;
    double W = (rcut > r) ? log(rcut / r) : 0.0;
    for (int k = 0; k < nl; ++k) {
        double beta = beta_k[k], ek = 1.0 - q_k[k] * q_k[k];
        double sk2 = sig_k[k] * sig_k[k], qk2 = q_k[k] * q_k[k];
        double F = 0.0, Gd = 0.0;
        for (int n = 0; n < nt; ++n) {
            if (W <= 0.0) break;
            double rp = r * exp(W * tau[n]);                       /* r' on the characteristic */
            double sp2 = s2 * pow(r / rp, 2.0 * (1.0 - beta));     /* sin^2 theta' */
            double nuk = nu_gauss(nu0_k[k], sig_k[k], q_k[k], rp, sp2);
            double psi = 0.0, dpsi = 0.0;                          /* Psi and 2 s'^2 dPsi/d(s'^2), without nu_k */
            for (int j = 0; j < nm; ++j) {
                double sj2 = sig_j[j] * sig_j[j], ej = 1.0 - q_j[j] * q_j[j];
                double Cj = sqrt(2.0 / SPH_PI) * SPH_G * mass_j[j] / sig_j[j];
                for (int m = 0; m < nu; ++m) {
                    double u = un[m], u2 = u * u, g = 1.0 - ej * u2;
                    double E = exp(-(u2 * rp * rp) / (2.0 * sj2) * (sp2 + (1.0 - sp2) / g));
                    double base = Cj * rp * rp * u2 / (sj2 * g * sqrt(g)) * E;
                    psi += uw[m] * base;
                    /* d/d(s'^2) of both exponents: (r'^2/2) [e_k/(sig_k^2 q_k^2) + e_j u^4/(sig_j^2 g)] */
                    dpsi += uw[m] * base * rp * rp * sp2 * (ek / (sk2 * qk2) + ej * u2 * u2 / (sj2 * g));
                }
            }
            double jac = W * wtau[n] * pow(rp / r, 2.0 * beta);    /* dr'/r' = W dtau */
            F += jac * nuk * psi;
            Gd += jac * nuk * dpsi;
        }
        /* nu_k tan(theta) dPhi/dtheta at the point itself */
        double nuk0 = nu_gauss(nu0_k[k], sig_k[k], q_k[k], r, s2);
        double P = 0.0;
        for (int j = 0; j < nm; ++j) {
            double sj2 = sig_j[j] * sig_j[j], ej = 1.0 - q_j[j] * q_j[j];
            double Cj = sqrt(2.0 / SPH_PI) * SPH_G * mass_j[j] / sig_j[j];
            for (int m = 0; m < nu; ++m) {
                double u = un[m], u2 = u * u, g = 1.0 - ej * u2;
                double E = exp(-(u2 * r * r) / (2.0 * sj2) * (s2 + (1.0 - s2) / g));
                P -= uw[m] * Cj * r * r * s2 * ej * u2 * u2 / (sj2 * g * sqrt(g)) * E;
            }
        }
        Tr += F;
        Tth += (1.0 - beta) * F;
        Tph += (1.0 - beta) * (F + Gd) + nuk0 * P;
        nutot += nuk0;
    }
    out[0] = Tr; out[1] = Tth; out[2] = Tph; out[3] = nutot;
}

/* bilinear interpolation of a [nr, nth] table in (ln r, theta), clamped at the edges (R-SPH3) */
static double interp_polar(const double* tab, int nr, const double* lnr, int nth, const double* th, double lr, double t) {
    int a = 0, b = 0;
    double fa = 0.0, fb = 0.0;
    if (nr > 1) {
        if (lr <= lnr[0]) { a = 0; fa = 0.0; }
        else if (lr >= lnr[nr - 1]) { a = nr - 2; fa = 1.0; }
        else { while (a < nr - 2 && lr >= lnr[a + 1]) ++a; fa = (lr - lnr[a]) / (lnr[a + 1] - lnr[a]); }
    }
    if (nth > 1) {
        if (t <= th[0]) { b = 0; fb = 0.0; }
        else if (t >= th[nth - 1]) { b = nth - 2; fb = 1.0; }
        else { while (b < nth - 2 && t >= th[b + 1]) ++b; fb = (t - th[b]) / (th[b + 1] - th[b]); }
    }
    int a1 = nr > 1 ? a + 1 : a, b1 = nth > 1 ? b + 1 : b;
    double v00 = tab[a * nth + b], v01 = tab[a * nth + b1], v10 = tab[a1 * nth + b], v11 = tab[a1 * nth + b1];
    return (1.0 - fa) * ((1.0 - fb) * v00 + fb * v01) + fa * ((1.0 - fb) * v10 + fb * v11);
}

/*
 * Eq. 26 numerator at one sky position (x', y') in pc: int dz' nu v_z'^2 (R-SPH3..5).
 * ratios: [3][nr][nth] = v_r^2, v_th^2, v_phi^2 on the polar grid rgrid (pc), thgrid (rad).
 */
double glad_oracle_jam_sph_los(double xp, double yp, double inc, int nl, const double* sig_k, const double* q_k,
                               const double* nu0_k, int nr, const double* rgrid, int nth, const double* thgrid,
                               const double* ratios, double rcut, int nz, const double* zeta, const double* wz) {
    double ci = cos(inc), si = sin(inc);
    double* lnr = (double*)malloc(sizeof(double) * nr);
    for (int a = 0; a < nr; ++a) lnr[a] = log(rgrid[a]);
    double rho = sqrt(xp * xp + yp * yp);
    double rho0 = rho > rgrid[0] ? rho : rgrid[0];
    double aa = asinh(rcut / rho0);
    double total = 0.0;
    for (int n = 0; n < nz; ++n) {
        double zp = rho0 * sinh(aa * zeta[n]);
        double dz = rho0 * aa * cosh(aa * zeta[n]) * wz[n];
        double x = xp, y = -yp * ci + zp * si, z = yp * si + zp * ci;
        double R2 = x * x + y * y, r = sqrt(R2 + z * z), R = sqrt(R2);
        if (!(r > 0.0)) continue;
        double ct = z / r, st = R / r, s2 = st * st;
        double cph = R > 0.0 ? x / R : 1.0, sph = R > 0.0 ? y / R : 0.0;
        double nu = 0.0;
        for (int k = 0; k < nl; ++k) nu += nu_gauss(nu0_k[k], sig_k[k], q_k[k], r, s2);
        double t = acos(fabs(ct));                     /* folded polar angle in [0, pi/2] */
        double lr = log(r);
        double vr2 = interp_polar(ratios, nr, lnr, nth, thgrid, lr, t);
        double vt2 = interp_polar(ratios + (size_t)nr * nth, nr, lnr, nth, thgrid, lr, t);
        double vp2 = interp_polar(ratios + (size_t)2 * nr * nth, nr, lnr, nth, thgrid, lr, t);
        double pr = zp / r, pt = ct * sph * si - st * ci, pp = cph * si;
        total += dz * nu * (vr2 * pr * pr + vt2 * pt * pt + vp2 * pp * pp);
    }
    free(lnr);
    return total;
}

static int sph_deproject(double surf0, double sigma_pc, double qp, double inc, double* q, double* dens0) {
    double ci = cos(inc), si = sin(inc);
    double d = qp * qp - ci * ci;
    if (!(d > 0.0) || !(si > 0.0) || !(qp > 0.0) || !(sigma_pc > 0.0)) return 0;
    *q = sqrt(d) / si;
    *dens0 = surf0 * qp / (*q * sigma_pc * sqrt(2.0 * SPH_PI));             /* Eq. 23 / 25 */
    return 1;
}

/*
 * JAM_sph for B parameter vectors; arguments as glad_oracle_jam_vrms_batch with beta = beta_ani (Eq. 20) and, instead
 * of the u rule alone: the polar grid (rgrid [nr] arcsec ascending, thgrid [nth] rad in [0, pi/2] ascending), the radial
 * rule (tau, wtau) [nt], the potential rule (un, uw) [nu], both on (0,1), and the LOS rule (zeta, wz) [nz] on (-1,1).
 * Outputs (may be NULL): vrms [B,nbins], chi2 [B], v2map [B,ny,nx] = int nu v_z'^2 dz' (km^2 s^-2 Lsun pc^-2),
 * moments [B,3,nr,nth] = v_r^2, v_th^2, v_phi^2 on the polar grid (km^2 s^-2), flags [B].
 */
int glad_oracle_jam_sph_vrms_batch(const float* dyn, int B, const float* lum_mge, int n_lum, long lum_stride,
                                   const float* mass_mge, int n_mass, long mass_stride, const float* beta,
                                   int beta_per_gaussian, int nx, int ny, const float* xs, const float* ys,
                                   const int32_t* bin_id, int nbins, const float* kern, int kk, const float* vrms_obs,
                                   const float* vrms_ivar, int nr, const float* rgrid, int nth, const float* thgrid,
                                   int nt, const float* tau, const float* wtau, int nu, const float* un, const float* uw,
                                   int nz, const float* zeta, const float* wz, double* vrms, double* chi2,
                                   double* v2map, double* moments, int32_t* flags) {
    if (B < 0 || n_lum <= 0 || n_mass < 0 || nx <= 0 || ny <= 0 || nbins <= 0 || kk <= 0 || (kk % 2) == 0 ||
        nr <= 0 || nth <= 0 || nt <= 0 || nu <= 0 || nz <= 0)
        return -1;
    int npx = nx * ny, npol = nr * nth;
    double *dt = malloc(sizeof(double) * nt), *dwt = malloc(sizeof(double) * nt), *du = malloc(sizeof(double) * nu),
           *dwu = malloc(sizeof(double) * nu), *dz = malloc(sizeof(double) * nz), *dwz = malloc(sizeof(double) * nz),
           *dth = malloc(sizeof(double) * nth);
    for (int i = 0; i < nt; ++i) { dt[i] = tau[i]; dwt[i] = wtau[i]; }
    for (int i = 0; i < nu; ++i) { du[i] = un[i]; dwu[i] = uw[i]; }
    for (int i = 0; i < nz; ++i) { dz[i] = zeta[i]; dwz[i] = wz[i]; }
    for (int i = 0; i < nth; ++i) dth[i] = thgrid[i];
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < B; ++b) {
        double inc = dyn[b * SPH_NDYN + 0], Dd = dyn[b * SPH_NDYN + 1];
        double Mbh = dyn[b * SPH_NDYN + 2], ups = dyn[b * SPH_NDYN + 3];
        double pc = Dd * SPH_PI / 0.648;                                       /* pc per arcsec */
        const float* lt = lum_mge + (size_t)b * lum_stride;
        const float* mt = mass_mge + (size_t)b * mass_stride;
        int nm = n_mass + (Mbh > 0.0 ? 1 : 0);
        double *sk = malloc(sizeof(double) * n_lum), *qk = malloc(sizeof(double) * n_lum),
               *nu0 = malloc(sizeof(double) * n_lum), *bk = malloc(sizeof(double) * n_lum),
               *sj = malloc(sizeof(double) * (nm + 1)), *qj = malloc(sizeof(double) * (nm + 1)),
               *mj = malloc(sizeof(double) * (nm + 1));
        double* rg = malloc(sizeof(double) * nr);
        double* rat = malloc(sizeof(double) * 3 * npol);
        double* sv2 = malloc(sizeof(double) * npx);
        double* sb = malloc(sizeof(double) * npx);
        int ok = (Dd > 0.0) && (Mbh >= 0.0);
        double smax = 0.0;
        for (int k = 0; k < n_lum && ok; ++k) {
            sk[k] = (double)lt[3 * k + 1] * pc;
            ok = sph_deproject((double)lt[3 * k + 0], sk[k], (double)lt[3 * k + 2], inc, &qk[k], &nu0[k]);
            bk[k] = beta_per_gaussian ? (double)beta[(size_t)b * n_lum + k] : (double)beta[b];
            if (!(bk[k] < 1.0)) ok = 0;
            if (sk[k] > smax) smax = sk[k];
        }
        for (int j = 0; j < n_mass && ok; ++j) {
            double rho0;
            sj[j] = (double)mt[3 * j + 1] * pc;
            ok = sph_deproject(ups * (double)mt[3 * j + 0], sj[j], (double)mt[3 * j + 2], inc, &qj[j], &rho0);
            mj[j] = pow(2.0 * SPH_PI, 1.5) * rho0 * sj[j] * sj[j] * sj[j] * qj[j];
        }
        if (ok && Mbh > 0.0) {                      /* R-D3: one round Gaussian of sigma 0.01" and mass M_BH */
            sj[n_mass] = SPH_SIGMA_BH_ARCSEC * pc; qj[n_mass] = 1.0; mj[n_mass] = Mbh;
        }
        int32_t fl = 0;
        if (!ok) {
            fl |= SPH_FLAG_DYN_INVALID;
            if (vrms) for (int l = 0; l < nbins; ++l) vrms[(size_t)b * nbins + l] = NAN;
            if (chi2) chi2[b] = INFINITY;
            if (v2map) for (int i = 0; i < npx; ++i) v2map[(size_t)b * npx + i] = NAN;
            if (moments) for (int i = 0; i < 3 * npol; ++i) moments[(size_t)b * 3 * npol + i] = NAN;
        } else {
            double rcut = SPH_RCUT_SIGMAS * smax;
            /* step 1: intrinsic moments at every polar grid point */
            for (int a = 0; a < nr; ++a) {
                rg[a] = (double)rgrid[a] * pc;
                for (int t = 0; t < nth; ++t) {
                    double o[4];
                    glad_oracle_jam_sph_intrinsic(rg[a], dth[t], n_lum, sk, qk, nu0, bk, nm, sj, qj, mj, rcut, nt, dt,
                                                  dwt, nu, du, dwu, o);
                    for (int c = 0; c < 3; ++c) rat[c * npol + a * nth + t] = o[3] > 0.0 ? o[c] / o[3] : 0.0;
                }
            }
            if (moments) memcpy(moments + (size_t)b * 3 * npol, rat, sizeof(double) * 3 * npol);
            /* step 2 (Eq. 26): LOS integral at every pixel centre; Sigma map (Eq. 21) */
            for (int iy = 0; iy < ny; ++iy)
                for (int ix = 0; ix < nx; ++ix) {
                    double xa = xs[ix], ya = ys[iy];
                    sv2[iy * nx + ix] = glad_oracle_jam_sph_los(xa * pc, ya * pc, inc, n_lum, sk, qk, nu0, nr, rg, nth,
                                                                dth, rat, rcut, nz, dz, dwz);
                    double sbv = 0.0;
                    for (int k = 0; k < n_lum; ++k) {
                        double s = lt[3 * k + 1], qp = lt[3 * k + 2];
                        sbv += (double)lt[3 * k + 0] * exp(-(xa * xa + ya * ya / (qp * qp)) / (2.0 * s * s));
                    }
                    sb[iy * nx + ix] = sbv;
                }
            if (v2map) memcpy(v2map + (size_t)b * npx, sv2, sizeof(double) * npx);
            /* Eq. 27-28, Eq. 32: rows a7 + a8, shared with the cylindrical path */
            double* vout = malloc(sizeof(double) * nbins);
            double x2 = 0.0;
            int bad = glad_oracle_kin_bins(sv2, sb, nx, ny, bin_id, nbins, kern, kk, vrms_obs, vrms_ivar, vout, &x2);
            if (bad) fl |= SPH_FLAG_BIN_INVALID;
            if (vrms) memcpy(vrms + (size_t)b * nbins, vout, sizeof(double) * nbins);
            if (chi2) chi2[b] = bad ? INFINITY : x2;
            free(vout);
        }
        if (flags) flags[b] = fl;
        free(sk); free(qk); free(nu0); free(bk); free(sj); free(qj); free(mj); free(rg); free(rat); free(sv2); free(sb);
    }
    free(dt); free(dwt); free(du); free(dwu); free(dz); free(dwz); free(dth);
    return 0;
}
