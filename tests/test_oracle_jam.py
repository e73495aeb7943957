"""Pins for the dynamics half of the oracle (CPU only): brute-force Jeans integrations,
limits and invariants.  None of them re-types the
single-quadrature formula the oracle implements."""
import math

import numpy as np
import pytest
from scipy import integrate
from scipy.special import erf

G = 0.004301                       # (km/s)^2 pc / Msun (reading R-D1)
SQ2PI = math.sqrt(2 * math.pi)


def gl(n, a=0.0, b=1.0):
    t, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b - a) * t + 0.5 * (b + a), 0.5 * (b - a) * w


def u_nodes(n):
    t, w = gl(n)
    return t * t, 2 * t * w


def deproject(surf0, sigma, qp, inc):
    """Independent statement: q from the oblate geometry q'^2 = q^2 sin^2 i + cos^2 i, central
    density from conservation of the total: 2 pi sigma^2 q' surf0 = (2 pi)^{3/2} sigma^3 q dens0."""
    q = math.sqrt((qp * qp - math.cos(inc) ** 2)) / math.sin(inc)
    total = 2 * math.pi * sigma ** 2 * qp * surf0
    return q, total / ((2 * math.pi) ** 1.5 * sigma ** 3 * q)


def kin_one_pixel(x_arcsec, y_arcsec, nu=64):
    un, uw = u_nodes(nu)
    return dict(xs=np.array([x_arcsec], np.float32), ys=np.array([y_arcsec], np.float32),
                bin_id=np.zeros((1, 1), np.int32), nbins=1, kernel=np.ones((1, 1), np.float32),
                vrms_obs=None, vrms_ivar=None, u_nodes=un.astype(np.float32), u_weights=uw.astype(np.float32))


# ------------------------------------------------------------------ spherical brute force
def spherical_sigv2(R, sig_l, I0, mass_of_s):
    """Sigma*sigma_los^2 (R) for an isotropic spherical Gaussian tracer in a spherical mass M(s):
    nu sigma_r^2 (r) = int_r^inf nu G M(s)/s^2 ds ;  Sigma sigma_los^2 = 2 int_0^inf nu sigma_r^2 dz."""
    nu0 = I0 / (SQ2PI * sig_l)
    nu = lambda r: nu0 * math.exp(-r * r / (2 * sig_l ** 2))
    nusr2 = lambda r: integrate.quad(lambda s: nu(s) * G * mass_of_s(s) / (s * s), r, r + 14 * sig_l,
                                     epsabs=0, epsrel=1e-11, limit=200)[0]
    val = integrate.quad(lambda z: nusr2(math.hypot(R, z)), 0.0, 12 * sig_l, epsabs=0, epsrel=1e-10, limit=200)[0]
    return 2 * val


@pytest.mark.parametrize("R", [10.0, 200.0, 700.0])
def test_spherical_isotropic_gaussian_pair_vs_brute_force_jeans(oracle, R):
    sig_l, sig_m, I0, S0 = 300.0, 500.0, 1000.0, 3000.0
    Mtot = 2 * math.pi * sig_m ** 2 * S0
    M = lambda s: Mtot * (erf(s / (math.sqrt(2) * sig_m)) - math.sqrt(2 / math.pi) * (s / sig_m) * math.exp(-s * s / (2 * sig_m ** 2)))
    brute = spherical_sigv2(R, sig_l, I0, M)
    inc = math.radians(60.0)
    qk, nu0 = deproject(I0, sig_l, 1.0, inc)
    qj, rho0 = deproject(S0, sig_m, 1.0, inc)
    un, uw = u_nodes(200)
    got = oracle.jam_sigv2_point(R * 0.6, R * 0.8, inc, [sig_l], [qk], [nu0], [1.0], [sig_m], [qj], [rho0], un, uw)
    assert got == pytest.approx(brute, rel=1e-8)
    vrms = math.sqrt(got / (I0 * math.exp(-R * R / (2 * sig_l ** 2))))
    # values printed in SURVEY.md 8(c) D1 (surveyor's probe, for cross-reference only)
    ref = {10.0: 54.113601, 200.0: 52.906359, 700.0: 41.677094}[R]
    assert vrms == pytest.approx(ref, rel=2e-7)


def test_keplerian_point_mass_limit_through_batch_api(oracle):
    """BH only (no mass MGE): the 0.01" Gaussian acts as a point mass for R >> 0.01"."""
    Dd = 775.0
    s = Dd * math.pi / 0.648                                  # pc per arcsec
    sig_as, I0, Mbh = 0.5, 800.0, 5e9
    sig_l = float(np.float32(sig_as)) * s
    for R_as in (0.3, 0.8):
        kin = kin_one_pixel(R_as, 0.0, nu=64)
        un, uw = u_nodes(4000)
        kin["u_nodes"], kin["u_weights"] = un.astype(np.float32), uw.astype(np.float32)
        out = oracle.jam_vrms_batch(np.array([[math.radians(70), Dd, Mbh, 1.0]]), np.array([[I0, sig_as, 1.0]]),
                                    np.zeros((0, 3)), np.array([0.0]), kin, want_maps=True)
        R = float(np.float32(R_as)) * s
        brute = spherical_sigv2(R, sig_l, float(np.float32(I0)), lambda r: Mbh)
        assert out["v2map"][0, 0, 0] == pytest.approx(brute, rel=2e-6)
        assert out["flags"][0] == 0


# ------------------------------------------------------------------ axisymmetric brute force
def axisym_sigv2(xp, yp, inc, I0, sig_l, qp_l, S0, sig_m, qp_m, beta_z, n_los=192, n_z=192, n_u=96):
    """Sigma*v_los^2 at sky point (x',y') [pc] by direct integration of the cylindrically-aligned
    axisymmetric Jeans equations (one luminous, one mass Gaussian):
        Phi = -sqrt(2/pi) G M / sigma  int_0^1 H(u) du,
        H = exp{-u^2/(2 sigma^2) [R^2 + z^2/g]}/sqrt(g),  g = 1-(1-q^2)u^2           (MGE potential)
        nu vz2 (R,z)  = int_z^inf nu dPhi/dz dz'
        nu vphi2      = b [R d(nu vz2)/dR + nu vz2] + R nu dPhi/dR,   nu vR2 = b nu vz2
        v_los^2       = (vR2 sin^2 phi + vphi2 cos^2 phi) sin^2 i + vz2 cos^2 i, cos phi = x/R
    integrated along the line of sight z' with x = x', y = -y' cos i + z' sin i, z = y' sin i + z' cos i.
    All integrals by Gauss-Legendre on numpy grids (nothing analytic beyond differentiating H)."""
    b = 1.0 / (1.0 - beta_z)
    ql, nu0 = deproject(I0, sig_l, qp_l, inc)
    qm, rho0 = deproject(S0, sig_m, qp_m, inc)
    M = (2 * math.pi) ** 1.5 * sig_m ** 3 * qm * rho0
    K = math.sqrt(2 / math.pi) * G * M / sig_m
    u, wu = gl(n_u)
    g = 1 - (1 - qm * qm) * u * u

    def nu(R, z):
        return nu0 * np.exp(-(R * R + z * z / (ql * ql)) / (2 * sig_l ** 2))

    def H(R, z):      # R, z broadcast against trailing u axis
        return np.exp(-u * u / (2 * sig_m ** 2) * (R[..., None] ** 2 + z[..., None] ** 2 / g)) / np.sqrt(g)

    def dPhi_dz(R, z):
        return K * np.sum(wu * (u * u * z[..., None] / (sig_m ** 2 * g)) * H(R, z), axis=-1)

    def dPhi_dR(R, z):
        return K * np.sum(wu * (u * u * R[..., None] / sig_m ** 2) * H(R, z), axis=-1)

    def d2Phi_dRdz(R, z):
        return K * np.sum(wu * (u * u * z[..., None] / (sig_m ** 2 * g)) * (-u * u * R[..., None] / sig_m ** 2) * H(R, z), axis=-1)

    zmax = 12 * sig_l * max(ql, 1.0)
    t, wt = gl(n_z)

    def nuvz2_and_dR(R, z):
        """[nu vz2](R,z) and its R-derivative, R, z arrays of the same shape; inner integral z' in [z, zmax]."""
        span = np.maximum(zmax - z, 0.0)
        zz = z[..., None] + span[..., None] * t               # [..., n_z]
        RR = np.broadcast_to(R[..., None], zz.shape)
        nn = nu(RR, zz)
        fz = dPhi_dz(RR, zz)
        val = np.sum(wt * nn * fz, axis=-1) * span
        dval = np.sum(wt * (-(RR / sig_l ** 2) * nn * fz + nn * d2Phi_dRdz(RR, zz)), axis=-1) * span
        return val, dval

    L = 12 * sig_l
    zl, wl = gl(n_los, -L, L)
    x = np.full_like(zl, xp)
    y = -yp * math.cos(inc) + zl * math.sin(inc)
    z = yp * math.sin(inc) + zl * math.cos(inc)
    R = np.hypot(x, y)
    za = np.abs(z)                                            # fields are even in z
    nvz2, dnvz2 = nuvz2_and_dR(R, za)
    nvphi2 = b * (R * dnvz2 + nvz2) + R * nu(R, za) * dPhi_dR(R, za)
    nvR2 = b * nvz2
    cos2 = (x / R) ** 2
    integrand = (nvR2 * (1 - cos2) + nvphi2 * cos2) * math.sin(inc) ** 2 + nvz2 * math.cos(inc) ** 2
    return float(np.sum(wl * integrand))


AXI_CASES = [  # (q'_L, q'_M, i deg, beta_z, x', y') and the SURVEY.md probe value (cross-reference only)
    ((0.7, 0.8, 75.0, 0.3, 150.0, 80.0), 2.028997e6),
    ((0.65, 0.9, 62.0, -0.3, 400.0, 30.0), 1.550679e6),
    ((0.8, 0.75, 88.0, 0.5, 50.0, 300.0), 1.730828e6),
]


@pytest.mark.parametrize("case,probe", AXI_CASES)
def test_flattened_inclined_anisotropic_pair_vs_brute_force_axisymmetric_jeans(oracle, case, probe):
    qpl, qpm, ideg, bz, xp, yp = case
    inc = math.radians(ideg)
    sig_l, sig_m, I0, S0 = 300.0, 450.0, 1000.0, 3000.0
    brute = axisym_sigv2(xp, yp, inc, I0, sig_l, qpl, S0, sig_m, qpm, bz)
    # convergence of the brute force itself
    brute2 = axisym_sigv2(xp, yp, inc, I0, sig_l, qpl, S0, sig_m, qpm, bz, n_los=128, n_z=128, n_u=64)
    assert brute == pytest.approx(brute2, rel=1e-8)
    ql, nu0 = deproject(I0, sig_l, qpl, inc)
    qm, rho0 = deproject(S0, sig_m, qpm, inc)
    un, uw = u_nodes(200)
    got = oracle.jam_sigv2_point(xp, yp, inc, [sig_l], [ql], [nu0], [1 / (1 - bz)], [sig_m], [qm], [rho0], un, uw)
    assert got == pytest.approx(brute, rel=1e-7)
    assert got == pytest.approx(probe, rel=1e-6)
    # and through the batch API (its own deprojection, arcsec -> pc scaling, Upsilon, float32 inputs)
    Dd = 775.0
    s = Dd * math.pi / 0.648
    kin = kin_one_pixel(xp / s, yp / s, nu=200)
    out = oracle.jam_vrms_batch(np.array([[inc, Dd, 0.0, 2.0]]), np.array([[I0, sig_l / s, qpl]]),
                                np.array([[S0 / 2.0, sig_m / s, qpm]]), np.array([bz]), kin, want_maps=True)
    assert out["v2map"][0, 0, 0] == pytest.approx(brute, rel=5e-6)
    sb = I0 * math.exp(-(xp ** 2 + yp ** 2 / qpl ** 2) / (2 * sig_l ** 2))        # Eq. 21
    assert out["sbmap"][0, 0, 0] == pytest.approx(sb, rel=2e-6)
    assert out["vrms"][0, 0] == pytest.approx(math.sqrt(brute / sb), rel=5e-6)


# ------------------------------------------------------------------ invariants of the batch API
def small_problem(rng, n_lum=4, n_mass=5, n=6, nbins=5, per_gaussian=True, B=3, mbh=3e9):
    lum = np.stack([rng.uniform(200, 2000, n_lum), np.geomspace(0.05, 3.0, n_lum), rng.uniform(0.7, 0.95, n_lum)], 1)
    mass = np.stack([rng.uniform(500, 5000, (B, n_mass)), np.broadcast_to(np.geomspace(0.04, 20.0, n_mass), (B, n_mass)),
                     rng.uniform(0.7, 1.0, (B, n_mass))], 2)
    dyn = np.stack([np.radians(rng.uniform(65, 88, B)), rng.uniform(600, 1000, B), np.full(B, mbh), rng.uniform(0.8, 1.2, B)], 1)
    beta = rng.uniform(-0.3, 0.5, (B, n_lum)) if per_gaussian else rng.uniform(-0.3, 0.5, B)
    ax = ((np.arange(n) - (n - 1) / 2) * 0.3).astype(np.float32)
    un, uw = u_nodes(48)
    kk = 3
    kern = rng.uniform(0.1, 1.0, (kk, kk)); kern /= kern.sum()
    kin = dict(xs=ax, ys=ax.copy(), bin_id=rng.integers(0, nbins, (n, n)).astype(np.int32), nbins=nbins,
               kernel=kern.astype(np.float32), vrms_obs=rng.uniform(200, 300, nbins).astype(np.float32),
               vrms_ivar=rng.uniform(0.01, 0.05, nbins).astype(np.float32),
               u_nodes=un.astype(np.float32), u_weights=uw.astype(np.float32))
    kin["bin_id"].flat[:nbins] = np.arange(nbins)            # no empty bin
    return dyn, lum, mass, beta, kin


def test_map_is_even_in_x_and_y(oracle):
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(0))
    m = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)["v2map"]
    np.testing.assert_allclose(m, m[:, :, ::-1], rtol=1e-13)
    np.testing.assert_allclose(m, m[:, ::-1, :], rtol=1e-13)


def test_linear_in_upsilon_and_mass_and_scales_with_distance(oracle):
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(1), mbh=0.0)
    base = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)
    d2 = dyn.copy(); d2[:, 3] *= 3.0
    ups = oracle.jam_vrms_batch(d2, lum, mass, beta, kin, want_maps=True)
    np.testing.assert_allclose(ups["v2map"], 3.0 * base["v2map"], rtol=1e-6)       # V^2 linear in Upsilon
    np.testing.assert_allclose(ups["vrms"], math.sqrt(3.0) * base["vrms"], rtol=1e-6)
    m2 = mass.copy(); m2[..., 0] *= 3.0
    scaled = oracle.jam_vrms_batch(dyn, lum, m2, beta, kin, want_maps=True)
    np.testing.assert_allclose(scaled["v2map"], ups["v2map"], rtol=1e-6)           # same as scaling the table
    # fixed angular model in Msun/pc^2: V^2 = G * (pc/arcsec) * Phi(arcsec units)  =>  V^2 ~ D_d   (R-D8)
    d3 = dyn.copy(); d3[:, 1] *= 1.5
    far = oracle.jam_vrms_batch(d3, lum, mass, beta, kin)
    np.testing.assert_allclose(far["vrms"], math.sqrt(1.5) * base["vrms"], rtol=1e-6)
    # luminosity scale drops out of v_rms
    l2 = lum.copy(); l2[:, 0] *= 7.0
    np.testing.assert_allclose(oracle.jam_vrms_batch(dyn, l2, mass, beta, kin)["vrms"], base["vrms"], rtol=1e-6)


def test_vrms_at_fixed_angular_kappa_scales_as_inverse_sqrt_Dd(oracle):
    """Eq. 29: with the mass given as a convergence (Sigma = Sigma_crit kappa, Sigma_crit ~ 1/D_d^2 at
    fixed D_dt, Eq. 13) v_rms ~ D_d^(-1/2)."""
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(2), mbh=0.0)
    base = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)["vrms"]
    f = 1.3
    d2 = dyn.copy(); d2[:, 1] *= f
    m2 = mass.copy(); m2[..., 0] /= f * f
    np.testing.assert_allclose(oracle.jam_vrms_batch(d2, lum, m2, beta, kin)["vrms"], base / math.sqrt(f), rtol=1e-6)


def test_round_isotropic_model_is_independent_of_inclination(oracle):
    rng = np.random.default_rng(3)
    dyn, lum, mass, beta, kin = small_problem(rng, per_gaussian=False)
    lum[:, 2] = 1.0; mass[..., 2] = 1.0; beta[:] = 0.0
    dyn[:, 1:] = dyn[0, 1:]; mass[:] = mass[0]
    out = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)["v2map"]
    np.testing.assert_allclose(out[1], out[0], rtol=1e-6)
    np.testing.assert_allclose(out[2], out[0], rtol=1e-6)
    np.testing.assert_allclose(out[0], out[0].T, rtol=1e-6)                        # and circularly symmetric


def test_scalar_beta_equals_per_gaussian_beta_and_shared_equals_per_vector_tables(oracle):
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(4), per_gaussian=False)
    a = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)
    b = oracle.jam_vrms_batch(dyn, np.broadcast_to(lum, (3,) + lum.shape).copy(), mass,
                              np.repeat(beta[:, None], lum.shape[0], 1), kin)
    np.testing.assert_allclose(a["vrms"], b["vrms"], rtol=1e-14)
    c = oracle.jam_vrms_batch(dyn[:1], lum, mass[0], beta[:1], kin)                # shared mass table
    np.testing.assert_allclose(c["vrms"][0], a["vrms"][0], rtol=1e-14)


def test_bh_gaussian_equals_explicit_mass_gaussian(oracle):
    """Reading R-D3: M_BH enters as one extra round Gaussian of sigma 0.01" with Sigma0 = M/(2 pi sigma^2)."""
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(5), B=1, mbh=4e9)
    a = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)
    s = float(dyn[0, 1]) * math.pi / 0.648
    ups = float(np.float32(dyn[0, 3]))
    row = np.array([[[4e9 / (2 * math.pi * (0.01 * s) ** 2) / ups, 0.01, 1.0]]])
    d0 = dyn.copy(); d0[:, 2] = 0.0
    b = oracle.jam_vrms_batch(d0, lum, np.concatenate([mass, row], 1), beta, kin)
    np.testing.assert_allclose(a["vrms"], b["vrms"], rtol=2e-7)
    assert (a["vrms"] > oracle.jam_vrms_batch(d0, lum, mass, beta, kin)["vrms"]).all()


def test_quadrature_convergence_of_default_rule(oracle):
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(6), B=1)
    ref_kin = dict(kin); un, uw = u_nodes(4000)
    ref_kin["u_nodes"], ref_kin["u_weights"] = un.astype(np.float32), uw.astype(np.float32)
    ref = oracle.jam_vrms_batch(dyn, lum, mass, beta, ref_kin, want_maps=True)["v2map"]
    for n, tol in ((64, 1e-5), (128, 1e-6)):
        k = dict(kin); un, uw = u_nodes(n)
        k["u_nodes"], k["u_weights"] = un.astype(np.float32), uw.astype(np.float32)
        got = oracle.jam_vrms_batch(dyn, lum, mass, beta, k, want_maps=True)["v2map"]
        assert np.max(np.abs(got / ref - 1)) < tol


# ------------------------------------------------------------------ PSF / bins / chi2 (rows a7-a8)
def test_constant_field_is_returned_in_every_bin(oracle):
    rng = np.random.default_rng(7)
    sb = rng.uniform(1.0, 5.0, (9, 11))
    kern = rng.uniform(0.0, 1.0, (5, 5))
    bins = rng.integers(-1, 4, (9, 11)).astype(np.int32); bins.flat[:4] = np.arange(4)
    vr, _, bad = oracle.kin_bins(123.0 ** 2 * sb, sb, bins, 4, kern)
    assert bad == 0
    np.testing.assert_allclose(vr, 123.0, rtol=1e-12)


def test_delta_kernel_single_pixel_bins_reproduce_raw_map_and_chi2(oracle):
    rng = np.random.default_rng(8)
    sb = rng.uniform(1.0, 5.0, (4, 5)); sv2 = rng.uniform(1e4, 9e4, (4, 5)) * sb
    bins = np.arange(20, dtype=np.int32).reshape(4, 5)
    obs = rng.uniform(100, 300, 20).astype(np.float32); ivar = rng.uniform(0.01, 0.1, 20).astype(np.float32)
    vr, chi2, bad = oracle.kin_bins(sv2, sb, bins, 20, np.ones((1, 1)), obs, ivar)
    np.testing.assert_allclose(vr, np.sqrt(sv2 / sb).ravel(), rtol=1e-14)
    assert chi2 == pytest.approx(float(np.sum(ivar.astype(np.float64) * (obs.astype(np.float64) - vr) ** 2)), rel=1e-13)


def test_kin_convolution_is_true_convolution_zero_padded_and_luminosity_weighted(oracle):
    rng = np.random.default_rng(9)
    ny, nx, kk, c = 6, 7, 3, 1
    sb = rng.uniform(1.0, 5.0, (ny, nx)); sv2 = rng.uniform(1e4, 9e4, (ny, nx)) * sb
    kern = rng.uniform(0.1, 1.0, (kk, kk)).astype(np.float32)
    bins = rng.integers(0, 3, (ny, nx)).astype(np.int32); bins[2, 3] = -1
    num = np.zeros((ny, nx)); den = np.zeros((ny, nx))
    for y in range(ny):
        for x in range(nx):
            for dy in range(kk):
                for dx in range(kk):
                    sy, sx = y - (dy - c), x - (dx - c)
                    if 0 <= sy < ny and 0 <= sx < nx:
                        num[y, x] += float(kern[dy, dx]) * sv2[sy, sx]
                        den[y, x] += float(kern[dy, dx]) * sb[sy, sx]
    expect = [math.sqrt(num[bins == l].sum() / den[bins == l].sum()) for l in range(3)]
    vr, _, bad = oracle.kin_bins(sv2, sb, bins, 3, kern)
    np.testing.assert_allclose(vr, expect, rtol=1e-13)
    # empty bin -> NaN + bad
    vr, chi2, bad = oracle.kin_bins(sv2, sb, bins, 4, kern)
    assert bad == 1 and math.isnan(vr[3])


def test_undeprojectable_vector_is_flagged(oracle):
    dyn, lum, mass, beta, kin = small_problem(np.random.default_rng(10))
    dyn[1, 0] = math.radians(30.0)                            # cos^2 i = 0.75 > q'^2  (Eq. 22)
    out = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)
    assert out["flags"].tolist() == [0, oracle.FLAG_DYN_INVALID, 0]
    assert np.isnan(out["vrms"][1]).all() and np.isinf(out["chi2"][1]) and np.isfinite(out["chi2"][[0, 2]]).all()
