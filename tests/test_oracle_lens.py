"""Pins for the lensing half of the oracle (CPU only).  Each test checks the oracle against
something other than itself: a closed form, an invariant, a library routine or a special
case (SURVEY.md 8(c) "Pins")."""
import math

import numpy as np
import pytest
from scipy.special import gamma as gamma_fn, gammaincinv

NL = 26


def lens_vec(**kw):
    """26-vector with everything off; keywords switch components on."""
    p = np.zeros(NL)
    p[3], p[4] = 2.0, 1.0          # gamma, q (valid defaults)
    p[12], p[13], p[14] = 1.0, 1.0, 1.0
    p[17], p[18], p[19] = 1.0, 1.0, 1.0
    p[22], p[23], p[24] = 1.0, 1.0, 1.0
    names = dict(xl=0, yl=1, thetaE=2, gamma=3, q=4, pa=5, gext=6, phiext=7, bh=8, xs=9, ys=10, Ies=11,
                 Res=12, ns=13, qs=14, phis=15, Ie1=16, Re1=17, n1=18, q1=19, phi1=20, Ie2=21, Re2=22,
                 n2=23, q2=24, phi2=25)
    for k, v in kw.items():
        p[names[k]] = v
    return p


def grid(n, pix, s=1):
    return dict(nx=n, ny=n, supersample=s, pix=pix, x0=-(n - 1) / 2 * pix, y0=-(n - 1) / 2 * pix)


DELTA = np.ones((1, 1), np.float32)


# ---------------------------------------------------------------- EPL deflection
def sie_alpha(x, y, thetaE, q):
    """Textbook SIE (Kormann+94 / Keeton 01), kappa = b_TM / (2 sqrt(q^2 x^2 + y^2))."""
    b = (2.0 / (1.0 + q)) * thetaE      # Eq. B.3 at gamma = 2
    bTM = q * b
    e = math.sqrt(1.0 - q * q)
    psi = math.sqrt(q * q * x * x + y * y)
    return bTM / e * math.atan(e * x / psi), bTM / e * math.atanh(e * y / psi)


@pytest.mark.parametrize("q", [0.3, 0.6, 0.8, 0.95])
def test_epl_gamma2_equals_sie_closed_form(oracle, q):
    rng = np.random.default_rng(1)
    for _ in range(20):
        x, y = rng.uniform(-3, 3, 2)
        ax, ay = oracle.epl_alpha(x, y, 1.7, 2.0, q)
        sx, sy = sie_alpha(x, y, 1.7, q)
        assert ax == pytest.approx(sx, rel=1e-10, abs=1e-12)
        assert ay == pytest.approx(sy, rel=1e-10, abs=1e-12)


def kappa_paper(x, y, thetaE, gam, q):
    """Eq. B.1-B.3 with r_soft = 0."""
    b = (2.0 / (1.0 + q)) ** (1.0 / (gam - 1.0)) * thetaE
    R = math.sqrt(x * x + y * y / (q * q))
    return (3.0 - gam) / 2.0 * (b / R) ** (gam - 1.0)


def test_epl_divergence_is_2kappa_and_curl_free(oracle):
    rng = np.random.default_rng(2)
    h = 1e-5
    for _ in range(40):
        gam, q, thetaE = rng.uniform(1.6, 2.4), rng.uniform(0.4, 1.0), rng.uniform(0.8, 2.0)
        x, y = rng.uniform(0.2, 2.5, 2) * rng.choice([-1, 1], 2)
        f = lambda xx, yy: oracle.epl_alpha(xx, yy, thetaE, gam, q)
        dax_dx = (f(x + h, y)[0] - f(x - h, y)[0]) / (2 * h)
        day_dy = (f(x, y + h)[1] - f(x, y - h)[1]) / (2 * h)
        dax_dy = (f(x, y + h)[0] - f(x, y - h)[0]) / (2 * h)
        day_dx = (f(x + h, y)[1] - f(x - h, y)[1]) / (2 * h)
        assert 0.5 * (dax_dx + day_dy) == pytest.approx(kappa_paper(x, y, thetaE, gam, q), rel=2e-7)
        assert dax_dy - day_dx == pytest.approx(0.0, abs=2e-8)


@pytest.mark.parametrize("gam", [1.5, 1.8, 2.0, 2.3])
def test_epl_round_lens_alpha_at_einstein_radius(oracle, gam):
    for ang in (0.0, 0.7, 2.1):
        x, y = 1.3 * math.cos(ang), 1.3 * math.sin(ang)
        ax, ay = oracle.epl_alpha(x, y, 1.3, gam, 1.0)
        assert ax == pytest.approx(x, rel=1e-12, abs=1e-14)
        assert ay == pytest.approx(y, rel=1e-12, abs=1e-14)
    # power-law radial dependence |alpha| = thetaE (r/thetaE)^(2-gamma) for q = 1
    ax, _ = oracle.epl_alpha(0.4, 0.0, 1.3, gam, 1.0)
    assert ax == pytest.approx(1.3 * (0.4 / 1.3) ** (2.0 - gam), rel=1e-12)


def test_epl_rotation_by_position_angle(oracle):
    """deflection() with PA = rotating the point into the lens frame and the answer back."""
    pa, q = 0.6, 0.7
    p = lens_vec(thetaE=1.5, gamma=2.1, q=q, pa=pa, xl=0.1, yl=-0.2)
    thx, thy = 0.9, 0.4
    dx, dy = thx - 0.1, thy + 0.2
    xl = dx * math.cos(pa) + dy * math.sin(pa)
    yl = -dx * math.sin(pa) + dy * math.cos(pa)
    ax_l, ay_l = oracle.epl_alpha(xl, yl, 1.5, 2.1, q)
    ax, ay = oracle.deflection(p, thx, thy)
    assert ax == pytest.approx(ax_l * math.cos(pa) - ay_l * math.sin(pa), rel=1e-12)
    assert ay == pytest.approx(ax_l * math.sin(pa) + ay_l * math.cos(pa), rel=1e-12)
    # a lens rotated by 90 deg has its major axis on y: alpha_x(x,0) of PA=90 equals alpha_y(0,x) of PA=0
    p0 = lens_vec(thetaE=1.5, gamma=2.1, q=q, pa=0.0)
    p90 = lens_vec(thetaE=1.5, gamma=2.1, q=q, pa=math.pi / 2)
    assert oracle.deflection(p90, 0.8, 0.0)[0] == pytest.approx(oracle.deflection(p0, 0.0, 0.8)[1], rel=1e-12)


# ---------------------------------------------------------------- shear, point mass
def test_shear_matches_gradient_of_eq49_and_has_zero_convergence(oracle):
    g, phi = 0.09, 1.42
    p = lens_vec(thetaE=0.0, gext=g, phiext=phi, xl=0.05, yl=-0.03)
    psi = lambda x, y: 0.5 * g * ((x - 0.05) ** 2 + (y + 0.03) ** 2) * math.cos(
        2 * math.atan2(y + 0.03, x - 0.05) - 2 * phi)                       # Eq. 49
    h = 1e-4
    for (x, y) in [(1.0, 0.5), (-0.7, 1.2), (0.3, -2.0)]:
        ax, ay = oracle.deflection(p, x, y)
        assert ax == pytest.approx((psi(x + h, y) - psi(x - h, y)) / (2 * h), rel=1e-7, abs=1e-9)
        assert ay == pytest.approx((psi(x, y + h) - psi(x, y - h)) / (2 * h), rel=1e-7, abs=1e-9)
        div = ((oracle.deflection(p, x + h, y)[0] - oracle.deflection(p, x - h, y)[0]) +
               (oracle.deflection(p, x, y + h)[1] - oracle.deflection(p, x, y - h)[1])) / (2 * h)
        assert div == pytest.approx(0.0, abs=1e-10)                           # kappa_shear = 0


def test_point_mass_deflection(oracle):
    th2 = 0.17 ** 2
    p = lens_vec(thetaE=0.0, bh=th2, xl=0.2, yl=0.1)
    for (x, y) in [(1.0, 0.5), (-0.7, 1.2), (0.21, 0.1)]:
        ax, ay = oracle.deflection(p, x, y)
        r = math.hypot(x - 0.2, y - 0.1)
        assert math.hypot(ax, ay) == pytest.approx(th2 / r, rel=1e-12)        # |alpha| = thetaE^2/theta
        assert ax * (y - 0.1) - ay * (x - 0.2) == pytest.approx(0.0, abs=1e-14)  # radial
        assert ax * (x - 0.2) > 0                                             # pointing outward (beta = theta - alpha)
    h = 1e-5
    x, y = 0.9, -0.4
    div = ((oracle.deflection(p, x + h, y)[0] - oracle.deflection(p, x - h, y)[0]) +
           (oracle.deflection(p, x, y + h)[1] - oracle.deflection(p, x, y - h)[1])) / (2 * h)
    assert div == pytest.approx(0.0, abs=1e-9)                                # kappa = 0 off-centre


def test_bh_theta2_helper(oracle):
    # theta_E^2 = 4GM/c^2 * (1+z_d)/D_dt, with 4GM/c^2 = 2 Schwarzschild radii; R_s(Msun) = 2953.25 m
    pc_m = 3.0856775814913673e16
    th2_rad = 2 * 2953.25 * 5e9 * (1 + 0.295) / (1823e6 * pc_m)
    expected = th2_rad * (648000 / math.pi) ** 2
    assert oracle.bh_theta2(5e9, 1823.0, 0.295) == pytest.approx(expected, rel=2e-4)  # G=0.004301 is 4 digits


# ---------------------------------------------------------------- Sersic
@pytest.mark.parametrize("n", [0.5, 1.0, 2.0, 3.3, 4.0, 5.0])
def test_sersic_bn_is_root_of_incomplete_gamma(oracle, n):
    assert oracle.sersic_bn(n) == pytest.approx(gammaincinv(2 * n, 0.5), rel=1e-12)


def test_sersic_half_is_gaussian_and_Re_isophote(oracle):
    Re, Ie, q, phi = 0.3, 2.0, 0.7, 0.4
    sig2 = Re * Re / (2 * math.log(2))
    for (dx, dy) in [(0.1, 0.2), (-0.4, 0.05)]:
        x = dx * math.cos(phi) + dy * math.sin(phi)
        y = -dx * math.sin(phi) + dy * math.cos(phi)
        R2 = x * x + y * y / (q * q)                                          # paper's R
        assert oracle.sersic(dx, dy, Ie, Re, 0.5, q, phi) == pytest.approx(2 * Ie * math.exp(-R2 / (2 * sig2)), rel=1e-12)
    for n in (1.0, 2.5, 4.0):                                                 # I(R_e) = I_e on the major axis
        assert oracle.sersic(Re * math.cos(phi), Re * math.sin(phi), Ie, Re, n, q, phi) == pytest.approx(Ie, rel=1e-12)
        # minor axis reaches I_e at q*R_e
        assert oracle.sersic(-q * Re * math.sin(phi), q * Re * math.cos(phi), Ie, Re, n, q, phi) == pytest.approx(Ie, rel=1e-12)


def test_sersic_total_flux_closed_form(oracle):
    """Unlensed (theta_E = 0) lens-light image, delta PSF: sum(pixels) pix^2 = 2 pi n q Re^2 Ie e^bn bn^-2n Gamma(2n)."""
    n, Re, Ie, q = 1.0, 0.25, 1.5, 0.7
    p = lens_vec(thetaE=0.0, Ie1=Ie, Re1=Re, n1=n, q1=q, phi1=0.5)
    g = grid(160, 0.05, s=4)
    img = oracle.lens_image_batch(p[None], g, DELTA)["images"][0]
    bn = gammaincinv(2 * n, 0.5)
    flux = 2 * math.pi * n * q * Re * Re * Ie * math.exp(bn) * bn ** (-2 * n) * gamma_fn(2 * n)
    assert img.sum() * 0.05 ** 2 == pytest.approx(flux, rel=2e-4)


# ---------------------------------------------------------------- ray-shoot + image
def test_sis_ring_of_centred_gaussian_source(oracle):
    thetaE, Re = 1.0, float(np.float32(0.2))      # the batch API reads float32 parameters
    p = lens_vec(thetaE=thetaE, gamma=2.0, q=1.0, Ies=1.0, Res=Re, ns=0.5, qs=1.0)
    g = grid(41, 0.08)
    img = oracle.lens_image_batch(p[None], g, DELTA)["images"][0]
    ax = g["x0"] + np.arange(41) * 0.08
    X, Y = np.meshgrid(ax, ax)
    r = np.hypot(X, Y)
    expect = 2.0 * np.exp(-np.log(2) * ((r - thetaE) / Re) ** 2)              # I_src(|theta - thetaE|)
    m = r > 1e-9
    np.testing.assert_allclose(img[m], expect[m], rtol=1e-10, atol=1e-14)


def test_no_lens_gives_unlensed_source_and_row_is_y(oracle):
    p = lens_vec(thetaE=0.0, Ies=1.0, Res=0.3, ns=1.5, qs=0.6, phis=0.3, xs=0.2, ys=-0.1)
    g = grid(30, 0.1)
    img = oracle.lens_image_batch(p[None], g, DELTA)["images"][0]
    for (iy, ix) in [(3, 20), (17, 5), (14, 16)]:
        x, y = g["x0"] + ix * 0.1, g["y0"] + iy * 0.1                          # row index increases with +y (R-L1)
        f = lambda v: float(np.float32(v))                                    # the batch API reads float32 parameters
        assert img[iy, ix] == pytest.approx(
            oracle.sersic(x - f(0.2), y - f(-0.1), 1.0, f(0.3), 1.5, f(0.6), f(0.3)), rel=1e-12)


def test_supersampling_is_mean_of_subpixel_samples(oracle):
    p = lens_vec(thetaE=1.1, gamma=2.2, q=0.7, pa=0.4, gext=0.05, phiext=1.0, bh=0.01,
                 Ies=1.0, Res=0.2, ns=2.0, qs=0.8, phis=0.9, xs=0.05, ys=0.1, Ie1=0.1, Re1=1.0, n1=3.0, q1=0.8)
    n, pix, s = 24, 0.12, 3
    coarse = oracle.lens_image_batch(p[None], grid(n, pix, s), DELTA)["images"][0]
    fine = oracle.lens_image_batch(p[None], grid(n * s, pix / s, 1), DELTA)["images"][0]   # same extent, sub-pixel centres
    np.testing.assert_allclose(coarse, fine.reshape(n, s, n, s).mean(axis=(1, 3)), rtol=1e-10)


# ---------------------------------------------------------------- PSF, chi2
def test_psf_of_point_image_is_the_psf_unflipped(oracle):
    """A one-pixel image convolved with an asymmetric PSF reproduces the PSF (true convolution, R-L8)."""
    rng = np.random.default_rng(5)
    psf = rng.uniform(0.1, 1.0, (5, 5)).astype(np.float32)
    n, pix = 21, 0.1
    iy0, ix0 = 9, 12
    g = grid(n, pix)
    p = lens_vec(thetaE=0.0, Ies=0.5, Res=1e-3, ns=0.5, qs=1.0, xs=g["x0"] + ix0 * pix, ys=g["y0"] + iy0 * pix)
    img = oracle.lens_image_batch(p[None], g, psf)["images"][0]
    peak = 1.0                                                                # I(0) = Ie e^{bn} = 0.5 * 2
    np.testing.assert_allclose(img[iy0 - 2:iy0 + 3, ix0 - 2:ix0 + 3], peak * psf.astype(np.float64), rtol=1e-6)
    assert abs(img.sum() - peak * psf.astype(np.float64).sum()) < 1e-6


def test_unit_sum_psf_conserves_interior_flux_and_is_linear(oracle):
    rng = np.random.default_rng(6)
    psf = rng.uniform(0.0, 1.0, (7, 7))
    psf = (psf / psf.sum()).astype(np.float32)
    p = lens_vec(thetaE=0.0, Ies=1.0, Res=0.15, ns=0.5, qs=0.9)                # compact, far from the edge
    g = grid(61, 0.05)
    raw = oracle.lens_image_batch(p[None], g, DELTA)["images"][0]
    blurred = oracle.lens_image_batch(p[None], g, psf)["images"][0]
    assert blurred.sum() == pytest.approx(raw.sum() * psf.astype(np.float64).sum(), rel=1e-9)
    # direct definition on a few pixels
    c = 3
    for (iy, ix) in [(30, 30), (28, 33), (0, 0), (60, 59)]:
        acc = 0.0
        for dy in range(7):
            for dx in range(7):
                sy, sx = iy - (dy - c), ix - (dx - c)
                if 0 <= sy < 61 and 0 <= sx < 61:
                    acc += float(psf[dy, dx]) * raw[sy, sx]
        assert blurred[iy, ix] == pytest.approx(acc, rel=1e-12, abs=1e-300)


def test_chi2_definitions(oracle):
    p = lens_vec(thetaE=1.0, gamma=2.0, q=0.8, Ies=1.0, Res=0.2, ns=1.0, qs=0.9, xs=0.05)
    g = grid(32, 0.1)
    psf = np.ones((3, 3), np.float32) / 9
    m = oracle.lens_image_batch(p[None], g, psf)["images"][0]
    m32 = m.astype(np.float32)
    sig = 0.05
    ivar = np.full(m.shape, 1 / sig ** 2, np.float32)
    r = oracle.lens_image_batch(p[None], g, psf, m32, ivar)
    assert r["chi2"][0] < 1e-6                                                # d = m (to fp32 rounding of d)
    k = 3.0
    r = oracle.lens_image_batch(p[None], g, psf, (m + k * sig).astype(np.float32), ivar)
    assert r["chi2"][0] == pytest.approx(k * k * m.size, rel=1e-4)            # d = m + k sigma -> k^2 N
    ivar2 = ivar.copy()
    ivar2[:16] = 0.0                                                          # masked half
    r = oracle.lens_image_batch(p[None], g, psf, (m + k * sig).astype(np.float32), ivar2)
    assert r["chi2"][0] == pytest.approx(k * k * m.size / 2, rel=1e-4)


def test_invalid_lens_vector_is_flagged_not_an_error(oracle):
    good = lens_vec(thetaE=1.0, Ies=1.0)
    bad = lens_vec(thetaE=1.0, Ies=1.0, gamma=3.5)
    g = grid(8, 0.2)
    r = oracle.lens_image_batch(np.stack([good, bad]), g, DELTA, np.zeros((8, 8), np.float32), np.ones((8, 8), np.float32))
    assert r["flags"].tolist() == [0, oracle.FLAG_LENS_INVALID]
    assert np.isfinite(r["chi2"][0]) and np.isinf(r["chi2"][1]) and np.isnan(r["images"][1]).all()


def test_joint_additivity_and_inf_propagation(oracle):
    a = np.array([10.0, 2.0, np.inf, 4.0])
    b = np.array([1.0, np.inf, 3.0, 0.5])
    out = oracle.joint_loglike(a, b)
    assert out[0] == -5.5 and out[3] == -2.25 and out[1] == -np.inf and out[2] == -np.inf
