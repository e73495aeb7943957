"""Pins for the oracle's 1-D multi-Gaussian expansion (Eq. 44-46).

None of these retypes the Euler sum: they check it against the exact integral transform it approximates
(closed form for a power law, numerical quadrature for a Sersic), against the profile it must reproduce when
summed back (the accuracy the paper prints), and against SI constants for Sigma_crit.
"""
import math

import numpy as np
import pytest
from scipy import integrate
from scipy.special import gamma as gamma_fn

import oracle
import workloads.generate as gen


@pytest.fixture(scope="module", autouse=True)
def _build():
    oracle.build()


@pytest.mark.parametrize("gam,q,thE", [(2.0, 0.8, 1.65), (1.8, 0.6, 1.9), (2.2, 1.0, 1.6), (2.45, 0.35, 0.7)])
def test_power_law_transform_closed_form(gam, q, thE):
    """R^-t = 2^(1-t/2)/Gamma(t/2) * int dln(sigma) sigma^-t exp(-R^2/2 sigma^2) (Mellin transform of a Gaussian),
    so for F = scale (3-g)/2 (b/R)^t the exact Eq. 44 is f = sqrt(2 pi) 2^(1-t/2)/Gamma(t/2) scale (3-g)/2 b^t sigma^-t."""
    t = gam - 1.0
    b = (2.0 / (1.0 + q)) ** (1.0 / t) * thE                      # Eq. B.3
    scale = 3897.0
    for sigma in (0.02, 0.3, 1.0, 7.0, 50.0):
        exact = math.sqrt(2 * math.pi) * 2 ** (1 - t / 2) / gamma_fn(t / 2) * scale * (3 - gam) / 2 * b ** t * sigma ** (-t)
        got = oracle.mge_f_sigma(oracle.PROFILE_EPL, [scale, thE, gam, q], sigma)
        assert abs(got / exact - 1.0) < 2e-7, (sigma, got, exact)


def test_euler_order_converges():
    """Eq. 45 is an approximation whose error falls with P (about 10^(-P/3) ... 10^(-2P/3)): P = 6 is visibly
    worse than P = 12, P = 16 agrees with the closed form to 1e-9."""
    prof, t = [1.0, 1.0, 2.0, 1.0], 1.0
    exact = math.sqrt(2 * math.pi) * 2 ** 0.5 / gamma_fn(0.5) * 0.5
    e = [abs(oracle.mge_f_sigma(oracle.PROFILE_EPL, prof, 1.0, P) / exact - 1.0) for P in (6, 12, 16)]
    assert e[0] > e[1] > e[2] or e[2] < 1e-9
    assert e[0] < 1e-3 and e[1] < 2e-7 and e[2] < 1e-9


@pytest.mark.parametrize("n,Re", [(1.0, 0.5), (2.5, 1.2), (4.0, 1.85)])
def test_sersic_transform_inverts_by_quadrature(n, Re):
    """Definition of the transform: F(R) = int dln(sigma) f(sigma)/sqrt(2 pi) exp(-R^2/2 sigma^2).  Integrating the
    oracle's f(sigma) (Eq. 45) numerically must give back the Sersic profile (itself pinned in test_oracle_lens)."""
    Ie, q = 0.7, 0.8
    prof = [Ie, Re, n, q]
    for R in (0.1 * Re, Re, 3.0 * Re):
        g = lambda ls: oracle.mge_f_sigma(oracle.PROFILE_SERSIC, prof, math.exp(ls)) / math.sqrt(2 * math.pi) * \
            math.exp(-R * R / (2 * math.exp(2 * ls)))
        val, _ = integrate.quad(g, math.log(1e-4 * Re), math.log(1e3 * Re), limit=400, epsabs=0, epsrel=1e-9)
        want = oracle.sersic(R, 0.0, Ie, Re, n, q, 0.0)
        assert abs(val / want - 1.0) < 2e-5, (R, val, want)


def _sum_back(mge, R):
    return (mge[None, :, 0] * np.exp(-R[:, None] ** 2 / (2 * mge[None, :, 1] ** 2))).sum(axis=1)


def test_21_gaussians_recover_profiles_to_paper_accuracy():
    """"fits each mass or light density profile using 21 Gaussians to recover the profile within ~0.5 %".
    Over the radii the two halves use (image +-2.5", kinematics +-1") the expansion summed back stays within 1 %
    of the profile (0.5 % in the mean) for the paper's sigma range (to 50")."""
    R = np.geomspace(0.1, 10.0, 200)
    m = oracle.mge1d(oracle.PROFILE_SERSIC, [1.0, 1.85, 4.0, 0.8], 21, 0.02, 50.0)
    want = np.array([oracle.sersic(r, 0.0, 1.0, 1.85, 4.0, 0.8, 0.0) for r in R])
    err = np.abs(_sum_back(m, R) / want - 1.0)
    assert err.max() < 0.012 and err.mean() < 0.005, (err.max(), err.mean())
    # A pure power law has no outer scale: Gaussians wider than sigma_hi = 50" are missing, which costs
    # ~1.6 % at 1" (SURVEY.md 8(d) quotes 0.2-1 % inside 1" for the same table) -- checked inside the kinematic FoV.
    gam, q, thE = 2.0, 0.8, 1.65
    Rk = np.geomspace(0.1, 1.0, 100)
    m = oracle.mge1d(oracle.PROFILE_EPL, [1.0, thE, gam, q], 21, 0.02, 50.0)
    b = (2.0 / (1.0 + q)) ** (1.0 / (gam - 1.0)) * thE
    want = (3 - gam) / 2 * (b / Rk) ** (gam - 1.0)
    err = np.abs(_sum_back(m, Rk) / want - 1.0)
    assert err.max() < 0.02 and err.mean() < 0.008, (err.max(), err.mean())
    # with the range wide enough that truncation does not matter and fine spacing, Eq. 46 converges to the profile
    m = oracle.mge1d(oracle.PROFILE_EPL, [1.0, thE, gam, q], 120, 1e-4, 1e6)
    Rin = np.geomspace(0.1, 5.0, 100)
    want = (3 - gam) / 2 * (b / Rin) ** (gam - 1.0)
    assert np.abs(_sum_back(m, Rin) / want - 1.0).max() < 1e-5


def test_rows_layout_weights_and_linearity():
    prof = [2.0, 1.2, 3.0, 0.7]
    m = oracle.mge1d(oracle.PROFILE_SERSIC, prof, 15, 0.05, 20.0)
    assert m.shape == (15, 3)
    assert np.allclose(m[:, 2], 0.7)
    assert np.allclose(m[1:, 1] / m[:-1, 1], (20.0 / 0.05) ** (1 / 14), rtol=1e-12)       # log-spaced
    assert m[0, 1] == pytest.approx(0.05, rel=1e-14) and m[-1, 1] == pytest.approx(20.0, rel=1e-12)
    dln = math.log(20.0 / 0.05) / 14
    f = [oracle.mge_f_sigma(oracle.PROFILE_SERSIC, prof, s) for s in m[:, 1]]
    w = m[:, 0] * math.sqrt(2 * math.pi) / (np.array(f) * dln)                           # Eq. 46 solved for w_n
    assert np.allclose(w[[0, -1]], 0.5, rtol=1e-12) and np.allclose(w[1:-1], 1.0, rtol=1e-12)
    m2 = oracle.mge1d(oracle.PROFILE_SERSIC, [6.0, 1.2, 3.0, 0.7], 15, 0.05, 20.0)
    assert np.allclose(m2[:, 0], 3.0 * m[:, 0], rtol=1e-12)
    with pytest.raises(ValueError):
        oracle.mge1d(4, prof, 15, 0.05, 20.0)          # kinds 0..3 exist (3 = eNFW through CSEs)
    with pytest.raises(ValueError):
        oracle.mge1d(0, prof, 15, 20.0, 0.05)


def test_epl_mge_matches_generator_closed_form():
    """workloads/generate.py builds the C2 mass tables from the closed form (no Euler sum, no trapezoid ends):
    interior rows must agree with the oracle's Eq. 45-46 to the Euler accuracy."""
    thE, gam, q, ddt, dd = 1.71, 2.07, 0.73, 2100.0, 820.0
    ref = gen._mass_mge_epl(thE, gam, q, ddt, dd, 20)
    sc = oracle.sigma_crit(ddt, dd, gen.Z_D)
    m = oracle.mge1d(oracle.PROFILE_EPL, [sc, thE, gam, q], 20, 0.02, 50.0)
    assert np.allclose(m[1:-1, 0], ref[1:-1, 0], rtol=3e-7)
    assert np.allclose(m[[0, -1], 0], 0.5 * ref[[0, -1], 0], rtol=3e-7)
    assert np.allclose(m[:, 1:], ref[:, 1:], rtol=1e-12)


def test_sigma_crit_si_units():
    """Eq. 13 in SI (CODATA G, IAU solar mass parameter, parsec) converted to Msun/pc^2; the oracle's
    G = 0.004301 (km/s)^2 pc/Msun is a 4-digit constant, hence 1e-4."""
    c, G, Msun, pc = 299792458.0, 6.6743e-11, 1.98841e30, 3.0856775814913673e16
    ddt, dd, zd = 1823.0, 775.0, 0.295
    si = c * c / (4 * math.pi * G) * (ddt * 1e6 * pc) / ((1 + zd) * (dd * 1e6 * pc) ** 2)     # kg / m^2
    want = si / Msun * pc * pc
    assert oracle.sigma_crit(ddt, dd, zd) == pytest.approx(want, rel=2e-4)
    assert 3000.0 < want < 5000.0


def test_model_tables_compose_the_joint_model():
    """R-M3: the self-consistent joint model derives lens[8], the luminous and the mass table from one vector."""
    wl = gen.make_workload("C2", None, B=3)
    lens, dyn = wl["lens"]["params"], wl["dyn"]["params"]
    ddt = np.array([1823.0, 2500.0, 1200.0], np.float32)
    l2, lum, mass = oracle.model_tables(lens, dyn, ddt, gen.Z_D, 12, 20, (0.02, 10.0), (0.02, 50.0))
    assert lum.shape == (3, 12, 3) and mass.shape == (3, 20, 3) and l2.dtype == np.float32
    for b in range(3):
        assert l2[b, 8] == pytest.approx(oracle.bh_theta2(float(dyn[b, 2]), float(ddt[b]), gen.Z_D), rel=1e-6)
        assert np.allclose(mass[b, :, 2], lens[b, 4]) and np.allclose(lum[b, :, 2], lens[b, 19])
    other = np.delete(np.arange(26), 8)
    assert np.array_equal(l2[:, other], lens[:, other])
    # element 0 is the truth vector with D_dt = 1823: its generator mass table is the same model
    ref = wl["dyn"]["mass_mge"][0]
    assert np.allclose(mass[0, 1:-1, 0], ref[1:-1, 0], rtol=1e-6)


def test_chameleon_transform_closed_form():
    """1/sqrt(R^2 + a) = sqrt(2/pi) int dln(sigma) sigma^-1 exp(-a/2 sigma^2) exp(-R^2/2 sigma^2) (Laplace transform of
    t^-1/2), so the exact Eq. 44 of the Chameleon (Eq. 47) is f = I_0/(1+q) (2/sigma)(e^{-a_c/2 sigma^2} - e^{-a_t/2 sigma^2}),
    a = 4 w^2/(1+q)^2.  Absolute accuracy of the Euler sum: ~1e-8 of the profile's scale at that sigma."""
    for I0, wc, wt, q in ((1.3, 0.1, 0.9, 0.8), (0.2, 0.03, 0.5, 0.6), (2.0, 0.4, 2.5, 1.0)):
        ac, at = 4 * wc * wc / (1 + q) ** 2, 4 * wt * wt / (1 + q) ** 2
        for sigma in (0.02, 0.1, 0.5, 2.0, 20.0):
            exact = I0 / (1 + q) * (2 / sigma) * (math.exp(-ac / (2 * sigma ** 2)) - math.exp(-at / (2 * sigma ** 2)))
            got = oracle.mge_f_sigma(oracle.PROFILE_CHAMELEON, [I0, wc, wt, q], sigma)
            assert abs(got - exact) < 3e-8 * I0 / (1 + q) * (2 / sigma), (sigma, got, exact)
    # summed back (Eq. 46), 21 Gaussians reproduce the profile over the image
    R = np.geomspace(0.1, 5.0, 100)
    m = oracle.mge1d(oracle.PROFILE_CHAMELEON, [1.3, 0.1, 0.9, 0.8], 21, 0.02, 50.0)
    want = np.array([oracle.chameleon(r, 0.0, 1.3, 0.1, 0.9, 0.8, 0.0) for r in R])
    err = np.abs(_sum_back(m, R) / want - 1.0)
    assert err.max() < 0.012, err.max()
    assert np.allclose(m[:, 2], 0.8)
