"""Pins for the quasar terms of the oracle (Eq. 35-36, quasar part; CPU only).
Each test checks the oracle against something other than itself: finite differences of the independently pinned
deflection, the paper's convergence (Eq. B.1-B.3), textbook closed forms of the point-mass and SIS lenses, SI constants,
and images found by MINPACK instead of the oracle's Newton iteration."""
import math

import numpy as np
import pytest
import scipy.constants as sc

from quasar_util import RXJ_LIKE, fermat, find_images, mock_quasar
from test_oracle_lens import kappa_paper, lens_vec


def rand_lens(rng):
    return lens_vec(xl=rng.uniform(-0.05, 0.05), yl=rng.uniform(-0.05, 0.05), thetaE=rng.uniform(1.2, 1.9),
                    gamma=rng.uniform(1.6, 2.4), q=rng.uniform(0.5, 1.0), pa=rng.uniform(0, math.pi),
                    gext=rng.uniform(0, 0.1), phiext=rng.uniform(0, math.pi), bh=rng.uniform(0.0, 0.05))


def d5(f, x, h):
    """five-point central first derivative, O(h^4)"""
    return (-f(x + 2 * h) + 8 * f(x + h) - 8 * f(x - h) + f(x - 2 * h)) / (12 * h)


# ---------------------------------------------------------------- potential and Hessian
def test_gradient_of_potential_is_the_deflection(oracle):
    rng = np.random.default_rng(11)
    for _ in range(25):
        p = rand_lens(rng)
        x, y = rng.uniform(-2.5, 2.5, 2)
        if math.hypot(x - p[0], y - p[1]) < 0.2:
            continue
        ax, ay = oracle.deflection(p, x, y)
        gx = d5(lambda t: oracle.potential(p, t, y), x, 1e-3)
        gy = d5(lambda t: oracle.potential(p, x, t), y, 1e-3)
        assert gx == pytest.approx(ax, rel=1e-8, abs=1e-9)
        assert gy == pytest.approx(ay, rel=1e-8, abs=1e-9)


def test_hessian_is_the_jacobian_of_the_deflection_and_its_trace_is_2kappa(oracle):
    rng = np.random.default_rng(12)
    for _ in range(25):
        p = rand_lens(rng)
        x, y = rng.uniform(-2.5, 2.5, 2)
        if math.hypot(x - p[0], y - p[1]) < 0.2:
            continue
        h = oracle.hessian(p, x, y)
        axx = d5(lambda t: oracle.deflection(p, t, y)[0], x, 1e-3)
        axy = d5(lambda t: oracle.deflection(p, x, t)[0], y, 1e-3)
        ayx = d5(lambda t: oracle.deflection(p, t, y)[1], x, 1e-3)
        ayy = d5(lambda t: oracle.deflection(p, x, t)[1], y, 1e-3)
        assert h[0] == pytest.approx(axx, rel=1e-7, abs=1e-8)
        assert h[1] == pytest.approx(axy, rel=1e-7, abs=1e-8)
        assert h[1] == pytest.approx(ayx, rel=1e-7, abs=1e-8)
        assert h[2] == pytest.approx(ayy, rel=1e-7, abs=1e-8)
        # kappa of Eq. B.1-B.3 in the lens frame; shear and point mass carry no convergence
        dx, dy = x - p[0], y - p[1]
        c, s = math.cos(p[5]), math.sin(p[5])
        kap = kappa_paper(dx * c + dy * s, -dx * s + dy * c, p[2], p[3], p[4])
        assert 0.5 * (h[0] + h[2]) == pytest.approx(kap, rel=1e-12)


def test_potential_closed_forms(oracle):
    # SIS: psi = theta_E r ; point mass: psi = theta_E^2 ln r ; shear along its axis: psi = +- gamma r^2 / 2
    assert oracle.potential(lens_vec(thetaE=1.3), 0.6, -0.8) == pytest.approx(1.3, rel=1e-13)
    assert oracle.potential(lens_vec(thetaE=0.0, bh=0.49), 1.2, 1.6) == pytest.approx(0.49 * math.log(2.0), rel=1e-13)
    p = lens_vec(thetaE=0.0, gext=0.07, phiext=0.3)
    assert oracle.potential(p, 2 * math.cos(0.3), 2 * math.sin(0.3)) == pytest.approx(0.5 * 0.07 * 4, rel=1e-12)
    assert oracle.potential(p, -2 * math.sin(0.3), 2 * math.cos(0.3)) == pytest.approx(-0.5 * 0.07 * 4, rel=1e-12)


def test_time_delay_constant_in_si(oracle):
    # D_dt / c (Eq. 3-4) for 1 Mpc and 1 arcsec^2, in days
    k = 1e6 * sc.parsec / sc.c / sc.day * sc.arcsec ** 2
    assert oracle.tdelay_const() == pytest.approx(k, rel=1e-9)
    assert oracle.tdelay_const() == pytest.approx(0.0280005, rel=1e-5)


# ---------------------------------------------------------------- closed-form lenses
def qso(theta, ref=0, dt=None, sigma_theta=0.005, sigma_dt=None):
    theta = np.asarray(theta, np.float64).reshape(-1, 2)
    n = len(theta)
    return dict(theta=theta, sigma_theta=np.full(n, sigma_theta), ref=ref,
                dt_obs=np.zeros(n) if dt is None else np.asarray(dt, np.float64),
                sigma_dt=np.ones(n) if sigma_dt is None else np.asarray(sigma_dt, np.float64))


def test_point_mass_lens_textbook_images_and_delay(oracle):
    # Schneider, Ehlers & Falco: theta_pm = (beta +- sqrt(beta^2 + 4 thE^2))/2, mu_pm = 1/(1 - (thE/theta_pm)^4),
    # phi(theta_-) - phi(theta_+) = thE^2 [ u sqrt(u^2+4)/2 + ln((sqrt(u^2+4)+u)/(sqrt(u^2+4)-u)) ], u = beta/thE
    thE, beta, D = math.sqrt(0.8125), 0.35, 2100.0        # theta_E^2 exact in float32 (the oracle reads float32 vectors)
    u = beta / thE
    tp, tm = 0.5 * (beta + math.sqrt(beta ** 2 + 4 * thE ** 2)), 0.5 * (beta - math.sqrt(beta ** 2 + 4 * thE ** 2))
    p = lens_vec(thetaE=0.0, bh=thE ** 2)
    ang = 0.4   # source direction
    th = [[tp * math.cos(ang), tp * math.sin(ang)], [tm * math.cos(ang), tm * math.sin(ang)]]
    dphi = thE ** 2 * (0.5 * u * math.sqrt(u * u + 4) + math.log((math.sqrt(u * u + 4) + u) / (math.sqrt(u * u + 4) - u)))
    out = oracle.quasar_batch(p[None], [D], qso(th, ref=0, dt=[0.0, 10.0], sigma_dt=[0.0, 2.0]))
    assert out["chi2_img"][0] == pytest.approx(0.0, abs=1e-18)
    np.testing.assert_allclose(out["beta"][0], [beta * math.cos(ang), beta * math.sin(ang)], rtol=1e-12)
    np.testing.assert_allclose(out["theta_pre"][0], th, rtol=1e-12)
    dt = oracle.tdelay_const() * D * dphi
    assert out["dt_pre"][0, 1] == pytest.approx(dt, rel=1e-12)
    assert out["dt_pre"][0, 0] == 0.0
    assert out["chi2_tmd"][0] == pytest.approx(((10.0 - dt) / 2.0) ** 2, rel=1e-12)
    # magnifications through the Hessian: det(I - H) = 1 - (thE/theta)^4
    for t in (tp, tm):
        h = oracle.hessian(p, t, 0.0)
        assert (1 - h[0]) * (1 - h[2]) - h[1] ** 2 == pytest.approx(1 - (thE / t) ** 4, rel=1e-12)


def test_sis_magnification_weighted_source_and_mapping_back(oracle):
    # SIS on the x axis: images beta +- thE, mu_+ = theta_+/(theta_+ - thE), mu_- = theta_-/(theta_- + thE) < 0,
    # Fermat difference 2 thE beta.  Move the observed outer image outwards by d: its source-plane position moves by d,
    # the modelled source is the |mu|-weighted mean and the predicted images are beta_bar +- thE.
    thE, beta, d, D = 1.125, 0.3, 0.02, 1500.0             # exact in float32
    tp, tm = beta + thE + d, beta - thE
    mp, mm = tp / (tp - thE), tm / (tm + thE)
    assert mm < 0
    bbar = (abs(mp) * (beta + d) + abs(mm) * beta) / (abs(mp) + abs(mm))
    p = lens_vec(thetaE=thE)
    out = oracle.quasar_batch(p[None], [D], qso([[tp, 0.0], [tm, 0.0]], ref=0, dt=[0, 0], sigma_dt=[0, 1.0]))
    np.testing.assert_allclose(out["beta"][0], [bbar, 0.0], rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(out["theta_pre"][0], [[bbar + thE, 0.0], [bbar - thE, 0.0]], rtol=1e-12, atol=1e-14)
    c2 = ((tp - bbar - thE) ** 2 + (tm - bbar + thE) ** 2) / 0.005 ** 2
    assert out["chi2_img"][0] == pytest.approx(c2, rel=1e-10)
    assert out["dt_pre"][0, 1] == pytest.approx(oracle.tdelay_const() * D * 2 * thE * bbar, rel=1e-11)
    # a signed (not absolute) magnification weight would give a different source: make sure this pin can tell
    wrong = (mp * (beta + d) + mm * beta) / (mp + mm)
    assert abs(wrong - bbar) > 1e-3


# ---------------------------------------------------------------- general model against MINPACK images
@pytest.fixture(scope="module")
def rxj(oracle):
    p = lens_vec(bh=oracle.bh_theta2(5e9, 1823.0, 0.295), **RXJ_LIKE)
    p = p.astype(np.float32).astype(np.float64)       # the oracle reads float32 vectors
    beta = np.array([0.08, -0.05])
    return p, beta


def test_exact_images_give_zero_chi2_and_fermat_delays(oracle, rxj):
    p, beta = rxj
    q0 = mock_quasar(oracle, p, beta, 1823.0, noise=False)
    assert len(q0["theta"]) == 4                      # a quad, like RXJ1131
    out = oracle.quasar_batch(p[None], [1823.0], q0)
    assert out["chi2_img"][0] < 1e-16
    assert out["chi2_tmd"][0] < 1e-16
    np.testing.assert_allclose(out["beta"][0], beta, atol=1e-11)
    np.testing.assert_allclose(out["theta_pre"][0], q0["theta"], atol=1e-11)
    # Fermat's principle: images are stationary points of phi (Eq. 2) -- finite differences of the potential alone
    for t in q0["theta"]:
        gx = d5(lambda s: fermat(oracle, p, (s, t[1]), beta), t[0], 1e-3)
        gy = d5(lambda s: fermat(oracle, p, (t[0], s), beta), t[1], 1e-3)
        assert abs(gx) < 1e-8 and abs(gy) < 1e-8
    # delays of tens of days for an RXJ1131-like quad (Tewes et al. 2013 measure ~91 d for image D)
    assert 5.0 < np.max(np.abs(q0["dt_obs"])) < 200.0


def test_predicted_images_solve_the_lens_equation_for_the_weighted_source(oracle, rxj):
    p, beta = rxj
    q1 = mock_quasar(oracle, p, beta, 1823.0, seed=5)
    rng = np.random.default_rng(6)
    B = 16
    lens = np.tile(p, (B, 1))
    lens[1:, 2] += rng.normal(0, 0.01, B - 1)        # a chain near the truth
    lens[1:, 3] += rng.normal(0, 0.02, B - 1)
    lens[1:, 4] += rng.normal(0, 0.01, B - 1)
    lens[1:, 6] += rng.normal(0, 0.005, B - 1)
    ddt = np.full(B, 1823.0) + rng.normal(0, 50, B)
    out = oracle.quasar_batch(lens, ddt, q1)
    assert np.all(out["last_step"] < 1e-12)
    K = oracle.tdelay_const()
    for b in range(B):
        pb = lens[b].astype(np.float32).astype(np.float64)       # the oracle reads float32 vectors
        imgs = find_images(oracle, pb, out["beta"][b])           # MINPACK, not the oracle's Newton steps
        w, bsum = 0.0, np.zeros(2)
        for i, t in enumerate(q1["theta"]):
            ax, ay = oracle.deflection(pb, t[0], t[1])
            # magnification by finite differences of the deflection (not the oracle's Hessian)
            J = np.array([[1 - d5(lambda s: oracle.deflection(pb, s, t[1])[0], t[0], 1e-3),
                           -d5(lambda s: oracle.deflection(pb, t[0], s)[0], t[1], 1e-3)],
                          [-d5(lambda s: oracle.deflection(pb, s, t[1])[1], t[0], 1e-3),
                           1 - d5(lambda s: oracle.deflection(pb, t[0], s)[1], t[1], 1e-3)]])
            mu = abs(1.0 / np.linalg.det(J))
            w += mu
            bsum += mu * np.array([t[0] - ax, t[1] - ay])
            # the predicted image is the MINPACK image nearest to the observed one
            near = imgs[np.argmin(np.hypot(*(imgs - t).T))]
            np.testing.assert_allclose(out["theta_pre"][b, i], near, atol=1e-10)
        np.testing.assert_allclose(out["beta"][b], bsum / w, rtol=1e-6, atol=1e-9)
        phi = np.array([fermat(oracle, pb, out["theta_pre"][b, i], out["beta"][b]) for i in range(4)])
        dt = K * float(np.float32(ddt[b])) * (phi - phi[q1["ref"]])
        np.testing.assert_allclose(out["dt_pre"][b], dt, rtol=1e-12, atol=1e-12)
        c2i = np.sum(np.sum((q1["theta"] - out["theta_pre"][b]) ** 2, axis=1) / q1["sigma_theta"] ** 2)
        m = q1["sigma_dt"] > 0
        c2t = np.sum(((q1["dt_obs"] - dt)[m] / q1["sigma_dt"][m]) ** 2)
        assert out["chi2_img"][b] == pytest.approx(c2i, rel=1e-12)
        assert out["chi2_tmd"][b] == pytest.approx(c2t, rel=1e-9)
    # chi2 at the truth is of the order of the number of data points (4 x 2 coordinates, 3 delays)
    assert out["chi2_img"][0] < 40.0 and out["chi2_tmd"][0] < 30.0


def test_time_delay_scales_with_ddt_and_is_independent_of_reference_shift(oracle, rxj):
    p, beta = rxj
    q1 = mock_quasar(oracle, p, beta, 1823.0, seed=2)
    a = oracle.quasar_batch(np.tile(p, (2, 1)), [1000.0, 3000.0], q1)
    np.testing.assert_allclose(a["dt_pre"][1], 3.0 * a["dt_pre"][0], rtol=1e-12)
    np.testing.assert_allclose(a["theta_pre"][1], a["theta_pre"][0], rtol=0, atol=0)
    q2 = dict(q1, ref=(q1["ref"] + 1) % 4)
    b = oracle.quasar_batch(p[None], [1000.0], q2)
    np.testing.assert_allclose(b["dt_pre"][0], a["dt_pre"][0] - a["dt_pre"][0, q2["ref"]], rtol=1e-12, atol=1e-12)


def test_invalid_mass_parameters_give_infinite_chi2(oracle, rxj):
    p, beta = rxj
    q1 = mock_quasar(oracle, p, beta, 1823.0, seed=2)
    bad = np.tile(p, (3, 1))
    bad[0, 3], bad[1, 4], bad[2, 2] = 3.2, 0.0, -1.0
    out = oracle.quasar_batch(bad, [1823.0] * 3, q1)
    assert np.all(np.isinf(out["chi2_img"])) and np.all(np.isinf(out["chi2_tmd"]))
    assert np.all(np.isnan(out["theta_pre"]))


@pytest.mark.parametrize("name", ["C1", "C2"])
def test_stored_quasar_observations_fit_the_truth_vector(oracle, name):
    """workloads.quasar_data holds rounded mock observations of the truth vector: the oracle must find them consistent
    with it (chi2 of the order of the 8 + 3 data points) and inconsistent with a vector far from it."""
    import workloads
    wl = workloads.make_workload(name, None, B=8)
    q = workloads.quasar_data(name)
    out = oracle.quasar_batch(wl["lens"]["params"], wl["ddt"], q)
    assert np.all(out["last_step"][0] < 1e-12)
    assert out["chi2_img"][0] < 40.0 and out["chi2_tmd"][0] < 30.0
    assert np.median(out["chi2_img"][1:] + out["chi2_tmd"][1:]) > 1e3
