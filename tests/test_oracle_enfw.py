"""Pins of the eNFW / core-steep-ellipsoid oracle (oracle/glad_oracle.c `glad_oracle_enfw`; Appendix A, Eq. A.1-A.7) and
of the CSE table this repository fits (workloads/fit_cse_nfw.py): Eq. A.1 itself, the circular NFW closed forms at q = 1, Poisson's
equation / curl / Hessian by finite differences at q < 1, rotation, the image and quasar entries, and the MGE profile kind."""
import math

import numpy as np
import pytest
from scipy import integrate

import workloads


@pytest.fixture(scope="module")
def halo(oracle):
    A, s = workloads.cse_table()
    oracle.set_cse_table(A, s)
    return A, s


def F_nfw(u):
    if u < 1:
        t = math.sqrt(1 - u * u)
        return math.atanh(t) / t
    if u > 1:
        t = math.sqrt(u * u - 1)
        return math.atan(t) / t
    return 1.0


def kappa_a1(u):
    """Eq. A.1 retyped (rho_s = 1)."""
    return 0.5 / (u * u - 1) * (1 - F_nfw(u)) if u != 1 else 1 / 6


def test_table_reproduces_eq_a1(oracle, halo):
    A, s = halo
    assert (A > 0).all() and 30 <= A.size <= 44 and np.all(np.diff(s) > 0)
    for u in np.geomspace(1e-6, 1e3, 181):
        cse = float(np.sum(A * 0.5 / (s * s + u * u) ** 1.5))                     # Eq. A.3-A.4
        assert cse == pytest.approx(kappa_a1(u), rel=1e-5), u                      # Oguri quotes 1e-4
        assert oracle.nfw_kappa(u) == pytest.approx(kappa_a1(u), rel=1e-13)
    # the fit script reproduces the stored table
    from workloads.fit_cse_nfw import fit
    A2, s2, err = fit()
    assert err < 1e-5 and np.allclose(A2[A2 > 0], A, rtol=1e-9) and np.allclose(s2[A2 > 0], s, rtol=1e-12)


def test_circular_halo_against_nfw_closed_forms(oracle, halo):
    """q = 1: alpha(R) = rho_s r_s [ln(u/2) + F(u)]/u (the textbook NFW deflection in Eq. A.1's normalisation), also by direct
    quadrature of 2/R int kappa R dR; kappa = Eq. A.1; psi' = alpha."""
    rho, rs = 0.3, 11.0
    for R in (0.05, 0.7, 3.0, 11.0, 40.0):
        u = R / rs
        e = oracle.enfw([rho, rs, 1.0, 0.0], R * 0.6, R * 0.8)
        a = math.hypot(e["ax"], e["ay"])
        closed = rho * rs * (math.log(u / 2) + F_nfw(u)) / u
        quad = 2 / R * integrate.quad(lambda r: rho * kappa_a1(r / rs) * r, 0, R, epsabs=0, epsrel=1e-11)[0]
        assert closed == pytest.approx(quad, rel=1e-6)      # ln(u/2) + F(u) cancels at small u
        assert a == pytest.approx(closed, rel=2e-5)                                # the table's accuracy
        assert e["ay"] / e["ax"] == pytest.approx(0.8 / 0.6, rel=1e-12)            # radial
        assert e["kappa"] == pytest.approx(rho * kappa_a1(u), rel=1e-5)
        h = 1e-4 * R
        dpsi = (oracle.enfw([rho, rs, 1.0, 0.0], (R + h) * 0.6, (R + h) * 0.8)["psi"] - oracle.enfw([rho, rs, 1.0, 0.0], (R - h) * 0.6, (R - h) * 0.8)["psi"]) / (2 * h)
        assert dpsi == pytest.approx(a, rel=1e-6)


def test_elliptical_halo_poisson_curl_hessian_rotation(oracle, halo):
    rng = np.random.default_rng(5)
    for _ in range(12):
        rho, rs, q, phi = rng.uniform(0.1, 0.4), rng.uniform(5, 20), rng.uniform(0.4, 0.95), rng.uniform(0, math.pi)
        x, y = rng.uniform(-3, 3, 2)
        nf = [rho, rs, q, phi]
        e = oracle.enfw(nf, x, y)
        h = 1e-4
        g = lambda f, dx, dy: (oracle.enfw(nf, x + dx, y + dy)[f] - oracle.enfw(nf, x - dx, y - dy)[f]) / (2 * h)
        axx, axy, ayx, ayy = g("ax", h, 0), g("ax", 0, h), g("ay", h, 0), g("ay", 0, h)
        c, s = math.cos(phi), math.sin(phi)
        xh, yh = x * c + y * s, -x * s + y * c
        u = math.sqrt(q) / rs * math.sqrt(xh * xh + yh * yh / q**2)                 # Eq. A.2
        assert 0.5 * (axx + ayy) == pytest.approx(rho * kappa_a1(u), rel=2e-5)     # Eq. 7 with Eq. A.1
        assert abs(axy - ayx) < 1e-7 * (abs(axx) + abs(ayy))                       # curl alpha = 0
        assert np.allclose(e["h"], [axx, 0.5 * (axy + ayx), ayy], rtol=1e-6, atol=1e-9)
        assert g("psi", h, 0) == pytest.approx(e["ax"], rel=1e-6) and g("psi", 0, h) == pytest.approx(e["ay"], rel=1e-6)
        assert e["kappa"] == pytest.approx(0.5 * (e["h"][0] + e["h"][2]), rel=1e-10)
        # rotating the halo and the position together rotates alpha
        e0 = oracle.enfw([rho, rs, q, 0.0], xh, yh)
        assert e["ax"] == pytest.approx(e0["ax"] * c - e0["ay"] * s, rel=1e-10, abs=1e-14)
        assert e["ay"] == pytest.approx(e0["ax"] * s + e0["ay"] * c, rel=1e-10, abs=1e-14)


def test_halo_in_the_image_and_quasar_entries(oracle, halo):
    wl = workloads.make_workload("C1")
    L = wl["lens"]
    B = wl["B"]
    nf = workloads.enfw_params(B)
    base = oracle.lens_image_batch(L["params"], L["grid"], L["psf"])
    off = nf.copy(); off[:, 0] = 0.0
    same = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], enfw=off)      # rho_s = 0: no halo, bitwise
    assert np.array_equal(base["images"], same["images"])
    with_h = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], enfw=nf)
    assert np.max(np.abs(with_h["images"] - base["images"])) > 1e-3 * base["images"].max()
    bad = nf.copy(); bad[1, 1] = -1.0; bad[2, 2] = 1.5
    f = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], enfw=bad)
    assert f["flags"].tolist() == [0, 1, 1] + [0] * (B - 3) and np.isnan(f["images"][1]).all()
    # a pure circular NFW lens (theta_E = 0) images a centred round Gaussian source into the ring I_src(|theta - alpha(theta)|)
    v = np.zeros((1, 26), np.float32)
    v[0, 3], v[0, 4] = 2.0, 1.0
    v[0, 11], v[0, 12], v[0, 13], v[0, 14] = 1.0, 0.25, 0.5, 1.0
    grid = dict(nx=41, ny=41, supersample=1, pix=0.1, x0=-2.0, y0=-2.0)
    delta = np.ones((1, 1), np.float32)
    h1 = np.array([[0.9, 9.0, 1.0, 0.0]], np.float32)
    img = oracle.lens_image_batch(v, grid, delta, enfw=h1)["images"][0]
    xs = -2.0 + 0.1 * np.arange(41)
    for (iy, ix) in [(20, 31), (8, 14), (30, 27)]:
        R = math.hypot(xs[ix], xs[iy]); u = R / 9.0
        a = 0.9 * 9.0 * (math.log(u / 2) + F_nfw(u)) / u
        want = 2.0 * math.exp(-math.log(2.0) * ((R - a) / 0.25) ** 2)              # Sersic n = 1/2: I_e e^{b_n} exp(-b_n (r/R_e)^2), b_n = ln 2
        assert img[iy, ix] == pytest.approx(want, rel=3e-4)
    q = workloads.quasar_data("C1")
    a = oracle.quasar_batch(L["params"], wl["ddt"], q)
    b = oracle.quasar_batch(L["params"], wl["ddt"], q, enfw=off)
    assert np.array_equal(a["chi2_img"], b["chi2_img"]) and np.array_equal(a["dt_pre"], b["dt_pre"])
    c = oracle.quasar_batch(L["params"], wl["ddt"], q, enfw=nf)
    assert np.isfinite(c["chi2_img"]).all() and not np.allclose(c["chi2_img"], a["chi2_img"])


def test_mge_of_the_halo_sums_back_to_eq_a1(oracle, halo):
    """Profile kind 3 of the 1-D MGE (Eq. 44-46 applied to the CSE sum): 30 Gaussians on 0.02-300 arcsec reproduce
    scale * kappa_enfw(R) of Eq. A.1 within 1 % over 0.1-30 arcsec (the range the dynamics uses: P:406 decomposes to 50 arcsec)."""
    scale, rs, q = 3897.5 * 0.25, 12.0, 0.8
    rows = oracle.mge1d(3, [scale, rs, 0.0, q], 30, 0.02, 300.0)
    assert np.all(rows[:, 2] == q)
    for R in np.geomspace(0.1, 30.0, 25):
        got = float(np.sum(rows[:, 0] * np.exp(-R * R / (2 * rows[:, 1] ** 2))))
        assert got == pytest.approx(scale * kappa_a1(math.sqrt(q) * R / rs), rel=1e-2), R


def test_model_tables_append_the_halo_rows(oracle, halo):
    """Self-consistent joint model with the halo: the mass table = the EPL rows (unchanged) followed by Eq. 46 of
    Sigma_crit kappa_enfw; summed back it gives Sigma_crit (kappa_epl + kappa_enfw) along the major axis within 2 %."""
    wl = workloads.make_workload("C1")
    L, D = wl["lens"], wl["dyn"]
    nf = workloads.enfw_params(wl["B"])
    a = oracle.model_tables(L["params"], D["params"], wl["ddt"], wl["z_d"], 8, 12, (0.05, 8.0), (0.02, 50.0))
    b = oracle.model_tables(L["params"], D["params"], wl["ddt"], wl["z_d"], 8, 12, (0.05, 8.0), (0.02, 50.0), enfw=nf,
                            halo=dict(n=20, sigma_lo=0.03, sigma_hi=400.0))
    assert b[2].shape == (wl["B"], 32, 3) and np.array_equal(b[2][:, :12], a[2]) and np.array_equal(b[0], a[0])
    for v in (0, 3):
        sc = oracle.sigma_crit(float(wl["ddt"][v]), float(D["params"][v, 1]), wl["z_d"])
        rows = b[2][v, 12:].astype(np.float64)
        assert np.allclose(rows[:, 2], nf[v, 2])
        for R in (0.3, 1.0, 4.0):
            got = float(np.sum(rows[:, 0] * np.exp(-R * R / (2 * rows[:, 1] ** 2))))
            want = sc * float(nf[v, 0]) * kappa_a1(math.sqrt(float(nf[v, 2])) * R / float(nf[v, 1]))
            assert got == pytest.approx(want, rel=2e-2)
