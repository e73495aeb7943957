"""Pins of the JAM_sph oracle (oracle/jam_sph_oracle.c) against things other than itself:
Poisson's equation for the MGE potential it integrates, the paper's Jeans equations (Eq. 17-18) checked by finite
differences of the computed moments, brute-force spherical Jeans integration with constant anisotropy (scipy.integrate.quad),
the independently pinned CYLINDRICAL oracle at beta = 0 (both alignments are then the same semi-isotropic model), and the
invariants.  A dropped term, a wrong sign / exponent / Jacobian or a swapped angle fails at least one of them."""
import math

import numpy as np
import pytest
from scipy import integrate, special

import workloads

G = 0.004301


def gl01(n):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (x + 1.0), 0.5 * w


def fine_rules(nt=160, nu=200, decades=5.0):
    t, wt = gl01(nt)
    s, ws = gl01(nu)
    L = decades * math.log(10.0)
    u = np.exp(-L * (1.0 - s))
    return t, wt, u, L * u * ws


def mge_potential(R, z, sig_j, q_j, mass_j):
    """Phi(R, z) of Gaussians stratified on spheroids, by scipy.integrate.quad (Emsellem et al. 1994)."""
    tot = 0.0
    for s, q, M in zip(sig_j, q_j, mass_j):
        e = 1.0 - q * q
        H = lambda u: math.exp(-u * u / (2 * s * s) * (R * R + z * z / (1 - e * u * u))) / math.sqrt(1 - e * u * u)
        tot += -math.sqrt(2 / math.pi) * G * M / s * integrate.quad(H, 0, 1, epsabs=0, epsrel=1e-12, limit=200)[0]
    return tot


def test_mge_potential_satisfies_poisson():
    """The potential form the oracle differentiates is the potential of the density of Eq. 25: Laplacian by finite
    differences = 4 pi G rho."""
    sig, q, M = [300.0, 800.0], [0.6, 0.85], [1e10, 5e10]
    for (R, z) in [(150.0, 80.0), (400.0, 30.0), (50.0, 500.0)]:
        h = 2.0
        P = lambda a, b: mge_potential(a, b, sig, q, M)
        lap = ((P(R + h, z) - 2 * P(R, z) + P(R - h, z)) / h**2 + (P(R + h, z) - P(R - h, z)) / (2 * h * R)
               + (P(R, z + h) - 2 * P(R, z) + P(R, z - h)) / h**2)
        rho = sum(Mj / ((2 * math.pi) ** 1.5 * s**3 * qq) * math.exp(-(R * R + z * z / qq**2) / (2 * s * s)) for s, qq, Mj in zip(sig, q, M))
        assert lap == pytest.approx(4 * math.pi * G * rho, rel=2e-5)


def moments(oracle, r, th, lum, mass, rules):
    t, wt, u, wu = rules
    sig_k, q_k, nu0_k, beta_k = lum
    sig_j, q_j, m_j = mass
    return oracle.jam_sph_intrinsic(r, th, sig_k, q_k, nu0_k, beta_k, sig_j, q_j, m_j, 6.0 * max(sig_k), t, wt, u, wu)


@pytest.mark.parametrize("beta", [0.0, 0.3, -0.4])
def test_jeans_equations_17_and_18_hold(oracle, beta):
    """Eq. 17 and Eq. 18 with F = nu v_r^2, V = nu v_phi^2 from the oracle, their r and theta derivatives by central
    differences, and dPhi/dr, dPhi/dtheta by central differences of the scipy potential (flattened tracer and mass)."""
    lum = ([250.0, 600.0], [0.55, 0.8], [3.0, 0.7], [beta, beta])
    mass = ([120.0, 500.0, 1500.0], [0.7, 0.6, 0.9], [2e9, 4e10, 9e10])
    rules = fine_rules()
    for (r, th) in [(200.0, 0.6), (450.0, 1.2), (90.0, 0.25)]:
        hr, ht = 1e-3 * r, 1e-3
        m0 = moments(oracle, r, th, lum, mass, rules)
        F, V, nu = m0[0], m0[2], m0[3]
        dFdr = (moments(oracle, r + hr, th, lum, mass, rules)[0] - moments(oracle, r - hr, th, lum, mass, rules)[0]) / (2 * hr)
        dFdt = (moments(oracle, r, th + ht, lum, mass, rules)[0] - moments(oracle, r, th - ht, lum, mass, rules)[0]) / (2 * ht)
        Phi = lambda rr, tt: mge_potential(rr * math.sin(tt), rr * math.cos(tt), *mass)
        dPdr = (Phi(r + hr, th) - Phi(r - hr, th)) / (2 * hr)
        dPdt = (Phi(r, th + ht) - Phi(r, th - ht)) / (2 * ht)
        lhs17 = dFdr + ((1 + beta) * F - V) / r
        lhs18 = (1 - beta) * dFdt + ((1 - beta) * F - V) / math.tan(th)
        scale17 = abs(nu * dPdr) + abs(dFdr) + abs(F / r)
        scale18 = abs(nu * dPdt) + abs(dFdt) + abs(F)
        assert abs(lhs17 + nu * dPdr) < 2e-5 * scale17, (r, th, lhs17, -nu * dPdr)
        assert abs(lhs18 + nu * dPdt) < 2e-5 * scale18, (r, th, lhs18, -nu * dPdt)
        assert m0[1] == pytest.approx((1 - beta) * F, rel=1e-13)          # Eq. 20


def test_per_gaussian_anisotropy_is_a_sum_of_single_gaussian_solutions(oracle):
    """The equations are linear in nu: a tracer of two Gaussians with different beta_k = the two single-Gaussian solutions."""
    mass = ([120.0, 900.0], [0.7, 0.8], [2e9, 6e10])
    rules = fine_rules(60, 80)
    both = moments(oracle, 300.0, 0.9, ([250.0, 600.0], [0.55, 0.8], [3.0, 0.7], [0.35, -0.2]), mass, rules)
    a = moments(oracle, 300.0, 0.9, ([250.0], [0.55], [3.0], [0.35]), mass, rules)
    b = moments(oracle, 300.0, 0.9, ([600.0], [0.8], [0.7], [-0.2]), mass, rules)
    np.testing.assert_allclose(both, a + b, rtol=1e-12)


def spherical_beta_jeans(r, sig_l, nu0, sig_m, M, beta, rmax_sig=6.0):
    """nu v_r^2 (r) of the spherical Jeans equation with constant beta, by quad: r^-2b int_r^rmax s^2b nu G M(s)/s^2 ds
    (rmax = 6 sigma is reading R-SPH1's cut; the tail beyond it is below 1e-6 of the integral for r <= 3 sigma)."""
    nu = lambda s: nu0 * math.exp(-s * s / (2 * sig_l**2))
    Menc = lambda s: M * (special.erf(s / (math.sqrt(2) * sig_m)) - math.sqrt(2 / math.pi) * s / sig_m * math.exp(-s * s / (2 * sig_m**2)))
    f = lambda s: s ** (2 * beta) * nu(s) * G * Menc(s) / (s * s)
    return r ** (-2 * beta) * integrate.quad(f, r, rmax_sig * sig_l, epsabs=0, epsrel=1e-11, limit=400)[0]


@pytest.mark.parametrize("beta", [0.0, 0.4, -0.5])
def test_spherical_constant_beta_against_brute_force_jeans(oracle, beta):
    """q = 1: intrinsic nu v_r^2 against the radial Jeans integral, v_phi^2 = v_theta^2, and the projected second moment
    against 2 int (1 - beta R^2/r^2) nu v_r^2 r dr / sqrt(r^2 - R^2) (Binney & Mamon 1982)."""
    sig_l, nu0, sig_m, M = 300.0, 2.0, 500.0, 3e10
    rules = fine_rules()
    for r in (40.0, 250.0, 900.0):
        m = moments(oracle, r, 0.8, ([sig_l], [1.0], [nu0], [beta]), ([sig_m], [1.0], [M]), rules)
        assert m[0] == pytest.approx(spherical_beta_jeans(r, sig_l, nu0, sig_m, M, beta), rel=1e-8)
        assert m[2] == pytest.approx(m[1], rel=1e-12)
        assert m[0] == pytest.approx(spherical_beta_jeans(r, sig_l, nu0, sig_m, M, beta, 12.0), rel=1e-6)   # the cut's own error
    # projection through the full LOS step, with exact ratios on a fine polar grid
    rg = np.geomspace(2.0, 6.0 * sig_l, 160)
    tg = np.linspace(0, math.pi / 2, 5)
    rat = np.zeros((3, rg.size, tg.size))
    for a, r in enumerate(rg):
        f = spherical_beta_jeans(r, sig_l, nu0, sig_m, M, beta) / (nu0 * math.exp(-r * r / (2 * sig_l**2)))
        rat[0, a, :], rat[1, a, :], rat[2, a, :] = f, (1 - beta) * f, (1 - beta) * f
    z, wz = np.polynomial.legendre.leggauss(200)
    for Rp in (30.0, 200.0, 700.0):
        g = lambda r: 2 * (1 - beta * Rp * Rp / (r * r)) * spherical_beta_jeans(r, sig_l, nu0, sig_m, M, beta) * r / math.sqrt(r * r - Rp * Rp)
        ref = integrate.quad(g, Rp, 6 * sig_l, epsabs=0, epsrel=1e-9, limit=400)[0]
        for (xp, yp, inc) in [(Rp, 0.0, 1.2), (0.0, Rp, 1.2), (Rp * 0.6, Rp * 0.8, 0.7)]:
            got = oracle.jam_sph_los(xp, yp, inc, [sig_l], [1.0], [nu0], rg, tg, rat, 6.0 * sig_l, z, wz)
            assert got == pytest.approx(ref, rel=3e-4), (Rp, xp, yp, inc)


def small_case(rng, B=2, n_lum=3, n_mass=4, beta=0.0, n=6):
    lum = np.stack([rng.uniform(200, 2000, n_lum), np.geomspace(0.15, 1.5, n_lum), rng.uniform(0.65, 0.9, n_lum)], 1)
    mass = np.stack([rng.uniform(500, 5000, (B, n_mass)), np.broadcast_to(np.geomspace(0.1, 8.0, n_mass), (B, n_mass)),
                     rng.uniform(0.7, 1.0, (B, n_mass))], 2)
    dyn = np.stack([np.radians(rng.uniform(62, 85, B)), rng.uniform(600, 1000, B), np.full(B, 2e9), rng.uniform(0.8, 1.2, B)], 1)
    xs = (np.arange(n) - (n - 1) / 2) * 0.3
    ys = (np.arange(n) - (n - 1) / 2) * 0.25
    kern = np.zeros((3, 3)); kern[1, 1] = 1.0
    bins = np.arange(n * n, dtype=np.int32).reshape(n, n)
    un, uw = workloads.gauss_legendre_u(160)
    kin = dict(xs=xs.astype(np.float32), ys=ys.astype(np.float32), bin_id=bins, nbins=n * n, kernel=kern.astype(np.float32),
               vrms_obs=np.full(n * n, 250, np.float32), vrms_ivar=np.full(n * n, 0.01, np.float32), u_nodes=un, u_weights=uw)
    return dyn.astype(np.float32), lum.astype(np.float32), mass.astype(np.float32), np.full(B, beta, np.float32), kin


def test_beta_zero_equals_the_cylindrical_oracle(oracle):
    """beta_ani = 0 (v_r^2 = v_theta^2) and beta_z = 0 (v_R^2 = v_z^2) are the same semi-isotropic model, so the whole JAM_sph
    pipeline (intrinsic moments on the polar grid, interpolation, LOS integral, frames) must reproduce the cylindrical
    single-quadrature map, which is pinned by brute-force axisymmetric Jeans integration (tests/test_oracle_jam.py)."""
    dyn, lum, mass, beta, kin = small_case(np.random.default_rng(21))
    sph = workloads.jam_sph_rules(kin, panels=12, nr=64, nth=17, nz=160, sigma_max=float(lum[:, 1].max()))
    a = oracle.jam_sph_vrms_batch(dyn, lum, mass, beta, kin, sph, want_maps=True)
    c = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)
    np.testing.assert_allclose(a["v2map"], c["v2map"], rtol=1.5e-3)
    np.testing.assert_allclose(a["vrms"], c["vrms"], rtol=1e-3)
    assert (a["flags"] == 0).all()


def test_invariants_and_flags(oracle):
    rng = np.random.default_rng(22)
    dyn, lum, mass, beta, kin = small_case(rng, beta=0.25)
    sph = workloads.jam_sph_rules(kin, panels=4, nr=12, nth=6, nz=48, sigma_max=float(lum[:, 1].max()))
    a = oracle.jam_sph_vrms_batch(dyn, lum, mass, beta, kin, sph, want_maps=True)
    v2 = a["v2map"]
    np.testing.assert_allclose(v2, v2[:, ::-1, :], rtol=1e-6)                 # even in y' (symmetric grid; fp32 rule, folded theta)
    np.testing.assert_allclose(v2, v2[:, :, ::-1], rtol=1e-6)                 # even in x'
    d2 = dyn.copy(); d2[:, 2] = 0.0; d2[:, 3] *= 2.0                          # no BH, Upsilon doubled: V^2 doubles
    d1 = dyn.copy(); d1[:, 2] = 0.0
    np.testing.assert_allclose(oracle.jam_sph_vrms_batch(d2, lum, mass, beta, kin, sph)["vrms"],
                               math.sqrt(2) * oracle.jam_sph_vrms_batch(d1, lum, mass, beta, kin, sph)["vrms"], rtol=1e-6)
    bg = np.broadcast_to(beta[:, None], (2, lum.shape[0])).copy()             # scalar beta == per-Gaussian beta
    np.testing.assert_allclose(oracle.jam_sph_vrms_batch(dyn, lum, mass, bg, kin, sph)["vrms"], a["vrms"], rtol=1e-13)
    radial = oracle.jam_sph_vrms_batch(dyn, lum, mass, beta + 0.3, kin, sph, want_maps=True)
    assert np.all(radial["moments"][:, 1] / radial["moments"][:, 0] == pytest.approx(1 - 0.55, rel=1e-6))
    bad = dyn.copy(); bad[1, 0] = math.radians(20.0)
    f = oracle.jam_sph_vrms_batch(bad, lum, mass, beta, kin, sph)
    assert f["flags"].tolist() == [0, 2] and np.isnan(f["vrms"][1]).all() and np.isinf(f["chi2"][1])
    f = oracle.jam_sph_vrms_batch(dyn, lum, mass, np.array([0.2, 1.0], np.float32), kin, sph)
    assert f["flags"].tolist() == [0, 2]


def test_fixed_mesh_truncation_is_small(oracle):
    """Reported, not gated at parity (the rules are inputs): the paper's mesh (16 x 16 rectangles of 7 x 7 Kronrod nodes,
    P:360) against a much finer rule on an RXJ1131-like MGE with a 0.01" black-hole Gaussian, at three polar points."""
    pc = 775 * math.pi / 0.648
    sig_k = np.geomspace(0.02, 10.0, 12) * pc
    lum = (sig_k, np.full(12, 0.75), 1.0 / sig_k**1.5, np.full(12, 0.2))
    sig_j = np.append(np.geomspace(0.02, 50.0, 12), 0.01) * pc
    mass = (sig_j, np.append(np.full(12, 0.8), 1.0), np.append(3e10 * (sig_j[:12] / pc) ** 1.0, 5e9))
    t, w = workloads.kronrod_composite(16)
    L = 5.0 * math.log(10.0)
    coarse = (t, w, np.exp(-L * (1 - t)), L * np.exp(-L * (1 - t)) * w)
    fine = fine_rules(400, 500)
    for (r_as, th) in [(0.02, 0.5), (0.3, 1.3), (1.5, 0.9)]:
        a = moments(oracle, r_as * pc, th, lum, mass, coarse)
        b = moments(oracle, r_as * pc, th, lum, mass, fine)
        assert np.max(np.abs(a[:3] / b[:3] - 1)) < 2e-5, (r_as, a, b)
