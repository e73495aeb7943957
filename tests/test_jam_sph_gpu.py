"""GPU parity of the JAM_sph path (glad_jam_sph_vrms_batch) against oracle/jam_sph_oracle.c through the C
ABI: the intrinsic moment ratios on the polar grid, the projected Sigma v^2 map, v_rms per bin (1e-4 relative each), chi2 and
flags, on small ragged cases, per-Gaussian anisotropy (several characteristic families), BH-only / no-BH models, and the
RXJ1131-shaped C2 workload with the paper's 112 x 112-node mesh and 20 x 10 polar grid."""
import math

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def glad_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2504_01302_b200 as m
    return m


def case(seed, nx=14, ny=11, B=4, n_lum=5, n_mass=6, nbins=9, mbh=3e9, per_gaussian=False):
    rng = np.random.default_rng(seed)
    lum = np.stack([rng.uniform(200, 2000, n_lum), np.geomspace(0.08, 2.5, n_lum), rng.uniform(0.65, 0.95, n_lum)], 1)
    mass = np.stack([rng.uniform(500, 5000, (B, n_mass)), np.broadcast_to(np.geomspace(0.05, 20.0, n_mass), (B, n_mass)),
                     rng.uniform(0.7, 1.0, (B, n_mass))], 2)
    dyn = np.stack([np.radians(rng.uniform(62, 88, B)), rng.uniform(600, 1000, B), np.full(B, mbh), rng.uniform(0.8, 1.2, B)], 1)
    beta = rng.uniform(-0.3, 0.4, (B, n_lum) if per_gaussian else B)
    if per_gaussian:
        beta[:, 1] = beta[:, 0]                                                 # two Gaussians share a characteristic family
    xs = (np.arange(nx) - (nx - 1) / 2) * 0.11
    ys = (np.arange(ny) - (ny - 1) / 2) * 0.13
    kern = rng.uniform(0.1, 1.0, (5, 5)); kern /= kern.sum()
    bins = rng.integers(-1, nbins, (ny, nx)).astype(np.int32)
    bins.flat[:nbins] = np.arange(nbins)
    un, uw = workloads.gauss_legendre_u(8)
    kin = dict(xs=xs.astype(np.float32), ys=ys.astype(np.float32), bin_id=bins, nbins=nbins, kernel=kern.astype(np.float32),
               vrms_obs=rng.uniform(200, 300, nbins).astype(np.float32), vrms_ivar=rng.uniform(0.01, 0.05, nbins).astype(np.float32),
               u_nodes=un, u_weights=uw)
    f = np.float32
    return dyn.astype(f), lum.astype(f), mass.astype(f), beta.astype(f), kin


def compare(glad_mod, oracle, c, sph, idx=None):
    dyn, lum, mass, beta, kin = c
    g = glad_mod.Glad(0)
    g.set_kin_data(kin)
    g.set_jam_sph_rules(sph)
    out = g.jam_sph_vrms_batch(dyn, lum, mass, beta, want_map=True, want_moments=True)
    sel = slice(None) if idx is None else idx
    ref = oracle.jam_sph_vrms_batch(dyn[sel], lum, mass[sel] if mass.ndim == 3 else mass, beta[sel], kin, sph, want_maps=True)
    mom, v2, vr = out["moments"].cpu().numpy()[sel], out["v2map"].cpu().numpy()[sel], out["vrms"].cpu().numpy()[sel]
    ok = ref["flags"] == 0
    assert (out["flags"].cpu().numpy()[sel] == ref["flags"]).all()
    errs = {}
    for name, a, b in (("moments", mom, ref["moments"]), ("v2map", v2, ref["v2map"]), ("vrms", vr, ref["vrms"])):
        a, b = a[ok], b[ok]
        scale = np.maximum(np.abs(b), 1e-6 * np.abs(b).max())
        errs[name] = float(np.max(np.abs(a - b) / scale))
        assert errs[name] < 1e-4, (name, errs)
    chi, rchi = out["chi2"].cpu().numpy()[sel][ok].astype(np.float64), ref["chi2"][ok]
    slack = 2 * np.sqrt(rchi * np.sum(kin["vrms_ivar"].astype(np.float64) * (1e-4 * ref["vrms"][ok]) ** 2, axis=1)) + 1e-3
    assert (np.abs(chi - rchi) <= slack).all()
    if (~ok).any():
        assert np.isnan(vr[~ok]).all() and np.isinf(out["chi2"].cpu().numpy()[sel][~ok]).all()
    g.close()
    return errs


def test_small_ragged_case_scalar_beta(glad_mod, oracle):
    c = case(31)
    sph = workloads.jam_sph_rules(c[4], panels=3, nr=9, nth=5, nz=40, sigma_max=2.5)
    print("JAM_sph small:", compare(glad_mod, oracle, c, sph))


def test_per_gaussian_beta_groups(glad_mod, oracle):
    c = case(32, per_gaussian=True)
    sph = workloads.jam_sph_rules(c[4], panels=3, nr=7, nth=6, nz=32, sigma_max=2.5)
    print("JAM_sph per-Gaussian beta:", compare(glad_mod, oracle, c, sph))


def test_bh_only_no_bh_shared_table_and_invalid_vectors(glad_mod, oracle):
    dyn, lum, mass, beta, kin = case(33)
    sph = workloads.jam_sph_rules(kin, panels=2, nr=6, nth=4, nz=32, sigma_max=2.5)
    compare(glad_mod, oracle, (dyn, lum, mass[:, :0, :], beta, kin), sph)              # n_mass = 0: black hole only
    d0 = dyn.copy(); d0[:, 2] = 0.0
    compare(glad_mod, oracle, (d0, lum, mass, beta, kin), sph)                          # no black hole
    compare(glad_mod, oracle, (dyn, lum, mass[0], beta, kin), sph)                      # one mass table shared by the batch
    bad = dyn.copy(); bad[1, 0] = math.radians(25.0)                                    # not deprojectable
    b2 = beta.copy(); b2[2] = 1.0                                                       # beta_ani >= 1
    compare(glad_mod, oracle, (bad, lum, mass, b2, kin), sph)


def test_c2_shaped_with_the_papers_mesh(glad_mod, oracle):
    """BASELINE.json configs[1]'s dynamics inputs (80 x 80 sky grid, 60 bins, 20 + 21 Gaussians, 1024 vectors on the GPU) through
    JAM_sph with the paper's fixed mesh: 16 x 16 rectangles of 7 x 7 Kronrod nodes and a 20 x 10 polar grid; 4 vectors sampled
    against the oracle (about 1e9 quadrature terms each)."""
    wl = workloads.make_workload("C2")
    D = wl["dyn"]
    sph = workloads.jam_sph_rules(D["kin"], sigma_max=float(D["lum_mge"][..., 1].max()))
    assert sph["tau"].size == 112 and sph["un"].size == 112 and sph["rgrid"].size * sph["thgrid"].size == 200
    c = (D["params"], D["lum_mge"], D["mass_mge"], D["beta"], D["kin"])
    print("JAM_sph C2:", compare(glad_mod, oracle, c, sph, idx=np.array([0, 1, 500, 1023])))
