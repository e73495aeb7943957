"""GPU edge cases through the C ABI: empty batch, invalid vectors, ragged / asymmetric / odd grids,
BH-only mass, K-sliced small batches, host-buffer entry point, error codes."""
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


@pytest.fixture(autouse=True, params=["tc", "simt"])
def jam_path(request, monkeypatch, glad_mod):
    """Every edge case runs on both forms of row a6: tcgen05 (default) and the FP32 SIMT kernel."""
    monkeypatch.setattr(glad_mod.Glad, "DEFAULT_JAM_PATH", request.param)
    return request.param


def u_nodes(n):
    return workloads.gauss_legendre_u(n)


def small_dyn(rng, nx, ny, xs=None, ys=None, n_lum=5, n_mass=7, nbins=9, B=5, mbh=3e9, kk=5, nu=40):
    lum = np.stack([rng.uniform(200, 2000, n_lum), np.geomspace(0.05, 3.0, n_lum), rng.uniform(0.7, 0.95, n_lum)], 1)
    mass = np.stack([rng.uniform(500, 5000, (B, n_mass)), np.broadcast_to(np.geomspace(0.04, 20.0, n_mass), (B, n_mass)),
                     rng.uniform(0.7, 1.0, (B, n_mass))], 2)
    dyn = np.stack([np.radians(rng.uniform(65, 88, B)), rng.uniform(600, 1000, B), np.full(B, mbh), rng.uniform(0.8, 1.2, B)], 1)
    beta = rng.uniform(-0.3, 0.5, (B, n_lum))
    xs = ((np.arange(nx) - (nx - 1) / 2) * 0.07) if xs is None else xs
    ys = ((np.arange(ny) - (ny - 1) / 2) * 0.09) if ys is None else ys
    un, uw = u_nodes(nu)
    kern = rng.uniform(0.1, 1.0, (kk, kk)); kern /= kern.sum()
    bins = rng.integers(-1, nbins, (ny, nx)).astype(np.int32)
    bins.flat[:nbins] = np.arange(nbins)
    kin = dict(xs=xs.astype(np.float32), ys=ys.astype(np.float32), bin_id=bins, nbins=nbins, kernel=kern.astype(np.float32),
               vrms_obs=rng.uniform(200, 300, nbins).astype(np.float32), vrms_ivar=rng.uniform(0.01, 0.05, nbins).astype(np.float32),
               u_nodes=un, u_weights=uw)
    return dyn.astype(np.float32), lum.astype(np.float32), mass.astype(np.float32), beta.astype(np.float32), kin


def compare_jam(glad_mod, oracle, dyn, lum, mass, beta, kin):
    g = glad_mod.Glad(0)
    g.set_kin_data(kin)
    out = g.jam_vrms_batch(dyn, lum, mass, beta, want_map=True)
    ref = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)
    np.testing.assert_allclose(out["v2map"].cpu().numpy(), ref["v2map"], rtol=1e-4)
    np.testing.assert_allclose(out["vrms"].cpu().numpy(), ref["vrms"], rtol=1e-4)
    np.testing.assert_allclose(out["chi2"].cpu().numpy(), ref["chi2"], rtol=2e-3)
    assert (out["flags"].cpu().numpy() == ref["flags"]).all()
    g.close()


@pytest.mark.parametrize("nx,ny", [(1, 1), (7, 5), (12, 9), (33, 18), (20, 20)])
def test_ragged_symmetric_grids_odd_and_even(glad_mod, oracle, nx, ny):
    compare_jam(glad_mod, oracle, *small_dyn(np.random.default_rng(nx * 100 + ny), nx, ny))


def test_asymmetric_grid_is_not_folded(glad_mod, oracle):
    rng = np.random.default_rng(3)
    xs = np.sort(rng.uniform(-0.9, 1.1, 13))
    ys = np.sort(rng.uniform(-0.5, 1.5, 10))
    compare_jam(glad_mod, oracle, *small_dyn(rng, 13, 10, xs=xs, ys=ys))


def test_bh_only_and_no_bh_and_shared_tables(glad_mod, oracle):
    rng = np.random.default_rng(4)
    dyn, lum, mass, beta, kin = small_dyn(rng, 10, 10)
    compare_jam(glad_mod, oracle, dyn, lum, mass[:, :0, :], beta, kin)          # n_mass = 0, BH only
    d0 = dyn.copy(); d0[:, 2] = 0.0
    compare_jam(glad_mod, oracle, d0, lum, mass, beta, kin)                      # no BH
    compare_jam(glad_mod, oracle, dyn, lum, mass[0], beta[:, 0].copy(), kin)     # shared mass table, scalar beta


def test_single_vector_uses_k_slices(glad_mod, oracle):
    dyn, lum, mass, beta, kin = small_dyn(np.random.default_rng(5), 24, 24, B=1, nu=64)
    compare_jam(glad_mod, oracle, dyn, lum, mass, beta, kin)


def test_invalid_vectors_are_flagged_not_errors(glad_mod, oracle):
    rng = np.random.default_rng(6)
    dyn, lum, mass, beta, kin = small_dyn(rng, 10, 10)
    dyn[1, 0] = math.radians(20.0)                      # not deprojectable
    dyn[3, 1] = -5.0                                    # D_d <= 0
    g = glad_mod.Glad(0)
    g.set_kin_data(kin)
    out = g.jam_vrms_batch(dyn, lum, mass, beta)
    fl = out["flags"].cpu().numpy()
    assert fl.tolist() == [0, glad_mod.FLAG_DYN_INVALID, 0, glad_mod.FLAG_DYN_INVALID, 0]
    v, c = out["vrms"].cpu().numpy(), out["chi2"].cpu().numpy()
    assert np.isnan(v[[1, 3]]).all() and np.isinf(c[[1, 3]]).all() and np.isfinite(v[[0, 2, 4]]).all()
    ref = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)
    assert (ref["flags"] == fl).all()
    # empty bin -> BIN_INVALID on every vector
    kin2 = dict(kin); kin2["nbins"] = kin["nbins"] + 1
    kin2["vrms_obs"] = np.append(kin["vrms_obs"], 250).astype(np.float32)
    kin2["vrms_ivar"] = np.append(kin["vrms_ivar"], 0.01).astype(np.float32)
    g.set_kin_data(kin2)
    out = g.jam_vrms_batch(dyn[[0]], lum, mass[[0]], beta[[0]])
    assert out["flags"].cpu().numpy()[0] == glad_mod.FLAG_BIN_INVALID and np.isinf(out["chi2"].cpu().numpy()[0])
    g.close()


def lens_vec(**kw):
    p = np.zeros(26, np.float32)
    p[3], p[4] = 2.0, 1.0
    p[12], p[13], p[14] = 1.0, 1.0, 1.0
    p[17], p[18], p[19] = 1.0, 1.0, 1.0
    p[22], p[23], p[24] = 1.0, 1.0, 1.0
    names = dict(xl=0, yl=1, thetaE=2, gamma=3, q=4, pa=5, gext=6, phiext=7, bh=8, xs=9, ys=10, Ies=11, Res=12, ns=13, qs=14,
                 phis=15, Ie1=16, Re1=17, n1=18, q1=19, phi1=20, Ie2=21, Re2=22, n2=23, q2=24, phi2=25)
    for k, v in kw.items():
        p[names[k]] = v
    return p


def test_lens_edge_cases(glad_mod, oracle):
    rng = np.random.default_rng(7)
    vecs = np.stack([
        lens_vec(thetaE=1.0, gamma=2.0, q=1.0, Ies=1.0, Res=0.2, ns=0.5, qs=1.0),                 # SIS ring, q = 1 (f = 0)
        lens_vec(thetaE=0.0, Ies=1.0, Res=0.3, ns=1.5, qs=0.6, phis=0.3, xs=0.2, ys=-0.1),        # no lens
        lens_vec(thetaE=1.2, gamma=2.4, q=0.35, pa=1.0, Ies=1.0, Res=0.25, ns=3.0, qs=0.7),       # flat, steep
        lens_vec(thetaE=1.1, gamma=1.6, q=0.7, pa=2.0, bh=0.04, gext=0.1, phiext=0.5, Ies=0.5, Res=0.2, ns=1.0,
                 qs=0.9, Ie1=0.2, Re1=1.0, n1=4.0, q1=0.8, phi1=2.0, Ie2=0.3, Re2=0.4, n2=1.2, q2=0.7, phi2=2.0),
        lens_vec(thetaE=1.0, gamma=3.5, Ies=1.0),                                                  # invalid gamma
        lens_vec(thetaE=1.1, gamma=2.1, q=0.1, pa=0.4, Ies=1.0, Res=0.3, ns=1.0, qs=0.8),         # very flat: 93 series terms
        lens_vec(thetaE=0.9, gamma=1.9, q=0.05, pa=2.2, Ies=1.0, Res=0.3, ns=2.0, qs=0.8),        # 177 terms (table holds 40)
    ])
    for (nx, ny, s, k) in [(37, 23, 2, 7), (8, 8, 1, 1), (50, 41, 3, 31)]:
        grid = dict(nx=nx, ny=ny, supersample=s, pix=0.1, x0=-(nx - 1) / 2 * 0.1 + 0.013, y0=-(ny - 1) / 2 * 0.1 - 0.02)
        psf = rng.uniform(0.0, 1.0, (k, k)); psf = (psf / psf.sum()).astype(np.float32)
        data = rng.normal(0, 1, (ny, nx)).astype(np.float32)
        ivar = rng.uniform(0.5, 2.0, (ny, nx)).astype(np.float32); ivar[0, :] = 0.0
        g = glad_mod.Glad(0)
        g.set_image_data(grid, psf, data, ivar)
        out = g.lens_image_batch(vecs)
        ref = oracle.lens_image_batch(vecs, grid, psf, data, ivar)
        fl = out["flags"].cpu().numpy()
        assert fl.tolist() == [0, 0, 0, 0, glad_mod.FLAG_LENS_INVALID, 0, 0] == ref["flags"].tolist()
        img = out["images"].cpu().numpy().astype(np.float64)
        for b in (0, 1, 2, 3, 5, 6):
            mx = np.abs(ref["images"][b]).max()
            err = np.abs(img[b] - ref["images"][b]) / np.maximum(np.abs(ref["images"][b]), 1e-6 * mx)
            assert err.max() < 1e-4, (nx, ny, s, k, b, err.max())
        ok = [0, 1, 2, 3, 5, 6]
        np.testing.assert_allclose(out["chi2"].cpu().numpy()[ok], ref["chi2"][ok], rtol=1e-5)
        assert np.isnan(img[4]).all() and np.isinf(out["chi2"].cpu().numpy()[4])
        g.close()


def test_empty_batch_state_errors_and_host_entry_point(glad_mod, oracle):
    import torch
    g = glad_mod.Glad(0)
    with pytest.raises(glad_mod.GladError):                                   # GLAD_ESTATE: no static data yet
        g.lens_image_batch(np.zeros((2, 26), np.float32))
    wl = workloads.make_workload("C1")
    L, D = wl["lens"], wl["dyn"]
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    out = g.lens_image_batch(np.zeros((0, 26), np.float32))                   # B = 0 is a no-op
    assert out["chi2"].numel() == 0
    with pytest.raises(glad_mod.GladError):                                   # even PSF size
        g.set_image_data(L["grid"], np.ones((4, 4), np.float32), L["data"], L["ivar"])
    dev = g.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"])["loglike"].cpu()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    host = torch.empty(wl["B"], dtype=torch.float32).pin_memory()
    g.joint_loglike_host(pin(L["params"]), pin(D["params"]), pin(D["lum_mge"]), pin(D["mass_mge"]), pin(D["beta"]), host)
    assert torch.equal(host, dev)                                             # same kernels, same bits
    n0 = g.launch_count
    g.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"])
    assert g.launch_count - n0 == 6                                           # 2 lens + 3 jam + 1 joint kernels
    g.close()
