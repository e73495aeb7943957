"""GPU parity of the pixelated-source evidence (glad_pixsrc_evidence_batch; paper Eq. 37-43) against the dense fp64
oracle (oracle/pixsrc.py) on the same seeded inputs.  Tolerances: 1e-5 relative on the log-evidence (the
bar BASELINE.json sets for a log-likelihood), 1e-4 relative on chi2 and E_S, 1e-4 of the image maximum per model pixel; the
source pixels are compared to 2e-3 of max |s_MP| (they are the solution of a system whose condition number reaches 1e5-1e6, fed
by an fp32 contraction; the evidence is stationary in s_MP, so it does not inherit that error)."""
import numpy as np
import pytest

import workloads
from test_parity_gpu import glad_mod, oracle_data_model  # noqa: F401

pytestmark = pytest.mark.gpu

EV_RTOL, C2_RTOL, PIX_RTOL, SRC_RTOL = 1e-5, 1e-4, 1e-4, 2e-3


def _compare(out, ref, sel=None):
    sel = np.arange(ref["logev"].size) if sel is None else sel
    ok = ref["flag"] == 0
    ev = out["logev"].cpu().numpy().astype(np.float64)[sel]
    c2 = out["chi2"].cpu().numpy().astype(np.float64)[sel]
    rg = out["reg"].cpu().numpy().astype(np.float64)[sel]
    fl = out["flags"].cpu().numpy()[sel]
    assert np.array_equal(fl != 0, ~ok)
    assert np.all(ev[~ok] == -np.inf) and np.all(c2[~ok] == np.inf)
    assert np.max(np.abs(ev[ok] - ref["logev"][ok]) / np.abs(ref["logev"][ok])) < EV_RTOL
    assert np.max(np.abs(c2[ok] - ref["chi2"][ok]) / ref["chi2"][ok]) < C2_RTOL
    assert np.max(np.abs(rg[ok] - ref["reg"][ok]) / ref["reg"][ok]) < 10 * C2_RTOL
    if out["model"] is not None:
        m = out["model"].cpu().numpy().astype(np.float64)[sel]
        for b in np.nonzero(ok)[0]:
            assert np.max(np.abs(m[b] - ref["model"][b])) < PIX_RTOL * np.abs(ref["model"][b]).max()
        assert np.all(np.isnan(m[~ok]))
    if out["s_mp"] is not None:
        s = out["s_mp"].cpu().numpy().astype(np.float64)[sel]
        for b in np.nonzero(ok)[0]:
            assert np.max(np.abs(s[b] - ref["s_mp"][b])) < SRC_RTOL * np.abs(ref["s_mp"][b]).max()
        assert np.all(np.isnan(s[~ok]))


def _setup(glad_mod, oracle, name, B):
    wl = workloads.make_workload(name, oracle_data_model(oracle), B=B)
    L = wl["lens"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    return wl, L, g


@pytest.mark.parametrize("nsx,nsy", [(12, 12), (9, 14), (32, 20), (15, 13)])
def test_c1_parity_ragged_source_grids(glad_mod, oracle, nsx, nsy):
    """C1 image (40 x 40, 5 x 5 PSF); N_s = 144, 126, 640, 195: ragged 64-tiles and Cholesky panels, n_sx != n_sy; masked pixels;
    one invalid mass model, one lambda <= 0, one pixel size <= 0.  N_s = 195 is odd: the trailing update of the Cholesky then runs
    its 8-byte instantiation (rows of A do not start on 16-byte boundaries), every other size the 16-byte one."""
    from oracle import pixsrc
    wl, L, g = _setup(glad_mod, oracle, "C1", 8)
    ivar = L["ivar"].copy()
    ivar[:3, :] = 0.0
    ivar[17:20, 5:9] = 0.0
    g.set_image_data(L["grid"], L["psf"], L["data"], ivar)
    pin = workloads.pixsrc_inputs(wl, nsx, nsy)
    lens = L["params"].copy()
    lens[5, 4] = 1.3                       # q > 1
    pin["lam"][6] = 0.0
    pin["src_grids"][7, 2] = -0.01
    out = g.pixsrc_evidence_batch(lens, pin["src_grids"], pin["lam"], nsx, nsy)
    ref = pixsrc.pixsrc_batch(lens, L["grid"], L["psf"], L["data"], ivar, pin["src_grids"], pin["lam"], nsx, nsy)
    assert list(ref["flag"]) == [0, 0, 0, 0, 0, 1, 1, 1]
    _compare(out, ref)
    assert list(out["flags"].cpu().numpy()[5:]) == [glad_mod.FLAG_LENS_INVALID] * 3


def test_c2_parity_paper_sizes(glad_mod, oracle):
    """C2 image (100 x 100 = the paper's N_d ~ 1e4, 21 x 21 PSF), 32 x 32 source pixels (N_s ~ 1e3, Table 1): the whole
    batch of 300 vectors runs in two scratch chunks on the device, three of them are checked against the dense oracle."""
    from oracle import pixsrc
    wl, L, g = _setup(glad_mod, oracle, "C2", 300)
    pin = workloads.pixsrc_inputs(wl, 32, 32)
    out = g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 32, 32, want_model=True, want_source=True)
    sel = np.array([0, 151, 299])
    ref = pixsrc.pixsrc_batch(L["params"][sel], L["grid"], L["psf"], L["data"], L["ivar"], pin["src_grids"][sel], pin["lam"][sel], 32, 32)
    assert np.all(ref["flag"] == 0)
    _compare(out, ref, sel)
    ev = out["logev"].cpu().numpy()
    assert np.all(np.isfinite(ev)) and np.all(out["flags"].cpu().numpy() == 0)
    # chunking does not change results: the same vectors alone, in a scratch limit that holds one vector at a time
    one = g.pixsrc_evidence_batch(L["params"][sel], pin["src_grids"][sel], pin["lam"][sel], 32, 32, want_model=False, want_source=False,
                                  scratch_mib=64)
    assert np.allclose(one["logev"].cpu().numpy(), ev[sel], rtol=2e-6)


def test_c1_parity_maximum_source_grid(glad_mod, oracle):
    """N_s = 64 x 64 = 4096, the largest source grid the entry accepts (more source pixels than the 1600 image pixels: most of them
    are held by the regulariser alone), two vectors."""
    from oracle import pixsrc
    wl, L, g = _setup(glad_mod, oracle, "C1", 2)
    pin = workloads.pixsrc_inputs(wl, 64, 64)
    out = g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 64, 64)
    ref = pixsrc.pixsrc_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], pin["src_grids"], pin["lam"], 64, 64)
    assert np.all(ref["flag"] == 0)
    _compare(out, ref)


def test_mass_sheet_degeneracy_of_the_evidence(glad_mod, oracle):
    """Eq. 5-9: with a (numerically flat) internal sheet, lambda_int x EPL and the source plane scaled by lambda_int, L is unchanged,
    so the evidence is too - the property holds at any size and needs no oracle."""
    import torch
    wl, L, g = _setup(glad_mod, oracle, "C1", 4)
    pin = workloads.pixsrc_inputs(wl, 16, 16)
    lens = L["params"].copy()
    lens[:, 6] = 0.0                      # shear and point mass are outside the transformation
    lens[:, 8] = 0.0
    base = g.pixsrc_evidence_batch(lens, pin["src_grids"], pin["lam"], 16, 16)
    lam_int = torch.tensor([0.8, 0.9, 1.1, 0.95], dtype=torch.float32, device="cuda")
    g.set_mass_sheet(lam_int, r_core=4000.0, r_tr=8000.0)
    sg = pin["src_grids"] * lam_int.cpu().numpy()[:, None]
    # the sheet pulls rays towards its own centre = the lens centre: beta -> lam beta about the lens centre
    c = lens[:, 0:2] * (1.0 - lam_int.cpu().numpy()[:, None])
    sg[:, 0:2] += c
    sh = g.pixsrc_evidence_batch(lens, sg, pin["lam"], 16, 16)
    g.set_mass_sheet(None)
    assert np.allclose(sh["chi2"].cpu().numpy(), base["chi2"].cpu().numpy(), rtol=2e-4)
    assert np.allclose(sh["logev"].cpu().numpy(), base["logev"].cpu().numpy(), rtol=2e-5)


def test_errors(glad_mod, oracle):
    wl, L, g = _setup(glad_mod, oracle, "C1", 2)
    pin = workloads.pixsrc_inputs(wl, 8, 8)
    with pytest.raises(glad_mod.GladError):
        g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 1, 8)
    with pytest.raises(glad_mod.GladError):
        g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 80, 80)
    g2 = glad_mod.Glad(0)
    with pytest.raises(glad_mod.GladError):
        g2.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 8, 8)


def test_lambda_hat_search_on_the_device(glad_mod, oracle):
    """Eq. 43: glad_pixsrc_lambda_opt_batch against scipy's bounded maximisation of the oracle's evidence.  The optimum is flat
    (curvature of ln P in ln lambda ~ N_s/2), so lambda_hat itself is compared at 1e-3 relative; ln P(lambda_hat) at 1e-5 (the bar of
    a log-likelihood), and, as the strict check of the final pass, every output against the oracle evaluated AT the device's lambda_hat."""
    from oracle import pixsrc
    wl = workloads.make_workload("C1", oracle_data_model(oracle))
    L = wl["lens"]
    nsx, nsy = 12, 10
    pin = workloads.pixsrc_inputs(wl, nsx, nsy)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    bad = L["params"].copy(); bad[2, 3] = 3.5                          # invalid mass model: flagged, lambda_hat irrelevant
    out = g.pixsrc_lambda_opt_batch(bad, pin["src_grids"], (1e-4, 1e4), nsx, nsy)
    lh = out["lam_hat"].cpu().numpy()
    ev = out["logev"].cpu().numpy().astype(np.float64)
    fl = out["flags"].cpu().numpy()
    assert fl[2] == glad_mod.FLAG_LENS_INVALID and np.isinf(ev[2]) and (np.delete(fl, 2) == 0).all()
    Bm = pixsrc.blurring_matrix(L["psf"], L["grid"]["nx"], L["grid"]["ny"])
    for b in (0, 1, 5):
        sg = dict(nx=nsx, ny=nsy, pix=float(pin["src_grids"][b, 2]), x0=float(pin["src_grids"][b, 0]), y0=float(pin["src_grids"][b, 1]))
        ref = pixsrc.pixsrc_lambda_opt(bad[b], L["grid"], L["psf"], L["data"], L["ivar"], sg, 1e-4, 1e4, Bm)
        assert 1e-4 < ref["lam_hat"] < 1e4                             # an interior maximum
        assert lh[b] == pytest.approx(ref["lam_hat"], rel=1e-3), b
        assert ev[b] == pytest.approx(ref["logev"], rel=1e-5), b
        at = pixsrc.pixsrc_evidence(bad[b], L["grid"], L["psf"], L["data"], L["ivar"], sg, lh[b], Bm)
        assert ev[b] == pytest.approx(at["logev"], rel=1e-6)
        assert out["chi2"].cpu().numpy()[b] == pytest.approx(at["chi2"], rel=1e-4)
        assert out["reg"].cpu().numpy()[b] == pytest.approx(at["reg"], rel=1e-3)
        s = out["s_mp"].cpu().numpy()[b]
        assert np.max(np.abs(s - at["s_mp"])) < 2e-3 * np.abs(at["s_mp"]).max()
    # the fixed-lambda entry at lambda_hat gives the same numbers bit for bit (same kernels after the search)
    again = g.pixsrc_evidence_batch(bad, pin["src_grids"], lh, nsx, nsy)
    ok = fl == 0
    assert np.array_equal(again["logev"].cpu().numpy()[ok], out["logev"].cpu().numpy()[ok])
    g.close()

