"""GPU parity for the internal mass sheet (glad_set_mass_sheet; Eq. 5-9, 50-51; SURVEY 8(f) rank 1 remainder) in the lens half, the
quasar terms and the self-consistent joint model, against the fp64 oracle on the same seeded inputs.  Tolerances are those of the
rows the sheet enters: BASELINE.json's 1e-4 per image pixel and 1e-5 on lnL, the MGE-row and quasar tolerances of test_mge_gpu.py /
test_quasar_gpu.py."""
import numpy as np
import pytest

import workloads
from quasar_util import mock_quasar
from test_mge_gpu import LUM_RANGE, MASS_RANGE, check_rows
from test_parity_gpu import check_images, rel
from test_quasar_gpu import chain, compare, truth

pytestmark = pytest.mark.gpu

RC, RT = 45.0, 45.09
SHEET = dict(rc=RC, rt=RT, n=8, sigma_lo=6.0, sigma_hi=2000.0)


@pytest.fixture(scope="module")
def glad_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2504_01302_b200 as m
    return m


def dm(oracle):
    def f(w):
        img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0]
        d = w["dyn"]
        vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
        return img, vr
    return f


@pytest.mark.parametrize("name,B,radii", [("C1", 8, (RC, RT)), ("C2", 6, (RC, RT)), ("C2", 4, (3.0, 7.0))])
def test_lens_half_with_sheet_matches_oracle(glad_mod, oracle, name, B, radii):
    wl = workloads.make_workload(name, dm(oracle), B=B)
    L = wl["lens"]
    lam = np.random.default_rng(7).uniform(0.5, 1.5, B).astype(np.float32)
    lam[0] = 1.0
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    plain = g.lens_image_batch(L["params"])
    g.set_mass_sheet(lam, *radii)
    out = g.lens_image_batch(L["params"])
    ref = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], lam=lam, sheet=radii)
    check_images(out["images"].cpu().numpy(), ref["images"])
    assert rel(out["chi2"].cpu().numpy(), ref["chi2"]) < 1e-5
    assert (out["flags"].cpu().numpy() == 0).all()
    # lambda = 1 is the model without a sheet (other kernel instantiation: equal to rounding, not bitwise)
    np.testing.assert_allclose(out["images"].cpu().numpy()[0], plain["images"].cpu().numpy()[0], rtol=2e-6, atol=1e-9)
    assert rel(out["chi2"].cpu().numpy()[1:], plain["chi2"].cpu().numpy()[1:].astype(np.float64)) > 1e-3
    # switching it off restores the plain path bitwise
    g.set_mass_sheet(None)
    again = g.lens_image_batch(L["params"])
    assert np.array_equal(again["images"].cpu().numpy(), plain["images"].cpu().numpy())
    g.close()


def test_mass_sheet_degeneracy_on_the_device(glad_mod):
    """Eq. 5-6 with a flat sheet: the image of the source shrunk by lambda (and gamma_ext -> lambda gamma_ext) is the image without."""
    wl = workloads.make_workload("C2", None, B=4)
    L = wl["lens"]
    p = L["params"].copy()
    p[:, 8] = 0.0                       # the point mass is outside the transformation
    p[:, 16] = 0.0                      # no lens light (it does not move with the source)
    p[:, 0:2] = 0.0                     # sheet and scaling about the same origin
    lam = np.array([0.6, 0.9, 1.2, 1.5], np.float32)
    q = p.copy()
    q[:, 9:11] *= lam[:, None]
    q[:, 12] *= lam
    q[:, 6] *= lam
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    ref = g.lens_image_batch(p)["images"].cpu().numpy()
    g.set_mass_sheet(lam, 4.5e4, 4.509e4)
    img = g.lens_image_batch(q)["images"].cpu().numpy()
    for b in range(4):
        assert np.max(np.abs(img[b] - ref[b])) < 1e-4 * ref[b].max()
    g.close()


def test_quasar_terms_with_sheet_match_oracle(glad_mod, oracle):
    p, beta = truth(oracle)
    q = mock_quasar(oracle, p, beta, 1823.0, seed=3)
    B = 129
    lens, ddt = chain(p, B, seed=31)
    lam = np.random.default_rng(8).normal(1.0, 0.03, B).astype(np.float32)
    lam[0] = 1.0
    g = glad_mod.Glad(0)
    g.set_quasar_data(q)
    g.set_mass_sheet(lam, RC, RT)
    out = g.quasar_chi2_batch(lens, ddt)
    ref = oracle.quasar_batch(lens, ddt, q, lam=lam, sheet=(RC, RT))
    conv = np.all(ref["last_step"] < 1e-10, axis=1)
    assert conv.mean() > 0.8 and conv[0]
    compare(out, ref, conv)
    # Eq. 9 on the device: flat sheet, gamma_ext -> lambda gamma_ext: same images, delays x lambda
    l2 = np.tile(p, (2, 1)).astype(np.float32)
    l2[:, 8] = 0.0                      # the point mass is outside the transformation
    lm = np.array([1.0, 0.8], np.float32)
    l2[1, 6] *= lm[1]
    g.set_mass_sheet(lm, 4.5e4, 4.509e4)
    o2 = g.quasar_chi2_batch(l2, np.array([1823.0, 1823.0], np.float32))
    tp, dtp = o2["theta_pre"].cpu().numpy(), o2["dt_pre"].cpu().numpy()
    np.testing.assert_allclose(tp[1], tp[0], atol=2e-7)
    np.testing.assert_allclose(dtp[1], float(lm[1]) * dtp[0], rtol=1e-5, atol=1e-5)
    g.close()


def test_joint_model_with_sheet_matches_oracle(glad_mod, oracle):
    B, n_lum, n_mass = 8, 20, 20
    wl = workloads.make_workload("C2", dm(oracle), B=B)
    L, D = wl["lens"], wl["dyn"]
    lens = L["params"].copy()
    lens[1:, :9] = chain(lens[0].astype(np.float64), B, seed=41)[0][1:, :9]
    lam = np.random.default_rng(9).uniform(0.7, 1.3, B).astype(np.float32)
    l2, lum, mass = oracle.model_tables(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, n_mass, LUM_RANGE, MASS_RANGE, lam=lam, sheet=SHEET)
    assert mass.shape == (B, n_mass + SHEET["n"], 3)
    q = mock_quasar(oracle, l2[0].astype(np.float64), lens[0, 9:11].astype(np.float64), float(wl["ddt"][0]), seed=8)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    g.set_quasar_data(q)
    g.set_mass_sheet(lam, RC, RT, SHEET["n"], SHEET["sigma_lo"], SHEET["sigma_hi"])
    out = g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"],
                                      want_tables=True)
    check_rows(out["lum_mge"].cpu().numpy(), lum.astype(np.float64), "lum")
    check_rows(out["mass_mge"].cpu().numpy(), mass.astype(np.float64), "mass")
    ol = oracle.lens_image_batch(l2, L["grid"], L["psf"], L["data"], L["ivar"], want_images=False, lam=lam, sheet=(RC, RT))
    od = oracle.jam_vrms_batch(D["params"], lum, mass, D["beta"], D["kin"])
    ok = (od["flags"] == 0) & np.isfinite(od["chi2"])
    assert ok.sum() >= B - 2 and (out["flags"].cpu().numpy()[ok] == 0).all()
    ref = -0.5 * (ol["chi2"] + od["chi2"])
    ll = out["loglike"].cpu().numpy().astype(np.float64)
    assert np.max(np.abs(ll[ok] - ref[ok]) / np.abs(ref[ok])) < 1e-5, (ll, ref)
    # every term of Eq. 53
    full = g.joint_loglike_full_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    oq = oracle.quasar_batch(l2, wl["ddt"], q, lam=lam, sheet=(RC, RT))
    okq = ok & np.all(oq["last_step"] < 1e-10, axis=1)
    reff = ref - 0.5 * (oq["chi2_img"] + oq["chi2_tmd"])
    llf = full["loglike"].cpu().numpy().astype(np.float64)
    assert okq.sum() >= B - 3
    assert np.max(np.abs(llf[okq] - reff[okq]) / np.abs(reff[okq])) < 1e-5, (llf, reff)
    # the sheet changes the dynamics: lnL differs from the run without it
    g.set_mass_sheet(None)
    base = g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    assert rel(base["chi2_dyn"].cpu().numpy()[ok], out["chi2_dyn"].cpu().numpy()[ok].astype(np.float64)) > 1e-3
    g.close()


def test_mass_sheet_errors_and_invalid_lambda(glad_mod, oracle):
    wl = workloads.make_workload("C1", None)
    L = wl["lens"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    lam = np.ones(8, np.float32)
    for bad in (dict(r_core=0.0), dict(r_core=50.0), dict(n_sheet=1), dict(n_sheet=65), dict(sigma_lo=0.0), dict(sigma_hi=1.0)):
        with pytest.raises(glad_mod.GladError):
            g.set_mass_sheet(lam, **bad)
    g.set_mass_sheet(lam[:5])                     # fewer lambdas than vectors
    with pytest.raises(glad_mod.GladError):
        g.lens_image_batch(L["params"])
    lam[3] = np.nan
    g.set_mass_sheet(lam)
    out = g.lens_image_batch(L["params"])
    fl = out["flags"].cpu().numpy()
    assert fl[3] == glad_mod.FLAG_LENS_INVALID and (np.delete(fl, 3) == 0).all()
    assert np.isposinf(out["chi2"].cpu().numpy()[3]) and np.isnan(out["images"].cpu().numpy()[3]).all()
    ref = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], lam=lam, sheet=(RC, RT))
    assert ref["flags"][3] == 1 and np.isposinf(ref["chi2"][3])
    g.close()
