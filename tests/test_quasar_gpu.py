"""GPU parity for SURVEY.md 8(f) rank 4 (quasar part): chi^2_img and chi^2_tmd (Eq. 35-36) of quasar_kernel and the full joint
entry (glad_joint_loglike_full_batch) against the fp64 oracle on the same seeded inputs.

Tolerances: both sides are fp64, so where the Newton iteration of "map it back" has converged on the oracle side
(last step < 1e-10 arcsec) predicted positions agree to 1e-9 arcsec, delays to 1e-7 relative (+1e-7 d), and the two chi^2
(returned as fp32) to 2e-6 relative; the joint log-likelihood keeps BASELINE.json's 1e-5.  Vectors far from the data, for which the
twelve Newton steps wander (chaotic in the last bits on either side), must still give a finite or infinite -- never NaN -- chi^2."""
import numpy as np
import pytest

import workloads
from quasar_util import RXJ_LIKE, mock_quasar
from test_oracle_lens import lens_vec

pytestmark = pytest.mark.gpu

LUM_RANGE, MASS_RANGE = (0.02, 10.0), (0.02, 50.0)


@pytest.fixture(scope="module")
def glad_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2504_01302_b200 as m
    return m


def truth(oracle):
    p = lens_vec(bh=oracle.bh_theta2(5e9, 1823.0, 0.295), **RXJ_LIKE)
    return p.astype(np.float32).astype(np.float64), np.array([0.08, -0.05])


def chain(p, B, seed, scale=1.0):
    """B vectors scattered about p like a converged MCMC chain (element 0 = p)."""
    rng = np.random.default_rng(seed)
    lens = np.tile(p, (B, 1))
    for col, s in ((0, 0.003), (1, 0.003), (2, 0.01), (3, 0.03), (4, 0.015), (5, 0.02), (6, 0.005), (7, 0.03)):
        lens[1:, col] += rng.normal(0, s * scale, B - 1)
    lens[1:, 8] *= np.exp(rng.normal(0, 0.3, B - 1))
    lens[:, 4] = np.minimum(lens[:, 4], 1.0)
    ddt = 1823.0 + rng.normal(0, 80.0, B)
    ddt[0] = 1823.0
    return lens.astype(np.float32), ddt.astype(np.float32)


def compare(out, ref, converged):
    c = converged
    assert c.sum() > 0
    np.testing.assert_allclose(out["beta"].cpu().numpy(), ref["beta"], rtol=0, atol=1e-10)     # no iteration involved
    np.testing.assert_allclose(out["theta_pre"].cpu().numpy()[c], ref["theta_pre"][c], rtol=0, atol=1e-9)
    np.testing.assert_allclose(out["dt_pre"].cpu().numpy()[c], ref["dt_pre"][c], rtol=1e-7, atol=1e-7)
    for k in ("chi2_img", "chi2_tmd"):
        got = out[k].cpu().numpy().astype(np.float64)
        np.testing.assert_allclose(got[c], ref[k][c], rtol=2e-6, atol=1e-9)
        assert not np.isnan(got).any()


@pytest.mark.parametrize("B,scale", [(1, 1.0), (5, 1.0), (257, 1.0), (1024, 2.0), (8192, 1.5)])   # up to BASELINE.json's largest batch
def test_quasar_terms_match_oracle_on_a_chain(glad_mod, oracle, B, scale):
    p, beta = truth(oracle)
    q = mock_quasar(oracle, p, beta, 1823.0, seed=3)
    lens, ddt = chain(p, B, seed=B, scale=scale)
    g = glad_mod.Glad(0)
    g.set_quasar_data(q)
    out = g.quasar_chi2_batch(lens, ddt)
    ref = oracle.quasar_batch(lens, ddt, q)
    conv = np.all(ref["last_step"] < 1e-10, axis=1)
    assert conv.mean() > 0.9 and conv[0]
    compare(out, ref, conv)
    assert g.launch_count == 1
    # chi2 only
    o2 = g.quasar_chi2_batch(lens, ddt, want_details=False)
    assert np.array_equal(o2["chi2_img"].cpu().numpy(), out["chi2_img"].cpu().numpy())
    g.close()


def test_quasar_terms_on_prior_wide_vectors_and_a_double(glad_mod, oracle):
    """C2's prior-wide draws (most are far from the quasar data) and a two-image system."""
    wl = workloads.make_workload("C2", None, B=256)
    lens, ddt = wl["lens"]["params"], wl["ddt"]
    p0 = lens[0].astype(np.float64)
    q = mock_quasar(oracle, p0, np.array([0.08, -0.05]), float(ddt[0]), seed=1)
    g = glad_mod.Glad(0)
    g.set_quasar_data(q)
    out = g.quasar_chi2_batch(lens, ddt)
    ref = oracle.quasar_batch(lens, ddt, q)
    compare(out, ref, np.all(ref["last_step"] < 1e-10, axis=1))
    # a double: source further out
    p, _ = truth(oracle)
    qd = mock_quasar(oracle, p, np.array([0.55, 0.35]), 1823.0, seed=2)
    assert len(qd["theta"]) == 2
    lens2, ddt2 = chain(p, 64, seed=9)
    g.set_quasar_data(qd)
    out = g.quasar_chi2_batch(lens2, ddt2)
    ref = oracle.quasar_batch(lens2, ddt2, qd)
    compare(out, ref, np.all(ref["last_step"] < 1e-10, axis=1))
    # positions only (no delays): chi2_tmd = 0
    g.set_quasar_data(dict(theta=qd["theta"], sigma_theta=qd["sigma_theta"], ref=0))
    o3 = g.quasar_chi2_batch(lens2, ddt2)
    assert (o3["chi2_tmd"].cpu().numpy() == 0).all()
    np.testing.assert_allclose(o3["chi2_img"].cpu().numpy(), ref["chi2_img"], rtol=2e-6)
    g.close()


def test_quasar_special_lenses_and_edges(glad_mod, oracle):
    g = glad_mod.Glad(0)
    with pytest.raises(glad_mod.GladError):                     # no data set
        g.quasar_chi2_batch(np.zeros((1, 26), np.float32), np.array([1000.0], np.float32))
    # eight images (GLAD_MAX_QIMG): the four of the quad, each listed twice with different noise
    p, beta = truth(oracle)
    q = mock_quasar(oracle, p, beta, 1823.0, seed=3)
    rng = np.random.default_rng(4)
    q8 = dict(theta=np.concatenate([q["theta"], q["theta"] + rng.normal(0, 0.003, (4, 2))]),
              sigma_theta=np.full(8, 0.004), ref=q["ref"], dt_obs=np.concatenate([q["dt_obs"]] * 2),
              sigma_dt=np.concatenate([q["sigma_dt"], np.maximum(q["sigma_dt"], 0.5)]))
    g.set_quasar_data(q8)
    lens, ddt = chain(p, 33, seed=5)
    compare(g.quasar_chi2_batch(lens, ddt), oracle.quasar_batch(lens, ddt, q8), np.ones(33, bool))
    with pytest.raises(glad_mod.GladError):                     # nine images
        g.set_quasar_data(dict(theta=np.zeros((9, 2)), sigma_theta=np.ones(9), ref=0))
    with pytest.raises(glad_mod.GladError):                     # bad reference / sigma
        g.set_quasar_data(dict(theta=np.zeros((2, 2)), sigma_theta=np.ones(2), ref=2))
    with pytest.raises(glad_mod.GladError):
        g.set_quasar_data(dict(theta=np.ones((2, 2)), sigma_theta=np.array([1.0, 0.0]), ref=0))
    # point mass only, SIS (q = 1, gamma = 2), no shear: the closed-form lenses of the oracle's pins
    pm = lens_vec(thetaE=0.0, bh=0.8125)
    sis = lens_vec(thetaE=1.125)
    th = np.array([[1.2, 0.5], [-0.7, -0.3]])
    qq = dict(theta=th, sigma_theta=np.full(2, 0.01), ref=1, dt_obs=np.array([12.0, 0.0]), sigma_dt=np.array([1.0, 0.0]))
    g.set_quasar_data(qq)
    two = np.stack([pm, sis]).astype(np.float32)
    dd = np.array([1500.0, 2500.0], np.float32)
    compare(g.quasar_chi2_batch(two, dd), oracle.quasar_batch(two, dd, qq), np.ones(2, bool))
    # invalid mass models -> +inf, NaN details; the valid neighbours are untouched
    bad = np.tile(p, (5, 1)).astype(np.float32)
    bad[1, 3], bad[2, 4], bad[3, 2] = 3.2, 0.0, -1.0
    g.set_quasar_data(q)
    out = g.quasar_chi2_batch(bad, np.full(5, 1823.0, np.float32))
    c2 = out["chi2_img"].cpu().numpy()
    assert np.isposinf(c2[1:4]).all() and np.isposinf(out["chi2_tmd"].cpu().numpy()[1:4]).all()
    assert np.isnan(out["theta_pre"].cpu().numpy()[1:4]).all() and np.isfinite(c2[[0, 4]]).all() and c2[0] == c2[4]
    g.set_quasar_data(None)                                     # cleared
    with pytest.raises(glad_mod.GladError):
        g.quasar_chi2_batch(bad, np.full(5, 1823.0, np.float32))
    g.close()


def test_full_joint_matches_oracle(glad_mod, oracle):
    """Eq. 53: one sampler vector -> MGE tables, theta_E,BH -> pixel chi2 + chi2_dyn + chi2_img + chi2_tmd."""
    def dm(w):
        img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0]
        d = w["dyn"]
        vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
        return img, vr
    B, n_lum, n_mass = 10, 20, 20
    wl = workloads.make_workload("C2", dm, B=B)
    L, D = wl["lens"], wl["dyn"]
    lens = L["params"].copy()
    # a chain near the truth in the mass parameters, so that the quasar terms are meaningful for every vector
    lens[1:, :9] = chain(lens[0].astype(np.float64), B, seed=21)[0][1:, :9]
    l2, lum, mass = oracle.model_tables(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, n_mass, LUM_RANGE, MASS_RANGE)
    q = mock_quasar(oracle, l2[0].astype(np.float64), lens[0, 9:11].astype(np.float64), float(wl["ddt"][0]), seed=8)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    with pytest.raises(glad_mod.GladError):                     # quasar data not set
        g.joint_loglike_full_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    g.set_quasar_data(q)
    out = g.joint_loglike_full_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    ol = oracle.lens_image_batch(l2, L["grid"], L["psf"], L["data"], L["ivar"], want_images=False)
    od = oracle.jam_vrms_batch(D["params"], lum, mass, D["beta"], D["kin"])
    oq = oracle.quasar_batch(l2, wl["ddt"], q)
    assert np.all(oq["last_step"] < 1e-10)
    ref = -0.5 * (ol["chi2"] + od["chi2"] + oq["chi2_img"] + oq["chi2_tmd"])
    ll = out["loglike"].cpu().numpy().astype(np.float64)
    assert (out["flags"].cpu().numpy() == 0).all() and np.isfinite(ref).all()
    assert np.max(np.abs(ll - ref) / np.abs(ref)) < 1e-5, (ll, ref)
    np.testing.assert_allclose(out["chi2_img"].cpu().numpy(), oq["chi2_img"], rtol=2e-6)
    np.testing.assert_allclose(out["chi2_tmd"].cpu().numpy(), oq["chi2_tmd"], rtol=2e-6)
    # the quasar terms change lnL by exactly their half-sum (same kernels otherwise), with and without the side stream
    base = g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    assert np.array_equal(base["chi2_lens"].cpu().numpy(), out["chi2_lens"].cpu().numpy())
    assert np.array_equal(base["chi2_dyn"].cpu().numpy(), out["chi2_dyn"].cpu().numpy())
    g.set_overlap(False)
    o1 = g.joint_loglike_full_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE, D["beta"])
    assert np.array_equal(o1["loglike"].cpu().numpy(), out["loglike"].cpu().numpy())
    g.close()
