"""GPU parity for the Chameleon light profile (Eq. 47, light part) through glad_set_light_profiles:
model images within 1e-4 per pixel, chi2 / lnL within 1e-5, on the C2 workload with the lens light (and then also the
source) switched to Chameleons."""
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


def chameleon_workload(B, source_too):
    wl = workloads.make_workload("C2", None, B=B)
    L = wl["lens"]
    rng = np.random.default_rng(7)
    p = L["params"].copy()
    # lens light 1 and 2 as the paper's two Chameleons (RXJ1131-like scales), same PA and centre as the mass
    for off, (c_lo, c_hi, t_lo, t_hi) in ((16, (0.05, 0.3, 1.0, 3.0)), (21, (0.02, 0.1, 0.3, 0.9))):
        p[:, off] = rng.uniform(0.01, 0.05, B)
        p[:, off + 1] = rng.uniform(c_lo, c_hi, B)
        p[:, off + 2] = rng.uniform(t_lo, t_hi, B)
        p[:, off + 3] = rng.uniform(0.6, 1.0, B)
        p[:, off + 4] = p[:, 5]
    if source_too:
        p[:, 11] = rng.uniform(0.05, 0.2, B)
        p[:, 12] = rng.uniform(0.02, 0.08, B)
        p[:, 13] = rng.uniform(0.15, 0.5, B)
    L["params"] = p.astype(np.float32)
    return wl


@pytest.mark.parametrize("source_too", [False, True])
def test_chameleon_images_and_chi2_match_oracle(glad_mod, oracle, source_too):
    B = 48
    wl = chameleon_workload(B, source_too)
    L = wl["lens"]
    kinds = [1 if source_too else 0, 1, 1]
    truth = oracle.lens_image_batch(L["params"][:1], L["grid"], L["psf"], kinds=kinds)["images"][0]
    nrng = np.random.default_rng(3)
    data = (truth + nrng.normal(0, 0.01, truth.shape)).astype(np.float32)
    ivar = np.full(truth.shape, 1e4, np.float32)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], data, ivar)
    g.set_light_profiles(*kinds)
    out = g.lens_image_batch(L["params"])
    idx = np.array([0, 1, 2, 3, 17, 47])
    ref = oracle.lens_image_batch(L["params"][idx], L["grid"], L["psf"], data, ivar, kinds=kinds)
    img = out["images"].cpu().numpy().astype(np.float64)[idx]
    for b in range(idx.size):
        mx = np.abs(ref["images"][b]).max()
        err = np.abs(img[b] - ref["images"][b]) / np.maximum(np.abs(ref["images"][b]), 1e-6 * mx)
        assert err.max() < 1e-4, (b, err.max())
    chi = out["chi2"].cpu().numpy().astype(np.float64)[idx]
    assert np.max(np.abs(chi - ref["chi2"]) / ref["chi2"]) < 1e-5
    assert (out["flags"].cpu().numpy() == 0).all()
    # back to Sersic: the same context gives the Sersic images again (the switch is per call, not sticky in scratch)
    g.set_light_profiles(0, 0, 0)
    s_out = g.lens_image_batch(wl["lens"]["params"][:2])["images"].cpu().numpy().astype(np.float64)
    s_ref = oracle.lens_image_batch(wl["lens"]["params"][:2], L["grid"], L["psf"])["images"]
    ok = np.isfinite(s_ref)
    assert np.allclose(s_out[ok], s_ref[ok], rtol=1e-4, atol=1e-10)
    g.close()


def test_chameleon_validity_and_errors(glad_mod, oracle):
    wl = chameleon_workload(4, False)
    L = wl["lens"]
    p = L["params"].copy()
    p[1, 17:19] = [0.9, 0.2]             # w_t < w_c
    p[2, 22] = 0.0                        # w_c = 0
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_light_profiles(0, 1, 1)
    out = g.lens_image_batch(p)
    ref = oracle.lens_image_batch(p, L["grid"], L["psf"], L["data"], L["ivar"], kinds=[0, 1, 1])
    assert list(out["flags"].cpu().numpy()) == list(ref["flags"]) == [0, 1, 1, 0]
    assert np.isinf(out["chi2"].cpu().numpy()[1:3]).all()
    with pytest.raises(glad_mod.GladError):
        g.set_light_profiles(0, 2, 0)
    g.close()


def test_joint_model_with_chameleon_tracer(glad_mod, oracle):
    """the paper decomposes I_light (Chameleons) into Gaussians for the dynamics.  With lens light 1 switched to a
    Chameleon the self-consistent entry expands it (GLAD_PROFILE_CHAMELEON) as the luminous tracer."""
    B = 10
    wl = chameleon_workload(B, False)
    L = wl["lens"]
    p = L["params"].copy()
    p[:, 21] = 0.0                                   # one Chameleon = the tracer; lens light 2 off
    p[:, 19] = p[:, 4]
    D = workloads.make_workload("C2", None, B=B)["dyn"]
    kinds = [0, 1, 0]
    lum_range, mass_range = (0.02, 10.0), (0.02, 50.0)
    l2, lum, mass = oracle.model_tables(p, D["params"], wl["ddt"], wl["z_d"], 16, 20, lum_range, mass_range,
                                        tracer_kind=oracle.PROFILE_CHAMELEON)
    img = oracle.lens_image_batch(l2[:1], L["grid"], L["psf"], kinds=kinds)["images"][0]
    vr = oracle.jam_vrms_batch(D["params"][:1], lum[:1], mass[:1], D["beta"][:1], D["kin"])["vrms"][0]
    nrng = np.random.default_rng(5)
    data = (img + nrng.normal(0, 0.01, img.shape)).astype(np.float32)
    ivar = np.full(img.shape, 1e4, np.float32)
    kin = dict(D["kin"])
    kin["vrms_obs"] = (vr * (1 + nrng.normal(0, 0.02, vr.shape))).astype(np.float32)
    kin["vrms_ivar"] = (1.0 / (0.02 * vr) ** 2).astype(np.float32)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], data, ivar)
    g.set_kin_data(kin)
    g.set_light_profiles(*kinds)
    out = g.joint_loglike_model_batch(p, D["params"], wl["ddt"], wl["z_d"], 16, lum_range, 20, mass_range, D["beta"], want_tables=True)
    got = out["lum_mge"].cpu().numpy().astype(np.float64)
    peak = np.abs(lum[:, :, 0]).max(axis=1, keepdims=True)
    assert (np.abs(got[:, :, 0] - lum[:, :, 0]) <= 3e-7 * np.abs(lum[:, :, 0]) + 1e-9 * peak).all()
    ol = oracle.lens_image_batch(l2, L["grid"], L["psf"], data, ivar, want_images=False, kinds=kinds)
    od = oracle.jam_vrms_batch(D["params"], lum, mass, D["beta"], kin)
    ref = oracle.joint_loglike(ol["chi2"], od["chi2"])
    ll = out["loglike"].cpu().numpy().astype(np.float64)
    assert np.isfinite(ref).all() and (out["flags"].cpu().numpy() == 0).all()
    assert np.max(np.abs(ll - ref) / np.abs(ref)) < 1e-5, (ll, ref)
    g.close()
