"""GPU parity of the eNFW halo (mass part; glad_set_enfw) against the oracle through the C ABI: the
ray-shot image and chi2 with EPL + shear + point mass + halo (1e-4 per pixel, 1e-5 on chi2), the quasar terms with the halo in
alpha, the Hessian and psi, the MGE profile kind GLAD_PROFILE_NFW_CSE, the halo rows of the self-consistent joint entry, and the
flags of invalid halos."""
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


@pytest.fixture(scope="module")
def table(oracle):
    A, s = workloads.cse_table()
    oracle.set_cse_table(A, s)
    return A, s


def oracle_dm(oracle):
    def dm(w):
        img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0] if w["lens"] else None
        vr = None
        if w["dyn"]:
            d = w["dyn"]
            vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
        return img, vr
    return dm


def test_images_and_chi2_with_a_halo(glad_mod, oracle, table):
    A, s = table
    wl = workloads.make_workload("C2", oracle_dm(oracle), B=24)
    L = wl["lens"]
    nf = workloads.enfw_params(24)
    nf[3, 0] = 0.0                                                     # one vector without halo
    nf[5, 2] = 1.0                                                     # a round halo
    bad = nf.copy(); bad[7, 1] = 0.0; bad[9, 2] = 1.2
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_enfw(bad, A, s)
    out = g.lens_image_batch(L["params"])
    ref = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], enfw=bad)
    fl = out["flags"].cpu().numpy()
    assert (fl == ref["flags"]).all() and fl[7] == 1 and fl[9] == 1 and fl.sum() == 2
    img = out["images"].cpu().numpy().astype(np.float64)
    worst = 0.0
    for b in np.flatnonzero(fl == 0):
        mx = np.abs(ref["images"][b]).max()
        err = np.abs(img[b] - ref["images"][b]) / np.maximum(np.abs(ref["images"][b]), 1e-6 * mx)
        worst = max(worst, err.max())
    assert worst < 1e-4, worst
    ok = fl == 0
    np.testing.assert_allclose(out["chi2"].cpu().numpy()[ok], ref["chi2"][ok], rtol=1e-5)
    assert np.isnan(img[7]).all() and np.isinf(out["chi2"].cpu().numpy()[7])
    # the halo changes the image; switching it off restores the plain path bitwise
    g.set_enfw(None)
    plain = g.lens_image_batch(L["params"])["images"].cpu().numpy()
    g2 = glad_mod.Glad(0)
    g2.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    assert np.array_equal(plain, g2.lens_image_batch(L["params"])["images"].cpu().numpy())
    assert np.abs(plain[0] - img[0]).max() > 1e-3 * plain[0].max()
    print(f"eNFW images: worst relative pixel error {worst:.2e}")
    g.close(); g2.close()


def test_quasar_terms_with_a_halo(glad_mod, oracle, table):
    A, s = table
    wl = workloads.make_workload("C2", B=64)
    L = wl["lens"]
    nf = workloads.enfw_params(64)
    nf[:, 0] *= 0.2                                                    # a perturbing halo: the quad of the truth model stays a quad
    q = workloads.quasar_data("C2")
    g = glad_mod.Glad(0)
    g.set_quasar_data(q)
    g.set_enfw(nf, A, s)
    out = g.quasar_chi2_batch(L["params"], wl["ddt"], want_details=True)
    ref = oracle.quasar_batch(L["params"], wl["ddt"], q, enfw=nf)
    conv = np.all(ref["last_step"] < 1e-10, axis=1)
    assert conv.sum() >= 8
    for k in ("chi2_img", "chi2_tmd"):
        a, b = out[k].cpu().numpy()[conv], ref[k][conv]
        assert np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-30)) < 1e-5, k
    np.testing.assert_allclose(out["beta"].cpu().numpy()[conv], ref["beta"][conv], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(out["theta_pre"].cpu().numpy()[conv], ref["theta_pre"][conv], rtol=1e-8, atol=1e-10)
    g.close()


def test_mge_kind_and_halo_rows_of_the_joint_model(glad_mod, oracle, table):
    A, s = table
    wl = workloads.make_workload("C2", oracle_dm(oracle), B=8)         # C2: the lens light that the luminous tracer is made from
    L, D, B = wl["lens"], wl["dyn"], wl["B"]
    nf = workloads.enfw_params(B)
    g = glad_mod.Glad(0)
    with pytest.raises(glad_mod.GladError):                           # kind 3 needs the table
        g.mge1d_batch(glad_mod.PROFILE_NFW_CSE, np.ones((2, 4), np.float32), 10, 0.05, 100.0)
    g.set_enfw(nf, A, s, n_gauss=14, sigma_range=(0.05, 300.0))
    prof = np.stack([nf[:, 0] * 3000.0, nf[:, 1], np.zeros(B), nf[:, 2]], 1).astype(np.float32)
    rows = g.mge1d_batch(glad_mod.PROFILE_NFW_CSE, prof, 18, 0.04, 250.0).cpu().numpy().astype(np.float64)
    want = oracle.mge1d_batch(3, prof, 18, 0.04, 250.0)
    np.testing.assert_allclose(rows[:, :, 1:], want[:, :, 1:], rtol=1e-6)
    assert np.max(np.abs(rows[:, :, 0] - want[:, :, 0])) < 2e-7 * np.abs(want[:, :, 0]).max()      # fp32 rows of an fp64 sum
    # joint model entry: tables and lnL with the halo in both halves
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    out = g.joint_loglike_model_batch(L["params"], D["params"], wl["ddt"], wl["z_d"], 10, (0.05, 8.0), 10, (0.02, 50.0), D["beta"],
                                      want_tables=True)
    lens2, lum, mass = oracle.model_tables(L["params"], D["params"], wl["ddt"], wl["z_d"], 10, 10, (0.05, 8.0), (0.02, 50.0), enfw=nf,
                                           halo=dict(n=14, sigma_lo=0.05, sigma_hi=300.0))
    gm = out["mass_mge"].cpu().numpy().astype(np.float64)
    assert gm.shape == mass.shape == (B, 24, 3)
    peak = np.abs(mass[:, :, 0]).max(axis=1, keepdims=True)
    assert np.max(np.abs(gm[:, :, 0] - mass[:, :, 0]) / peak) < 1e-6
    ol = oracle.lens_image_batch(lens2, L["grid"], L["psf"], L["data"], L["ivar"], want_images=False, enfw=nf)
    od = oracle.jam_vrms_batch(D["params"], lum, mass, D["beta"], D["kin"])
    ref = oracle.joint_loglike(ol["chi2"], od["chi2"])
    ll = out["loglike"].cpu().numpy()
    assert np.isfinite(ref).all() and np.max(np.abs(ll - ref) / np.abs(ref)) < 1e-5, (ll, ref)
    with pytest.raises(glad_mod.GladError):                           # the pixelated-source entry does not take the halo
        pin = workloads.pixsrc_inputs(wl, 8, 8)
        g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 8, 8)
    g.close()
