"""GPU parity for SURVEY.md 8(f) rank 1: the on-device 1-D MGE (Eq. 44-46) and the self-consistent joint model
(glad_joint_loglike_model_batch) against the fp64 oracle on the same seeded inputs.

Tolerances: the MGE rows are fp64 arithmetic rounded to fp32 on the device and fp64 in the oracle: 3e-7
relative (fp32 rounding) plus max(1e-9, 1e-13 x 10^(P/3)) of the table's largest amplitude absolute (1e-9 up to the
default P = 12; the 1-2 ulp of the device's exp/log/sincos on arguments of size ~50 set the floor) -- the Euler sum of Eq. 45 cancels 10^(P/3)-fold, so each side carries rounding noise of ~25 terms x 1e4 x 2e-16 of the profile's scale, which
is all there is in the amplitudes far below the peak.  The joint log-likelihood keeps BASELINE.json's 1e-5."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

LUM_RANGE, MASS_RANGE = (0.02, 10.0), (0.02, 50.0)


@pytest.fixture(scope="module")
def glad_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2504_01302_b200 as m
    return m


def check_rows(got, ref, what="", P=12):
    got = np.asarray(got, np.float64)
    assert got.shape == ref.shape
    # sigma_n, q': the fp32 rounding of the oracle's values (one ulp of slack for exp())
    assert np.allclose(got[:, :, 1:], ref[:, :, 1:], rtol=1.2e-7, atol=0)
    peak = np.abs(ref[:, :, 0]).max(axis=1, keepdims=True)
    # rounding noise of the Euler sum: ~25 terms x 10^(P/3) x fp64 epsilon of the profile's scale (1e-9 at P = 12)
    excess = np.abs(got[:, :, 0] - ref[:, :, 0]) - (3e-7 * np.abs(ref[:, :, 0]) + max(1e-9, 1e-13 * 10.0 ** (P / 3.0)) * peak)
    i = np.unravel_index(np.argmax(excess), excess.shape)
    assert excess.max() <= 0, (what, i, got[i][0], ref[i][0], float(peak[i[0], 0]))


def _profiles(rng, B):
    ser = np.stack([rng.uniform(0.01, 3.0, B), rng.uniform(0.1, 2.5, B), rng.uniform(0.5, 6.0, B), rng.uniform(0.3, 1.0, B)], 1)
    epl = np.stack([rng.uniform(1e3, 6e3, B), rng.uniform(0.5, 2.0, B), rng.uniform(1.5, 2.6, B), rng.uniform(0.3, 1.0, B)], 1)
    wc = rng.uniform(0.02, 0.3, B)
    cham = np.stack([rng.uniform(0.01, 3.0, B), wc, wc * rng.uniform(1.5, 20.0, B), rng.uniform(0.3, 1.0, B)], 1)
    return ser.astype(np.float32), epl.astype(np.float32), cham.astype(np.float32)


@pytest.mark.parametrize("n_gauss,lo,hi,P", [(21, 0.02, 50.0, 0), (2, 0.1, 1.0, 12), (64, 0.005, 200.0, 8), (37, 0.02, 10.0, 15)])
def test_mge1d_rows_match_oracle(glad_mod, oracle, n_gauss, lo, hi, P):
    rng = np.random.default_rng(11)
    B = 67                                        # not a multiple of anything the kernel uses
    ser, epl, cham = _profiles(rng, B)
    g = glad_mod.Glad(0)
    for kind, prof in ((glad_mod.PROFILE_SERSIC, ser), (glad_mod.PROFILE_EPL, epl), (glad_mod.PROFILE_CHAMELEON, cham)):
        got = g.mge1d_batch(kind, prof, n_gauss, lo, hi, P).cpu().numpy().astype(np.float64)
        ref = oracle.mge1d_batch(kind, prof, n_gauss, lo, hi, P if P else oracle.MGE_EULER_P)
        check_rows(got, ref, kind, P if P else oracle.MGE_EULER_P)
    g.close()


def test_mge1d_argument_errors(glad_mod):
    g = glad_mod.Glad(0)
    prof = np.ones((3, 4), np.float32)
    for bad in (dict(kind=3), dict(n=1), dict(lo=0.0), dict(lo=2.0, hi=1.0), dict(P=16), dict(n=65)):
        a = dict(kind=0, n=10, lo=0.02, hi=10.0, P=0)
        a.update(bad)
        with pytest.raises(glad_mod.GladError):
            g.mge1d_batch(a["kind"], prof, a["n"], a["lo"], a["hi"], a["P"])
    assert g.mge1d_batch(0, np.zeros((0, 4), np.float32), 10, 0.02, 10.0).shape == (0, 10, 3)
    g.close()


@pytest.mark.parametrize("name,B,n_lum,n_mass", [("C1", 8, 10, 10), ("C2", 12, 20, 20)])
def test_joint_model_matches_oracle(glad_mod, oracle, name, B, n_lum, n_mass):
    """One vector -> (luminous MGE of the lens light, mass MGE of Sigma_crit kappa_epl, theta_E,BH) -> both halves."""
    def dm(w):
        img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0]
        d = w["dyn"]
        vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
        return img, vr
    wl = workloads.make_workload(name, dm, B=B)
    L, D = wl["lens"], wl["dyn"]
    lens = L["params"].copy()
    if name == "C1":                              # C1 has no lens light: give the tracer a Sersic (I_e tiny: image unchanged)
        lens[:, 16:21] = np.array([1e-9, 0.8, 3.0, 0.8, 0.0], np.float32)
        lens[:, 19] = lens[:, 4]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    out = g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, LUM_RANGE, n_mass, MASS_RANGE,
                                      D["beta"], want_tables=True)
    l2, lum, mass = oracle.model_tables(lens, D["params"], wl["ddt"], wl["z_d"], n_lum, n_mass, LUM_RANGE, MASS_RANGE)
    check_rows(out["lum_mge"].cpu().numpy(), lum.astype(np.float64), "lum")
    check_rows(out["mass_mge"].cpu().numpy(), mass.astype(np.float64), "mass")
    ol = oracle.lens_image_batch(l2, L["grid"], L["psf"], L["data"], L["ivar"], want_images=False)
    od = oracle.jam_vrms_batch(D["params"], lum, mass, D["beta"], D["kin"])
    ref = oracle.joint_loglike(ol["chi2"], od["chi2"])
    ll = out["loglike"].cpu().numpy().astype(np.float64)
    assert (out["flags"].cpu().numpy() == 0).all() and np.isfinite(ref).all()
    assert np.max(np.abs(ll - ref) / np.abs(ref)) < 1e-5, (ll, ref)
    c2l = out["chi2_lens"].cpu().numpy().astype(np.float64)
    assert np.max(np.abs(c2l - ol["chi2"]) / ol["chi2"]) < 1e-5
    # the model entry is the plain joint entry fed with the derived tables (bitwise: same kernels, same inputs)
    o2 = g.joint_loglike_batch(l2, D["params"], out["lum_mge"], out["mass_mge"], D["beta"])
    assert np.array_equal(o2["chi2_dyn"].cpu().numpy(), out["chi2_dyn"].cpu().numpy())
    g.close()


def test_joint_model_argument_errors_and_invalid_vectors(glad_mod, oracle):
    wl = workloads.make_workload("C1", None)
    L, D = wl["lens"], wl["dyn"]
    lens = L["params"].copy()
    lens[:, 16:21] = np.array([1e-9, 0.8, 3.0, 0.8, 0.0], np.float32)
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    ok = dict(n_lum=10, lum=LUM_RANGE, n_mass=10, mass=MASS_RANGE, zd=wl["z_d"])
    for bad in (dict(n_lum=1), dict(n_mass=65), dict(lum=(0.0, 1.0)), dict(mass=(5.0, 1.0)), dict(zd=-1.0)):
        a = dict(ok); a.update(bad)
        with pytest.raises(glad_mod.GladError):
            g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], a["zd"], a["n_lum"], a["lum"], a["n_mass"], a["mass"], D["beta"])
    with pytest.raises(glad_mod.GladError):
        g.joint_loglike_model_batch(lens, D["params"], wl["ddt"][:3], wl["z_d"], 10, LUM_RANGE, 10, MASS_RANGE, D["beta"])
    # a physically invalid vector (gamma outside (1,3)) is flagged, lnL = -inf, the rest of the batch is untouched
    good = g.joint_loglike_model_batch(lens, D["params"], wl["ddt"], wl["z_d"], 10, LUM_RANGE, 10, MASS_RANGE, D["beta"])
    ll_good = good["loglike"].cpu().numpy().copy()
    lens_bad = lens.copy(); lens_bad[2, 3] = 3.5
    out = g.joint_loglike_model_batch(lens_bad, D["params"], wl["ddt"], wl["z_d"], 10, LUM_RANGE, 10, MASS_RANGE, D["beta"])
    ll = out["loglike"].cpu().numpy()
    assert np.isneginf(ll[2]) and out["flags"].cpu().numpy()[2] != 0
    keep = np.arange(8) != 2
    assert np.array_equal(ll[keep], ll_good[keep]) and (out["flags"].cpu().numpy()[keep] == 0).all()
    g.close()
