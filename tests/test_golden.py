"""The stored oracle values under tests/golden/ (written by tests/golden/make_golden.py, oracle only) still come out
of the oracle: guards the definition of "correct" against silent drift.  The GPU half compares the CUDA path with
the same stored values."""
import os
import sys

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))


def load(name):
    return np.loadtxt(os.path.join(HERE, "golden", name + ".txt"))


def test_oracle_reproduces_golden(oracle):
    import make_golden
    vals = {}
    vals.update(make_golden.c1_values())
    vals.update(make_golden.mge_values())
    vals.update(make_golden.pixsrc_values())
    assert len(vals) == 10
    for name, v in vals.items():
        ref = load(name)
        assert np.allclose(np.ravel(v), np.ravel(ref), rtol=1e-10, atol=0), name


@pytest.mark.gpu
def test_gpu_matches_golden_c1(oracle):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import make_golden
    import workloads
    from paper_2504_01302_b200 import PROFILE_EPL, PROFILE_SERSIC, Glad
    wl = workloads.make_workload("C1", make_golden.data_model)
    L, D = wl["lens"], wl["dyn"]
    g = Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    out = g.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"])
    ll = out["loglike"].cpu().numpy().astype(np.float64)
    ref = load("c1_loglike")
    assert np.max(np.abs(ll - ref) / np.abs(ref)) < 1e-5
    vr = g.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"])["vrms"].cpu().numpy().astype(np.float64)
    refv = load("c1_vrms").reshape(vr.shape)
    assert np.max(np.abs(vr - refv) / refv) < 1e-4
    img = g.lens_image_batch(L["params"])["images"].cpu().numpy().astype(np.float64)
    row = load("c1_image_row20_vec0")
    assert np.max(np.abs(img[0, 20, :] - row) / np.maximum(np.abs(row), 1e-6 * np.abs(row).max())) < 1e-4
    for kind, prof, name in ((PROFILE_SERSIC, [1.0, 1.85, 4.0, 0.8], "mge_sersic_n4_re1.85_q0.8_21g_0.02_50"),
                             (PROFILE_EPL, [1.0, 1.65, 2.0, 0.8], "mge_epl_sc1_te1.65_g2_q0.8_21g_0.02_50")):
        a = g.mge1d_batch(kind, np.array([prof], np.float32), 21, 0.02, 50.0).cpu().numpy()[0, :, 0].astype(np.float64)
        r = load(name)
        assert np.all(np.abs(a - r) <= 3e-7 * np.abs(r) + 1e-9 * np.abs(r).max())
    pin = workloads.pixsrc_inputs(wl, 16, 12)
    po = g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], 16, 12)
    ev, c2 = load("c1_pixsrc_logev_16x12"), load("c1_pixsrc_chi2_16x12")
    assert np.max(np.abs(po["logev"].cpu().numpy() - ev) / np.abs(ev)) < 1e-5
    assert np.max(np.abs(po["chi2"].cpu().numpy() - c2) / c2) < 1e-4
    s0 = load("c1_pixsrc_smp_vec0_16x12")
    assert np.max(np.abs(po["s_mp"].cpu().numpy()[0].reshape(-1) - s0)) < 2e-3 * np.abs(s0).max()
    g.close()
