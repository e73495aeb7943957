#!/usr/bin/env python
"""Writes tests/golden/*.txt from the fp64 oracle ONLY (never from the CUDA path).

The paper prints no model image, v_rms map or likelihood value for any parameter vector, so
these are not the paper's numbers: they freeze the oracle's own results on the seeded C1 workload so that a later
change to the oracle's arithmetic cannot pass unnoticed (tests/test_golden.py), and they give the GPU tests a
second, stored copy of the expected values.  Re-run only together with a commit message that names the passage or
DESIGN.md reading that justifies the change:
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
import workloads  # noqa: E402


def data_model(w):
    img = oracle.lens_image_batch(w["lens"]["params"], w["lens"]["grid"], w["lens"]["psf"])["images"][0]
    d = w["dyn"]
    vr = oracle.jam_vrms_batch(d["params"], d["lum_mge"], d["mass_mge"], d["beta"], d["kin"])["vrms"][0]
    return img, vr


def c1_values():
    wl = workloads.make_workload("C1", data_model)
    L, D = wl["lens"], wl["dyn"]
    ol = oracle.lens_image_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"])
    od = oracle.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], D["kin"])
    ll = oracle.joint_loglike(ol["chi2"], od["chi2"])
    return {"c1_chi2_lens": ol["chi2"], "c1_chi2_dyn": od["chi2"], "c1_loglike": ll, "c1_vrms": od["vrms"],
            "c1_image_row20_vec0": ol["images"][0, 20, :]}


def mge_values():
    return {"mge_sersic_n4_re1.85_q0.8_21g_0.02_50": oracle.mge1d(oracle.PROFILE_SERSIC, [1.0, 1.85, 4.0, 0.8], 21, 0.02, 50.0)[:, 0],
            "mge_epl_sc1_te1.65_g2_q0.8_21g_0.02_50": oracle.mge1d(oracle.PROFILE_EPL, [1.0, 1.65, 2.0, 0.8], 21, 0.02, 50.0)[:, 0]}


def pixsrc_values():
    """Pixelated-source evidence (Eq. 37-43) of the 8 C1 vectors on 16 x 12 source grids (workloads.pixsrc_inputs)."""
    from oracle import pixsrc
    wl = workloads.make_workload("C1", data_model)
    L = wl["lens"]
    pin = workloads.pixsrc_inputs(wl, 16, 12)
    r = pixsrc.pixsrc_batch(L["params"], L["grid"], L["psf"], L["data"], L["ivar"], pin["src_grids"], pin["lam"], 16, 12)
    return {"c1_pixsrc_logev_16x12": r["logev"], "c1_pixsrc_chi2_16x12": r["chi2"], "c1_pixsrc_smp_vec0_16x12": r["s_mp"][0].reshape(-1)}


def main():
    oracle.build()
    vals = {}
    vals.update(c1_values())
    vals.update(mge_values())
    vals.update(pixsrc_values())
    for name, v in vals.items():
        np.savetxt(os.path.join(HERE, name + ".txt"), np.atleast_1d(v), fmt="%.17e",
                   header=f"{name}: written by tests/golden/make_golden.py from oracle/ only (fp64); not a published value")


if __name__ == "__main__":
    main()
