"""CPU-only checks of the seeded generator (shapes, determinism, symmetry, deprojectability)."""
import numpy as np

import workloads


def test_deterministic_and_shapes():
    a = workloads.make_workload("C2", B=8)
    b = workloads.make_workload("C2", B=8)
    for half in ("lens", "dyn"):
        for k, v in a[half].items():
            if isinstance(v, np.ndarray):
                assert np.array_equal(v, b[half][k]), k
    assert a["lens"]["params"].shape == (8, 26) and a["lens"]["params"].dtype == np.float32
    assert a["lens"]["psf"].shape == (21, 21) and abs(a["lens"]["psf"].sum() - 1) < 1e-5
    d = a["dyn"]
    assert d["lum_mge"].shape == (20, 3) and d["mass_mge"].shape == (8, 20, 3) and d["beta"].shape == (8,)
    k = d["kin"]
    assert k["xs"].shape == (80,) and k["bin_id"].shape == (80, 80) and k["kernel"].shape == (15, 15)
    assert np.array_equal(k["xs"], -k["xs"][::-1])                    # exactly mirror-symmetric grid
    assert set(np.unique(k["bin_id"])) == set(range(60))
    assert abs(k["kernel"].sum() - 1) < 1e-5 and abs(float(k["u_weights"].sum()) - 1.0) < 1e-5


def test_every_draw_is_deprojectable_and_truth_is_element_zero():
    w = workloads.make_workload("C5", B=6)
    d = w["dyn"]
    cos2 = np.cos(d["params"][:, 0]) ** 2
    assert (d["lum_mge"][..., 2].min(axis=-1) ** 2 > cos2).all()       # Eq. 22
    assert (d["mass_mge"][..., 2].min(axis=-1) ** 2 > cos2).all()
    assert abs(w["lens"]["params"][0, 2] - 1.65) < 1e-6 and abs(d["params"][0, 1] - 775.0) < 1e-3
    assert d["lum_mge"].shape == (6, 30, 3) and d["beta"].shape == (6, 30)


def test_sweep_cells_and_subset():
    assert sum(1 for k in workloads.CONFIGS if k.startswith("C3-")) == 18
    w = workloads.make_workload("C3-10-40-256", B=5)
    assert w["lens"] is None and w["dyn"]["kin"]["nbins"] == 100
    s = workloads.subset(w, [0, 3])
    assert s["B"] == 2 and np.array_equal(s["dyn"]["params"][1], w["dyn"]["params"][3])
    assert s["dyn"]["mass_mge"].shape[0] == 2


def test_pixsrc_inputs():
    w = workloads.make_workload("C2", B=5)
    a, b = workloads.pixsrc_inputs(w, 32, 24), workloads.pixsrc_inputs(w, 32, 24)
    assert a["src_grids"].shape == (5, 3) and a["src_grids"].dtype == np.float32 and a["lam"].shape == (5,)
    assert np.array_equal(a["src_grids"], b["src_grids"]) and np.array_equal(a["lam"], b["lam"])
    assert (a["lam"] > 0).all() and (a["src_grids"][:, 2] > 0).all()
    # the grid is centred on the vector's source position
    cx = a["src_grids"][:, 0] + 15.5 * a["src_grids"][:, 2]
    assert np.allclose(cx, w["lens"]["params"][:, 9], atol=1e-5)
