"""CPU-only checks of the boundary: libglad.so loads, exports every symbol glad.h declares, the host
helper agrees with the paper's definition, and the binding refuses to run without a GPU."""
import ctypes
import math
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "glad.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(glad_[a-z0-9_]+)\s*\(", txt)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2504_01302_b200 import EXPORTS, build
    lib = ctypes.CDLL(build())
    decl = declared_symbols()
    assert len(decl) >= 12
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in glad.h but not exported"
    assert sorted(EXPORTS) == decl, "binding and header disagree on the entry points"


def test_bh_theta2_host_helper():
    from paper_2504_01302_b200 import bh_theta2
    # theta_E^2 = 4 G M (1+z_d) / (c^2 D_dt)  (Eq. 4); 2 G Msun / c^2 = 2953.25 m
    pc_m = 3.0856775814913673e16
    expected = 2 * 2953.25 * 5e9 * 1.295 / (1823e6 * pc_m) * (648000 / math.pi) ** 2
    assert bh_theta2(5e9, 1823.0, 0.295) == pytest.approx(expected, rel=2e-4)
    assert bh_theta2(0.0, 1823.0, 0.295) == 0.0


def test_no_cpu_fallback():
    import torch
    from paper_2504_01302_b200 import Glad, GladError
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(GladError):
        Glad(0)


def test_product_does_not_import_oracle_or_work_dir():
    pkg = os.path.join(ROOT, "paper_2504_01302_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower() or f == "__init__.py" and False, f"{f} mentions the oracle"
                assert "_work" not in src


def test_binding_constants_match_header():
    """The binding sizes its profile arrays from its own KERNELS tuple and mirrors the flag / size constants: they must equal glad.h's."""
    import paper_2504_01302_b200 as m
    from paper_2504_01302_b200.binding import Glad
    txt = open(os.path.join(ROOT, "include", "glad.h")).read()
    dv = {k: int(v) for k, v in re.findall(r"#define\s+(GLAD_[A-Z0-9_]+)\s+(-?\d+)\b", txt)}
    assert dv["GLAD_NKERNELS"] == len(Glad.KERNELS)
    assert dv["GLAD_NLENS"] == m.NLENS and dv["GLAD_NDYN"] == m.NDYN
    assert (dv["GLAD_FLAG_LENS_INVALID"], dv["GLAD_FLAG_DYN_INVALID"], dv["GLAD_FLAG_BIN_INVALID"], dv["GLAD_FLAG_PIXSRC_NOT_PD"]) == \
        (m.FLAG_LENS_INVALID, m.FLAG_DYN_INVALID, m.FLAG_BIN_INVALID, m.FLAG_PIXSRC_NOT_PD)
