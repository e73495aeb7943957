"""Out-of-bounds writes: compute-sanitizer is closed on the GPU pool (profiles/r2_sanitizer.md), so every output buffer the binding
hands to the C ABI is allocated here inside a larger sentinel-filled block and the guard bands on both sides must come back
untouched, on ragged shapes (odd batch, image and sky sizes that are not multiples of any tile, a source grid that is not a multiple
of the 64-wide Cholesky panel, the last chunk of a chunked pixelated-source call).  Results must also equal, bit for bit, those of
the ordinary allocation: a kernel that reads beyond its inputs or depends on what lies next to its outputs fails that."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

GUARD = 4096          # bytes on each side


@pytest.fixture(scope="module")
def glad_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2504_01302_b200 as m
    return m


class GuardedTorch:
    """Stands in for the `torch` module inside the binding: empty() returns the interior of a guarded block."""

    def __init__(self, torch):
        self._t = torch
        self.blocks = []

    def __getattr__(self, name):
        return getattr(self._t, name)

    def empty(self, shape, dtype=None, device=None, **kw):
        t = self._t
        if device is None or t.device(device).type != "cuda":
            return t.empty(shape, dtype=dtype, device=device, **kw)
        shape = (shape,) if isinstance(shape, int) else tuple(shape)
        nbytes = int(np.prod(shape, dtype=np.int64)) * t.empty((), dtype=dtype).element_size()
        pad = (-nbytes) % 16
        raw = t.full((GUARD + nbytes + pad + GUARD,), 0xA5, dtype=t.uint8, device=device)
        self.blocks.append((raw, nbytes))
        return raw[GUARD:GUARD + nbytes].view(dtype).reshape(shape)

    def check(self):
        self._t.cuda.synchronize()
        for raw, nbytes in self.blocks:
            lo, hi = raw[:GUARD], raw[GUARD + nbytes:]
            assert bool((lo == 0xA5).all()) and bool((hi == 0xA5).all()), f"guard band of a {nbytes}-byte output was written"
        n = len(self.blocks)
        self.blocks = []
        return n


@pytest.fixture()
def guarded(glad_mod, monkeypatch):
    import torch
    from paper_2504_01302_b200 import binding
    gt = GuardedTorch(torch)
    monkeypatch.setattr(binding, "torch", gt)
    return gt


def same(a, b):
    for k in a:
        if a[k] is None:
            continue
        x, y = a[k].cpu().numpy(), b[k].cpu().numpy()
        assert np.array_equal(x, y, equal_nan=True), k


def ragged_workload(B):
    wl = workloads.make_workload("C1", B=B)
    return wl


def test_joint_lens_and_dynamics_outputs_stay_inside(glad_mod, guarded):
    wl = ragged_workload(7)
    L, D = wl["lens"], wl["dyn"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    a = g.lens_image_batch(L["params"])
    b = g.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], want_map=True)
    c = g.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"])
    g.set_jam_options("simt")
    d = g.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], want_map=True)
    g.set_jam_options("auto")
    assert guarded.check() >= 10
    import torch
    from paper_2504_01302_b200 import binding
    binding.torch = torch
    g2 = glad_mod.Glad(0)
    g2.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g2.set_kin_data(D["kin"])
    same(a, g2.lens_image_batch(L["params"]))
    same(b, g2.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], want_map=True))
    same(c, g2.joint_loglike_batch(L["params"], D["params"], D["lum_mge"], D["mass_mge"], D["beta"]))
    g2.set_jam_options("simt")
    same(d, g2.jam_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], want_map=True))
    g.close(); g2.close()


def test_model_quasar_and_mge_outputs_stay_inside(glad_mod, guarded):
    wl = workloads.make_workload("C2", B=5)
    L, D = wl["lens"], wl["dyn"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_kin_data(D["kin"])
    g.set_quasar_data(workloads.quasar_data("C2"))
    g.quasar_chi2_batch(L["params"], wl["ddt"], want_details=True)
    g.joint_loglike_model_batch(L["params"], D["params"], wl["ddt"], wl["z_d"], 9, (0.05, 8.0), 11, (0.02, 50.0), D["beta"], want_tables=True)
    g.joint_loglike_full_batch(L["params"], D["params"], wl["ddt"], wl["z_d"], 9, (0.05, 8.0), 11, (0.02, 50.0), D["beta"])
    prof = np.stack([np.full(5, 100.0), np.linspace(0.5, 2.0, 5), np.linspace(1.0, 4.0, 5), np.full(5, 0.8)], 1).astype(np.float32)
    g.mge1d_batch(0, prof, 13, 0.03, 40.0)
    A, s = workloads.cse_table()
    g.set_enfw(workloads.enfw_params(5), A, s)
    g.lens_image_batch(L["params"])
    g.quasar_chi2_batch(L["params"], wl["ddt"], want_details=True)
    assert guarded.check() >= 12
    g.close()


def test_jam_sph_outputs_stay_inside(glad_mod, guarded):
    wl = ragged_workload(5)
    D = wl["dyn"]
    g = glad_mod.Glad(0)
    g.set_kin_data(D["kin"])
    sph = workloads.jam_sph_rules(D["kin"], panels=3, nr=9, nth=5, nz=40, sigma_max=float(D["lum_mge"][..., 1].max()))
    g.set_jam_sph_rules(sph)
    g.jam_sph_vrms_batch(D["params"], D["lum_mge"], D["mass_mge"], D["beta"], want_map=True, want_moments=True)
    assert guarded.check() >= 5
    g.close()


def test_pixsrc_outputs_stay_inside_with_ragged_panels_and_chunks(glad_mod, guarded):
    wl = ragged_workload(5)
    L = wl["lens"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    for nsx, nsy in ((9, 11), (13, 10)):                             # N_s = 99 and 130: one ragged panel, two panels and a tail
        pin = workloads.pixsrc_inputs(wl, nsx, nsy)
        full = g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], nsx, nsy)
        assert guarded.check() >= 5
        # a scratch limit that forces chunks of fewer vectors than the batch
        small = g.pixsrc_evidence_batch(L["params"], pin["src_grids"], pin["lam"], nsx, nsy, scratch_mib=3)
        assert guarded.check() >= 5
        same(full, small)
        lo = g.pixsrc_lambda_opt_batch(L["params"], pin["src_grids"], (1e-4, 1e3), nsx, nsy, scratch_mib=3)
        assert guarded.check() >= 6
        assert np.isfinite(lo["lam_hat"].cpu().numpy()).all()
    g.close()
