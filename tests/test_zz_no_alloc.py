"""glad_lens_image_noalloc (the entry point that allocates nothing: its scratch is a file-scope device array) against
glad_lens_image_batch, the existing path, through the C ABI: images, chi2 and flags must be IDENTICAL (same kernels, same inputs;
the tests of the existing path hold it to 1e-4 per pixel against the oracle), on two calls in a row with different batches -- the
second call finds the first call's constants in the shared array -- and with the mass sheet and an eNFW halo set.  A batch beyond
GLAD_LENS_NOALLOC_MAX_B is rejected with GLAD_ESHAPE.  Collected last (pytest -x): named test_zz_*."""
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


_driver_warm = False      # the process's first launch of a kernel may make the DRIVER load its code / size local memory


def run_both(glad_mod, g, params_np):
    import torch
    global _driver_warm
    p = torch.as_tensor(params_np, dtype=torch.float32).cuda()
    B = p.shape[0]
    ny, nx = g.image_shape
    out = dict(images=torch.full((B, ny, nx), -7.0, dtype=torch.float32, device="cuda"),
               chi2=torch.full((B,), -7.0, dtype=torch.float32, device="cuda"),
               flags=torch.full((B,), -7, dtype=torch.int32, device="cuda"))
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    g.lens_image_noalloc(p, out)
    # neither torch's allocator nor the library (cudaMalloc shows in the device's free memory) allocated anything
    assert torch.cuda.memory_allocated() == before
    assert torch.cuda.mem_get_info()[0] == free_before or not _driver_warm
    _driver_warm = True
    torch.cuda.synchronize()
    ref = g.lens_image_batch(p)
    torch.cuda.synchronize()
    for k in ("images", "chi2", "flags"):
        a, b = out[k].cpu().numpy(), ref[k].cpu().numpy()
        assert np.array_equal(a, b, equal_nan=True), k
    return out


def test_two_calls_in_a_row_match_the_existing_path(glad_mod):
    wl = workloads.make_workload("C2", B=40)
    L = wl["lens"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    prm = L["params"].copy()
    prm[3, 4] = 1.5                                                      # an invalid vector (q > 1): flagged, NaN image, on both paths
    first = run_both(glad_mod, g, prm)
    fl = first["flags"].cpu().numpy()
    assert fl[3] != 0 and (np.delete(fl, 3) == 0).all()
    img = first["images"].cpu().numpy()
    assert np.isfinite(np.delete(img, 3, axis=0)).all() and np.abs(img[0]).max() > 0
    # second call: fewer vectors, other parameters; the array still holds the first call's constants beyond row 13
    prm2 = prm[::-1][:13].copy()
    prm2[:, 2] *= 1.01
    second = run_both(glad_mod, g, prm2)
    assert not np.array_equal(second["images"].cpu().numpy()[0], img[0])
    # a second context on the same device shares the array and its address
    g2 = glad_mod.Glad(0)
    g2.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    run_both(glad_mod, g2, prm)
    g.close(); g2.close()


def test_with_mass_sheet_and_halo_and_the_size_limit(glad_mod):
    import torch
    wl = workloads.make_workload("C1", B=8)
    L = wl["lens"]
    g = glad_mod.Glad(0)
    g.set_image_data(L["grid"], L["psf"], L["data"], L["ivar"])
    g.set_mass_sheet(np.linspace(0.8, 1.1, 8).astype(np.float32))
    A, s = workloads.cse_table()
    g.set_enfw(workloads.enfw_params(8), A, s)
    run_both(glad_mod, g, L["params"])
    run_both(glad_mod, g, L["params"][:5])
    g.set_mass_sheet(None)
    g.set_enfw(None)
    run_both(glad_mod, g, L["params"])
    nb = glad_mod.LENS_NOALLOC_MAX_B + 1
    big = torch.zeros((nb, glad_mod.NLENS), dtype=torch.float32, device="cuda")
    with pytest.raises(glad_mod.GladError, match="GLAD_LENS_NOALLOC_MAX_B"):
        g.lens_image_noalloc(big, dict(images=None, chi2=None, flags=None))
    g.close()
