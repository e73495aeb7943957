"""GPU parity of row a6 on the kernel instantiations and size limits the config tests do not reach:
jam_quad_tc_kernel<2,32,16> (folded maps wider than 96 columns) at the GLAD_MAX_SKY = 256 boundary in two-MMA mode with
ragged 8-blocks, three bf16 terms per operand (glad_set_jam_options(.., 3, ..)) in one-MMA and multi-MMA mode, the FP32 SIMT
kernel at the sizes production routes to it (more than 128 folded rows), explicit K-slices / flush lengths, and the shared-
memory limit of the binning kernel reported as GLAD_ESHAPE when the static data is set."""
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


def dyn_case(seed, xs, ys, n_lum=5, n_mass=7, nbins=12, B=3, kk=5, nu=40, mbh=3e9):
    rng = np.random.default_rng(seed)
    nx, ny = len(xs), len(ys)
    lum = np.stack([rng.uniform(200, 2000, n_lum), np.geomspace(0.05, 3.0, n_lum), rng.uniform(0.7, 0.95, n_lum)], 1)
    mass = np.stack([rng.uniform(500, 5000, (B, n_mass)), np.broadcast_to(np.geomspace(0.04, 20.0, n_mass), (B, n_mass)),
                     rng.uniform(0.7, 1.0, (B, n_mass))], 2)
    dyn = np.stack([np.radians(rng.uniform(65, 88, B)), rng.uniform(600, 1000, B), np.full(B, mbh), rng.uniform(0.8, 1.2, B)], 1)
    beta = rng.uniform(-0.3, 0.5, (B, n_lum))
    un, uw = workloads.gauss_legendre_u(nu)
    kern = rng.uniform(0.1, 1.0, (kk, kk)); kern /= kern.sum()
    bins = rng.integers(-1, nbins, (ny, nx)).astype(np.int32)
    bins.flat[:nbins] = np.arange(nbins)
    kin = dict(xs=np.asarray(xs, np.float32), ys=np.asarray(ys, np.float32), bin_id=bins, nbins=nbins, kernel=kern.astype(np.float32),
               vrms_obs=rng.uniform(200, 300, nbins).astype(np.float32), vrms_ivar=rng.uniform(0.01, 0.05, nbins).astype(np.float32),
               u_nodes=un, u_weights=uw)
    return dyn.astype(np.float32), lum.astype(np.float32), mass.astype(np.float32), beta.astype(np.float32), kin


def centred(n, step):
    return (np.arange(n) - (n - 1) / 2) * step


def compare(glad_mod, oracle, case, **opts):
    dyn, lum, mass, beta, kin = case
    g = glad_mod.Glad(0)
    if opts:
        g.set_jam_options(**opts)
    g.set_kin_data(kin)
    out = g.jam_vrms_batch(dyn, lum, mass, beta, want_map=True)
    ref = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin, want_maps=True)
    v2 = out["v2map"].cpu().numpy()
    np.testing.assert_allclose(v2, ref["v2map"], rtol=1e-4)
    np.testing.assert_allclose(out["vrms"].cpu().numpy(), ref["vrms"], rtol=1e-4)
    assert (out["flags"].cpu().numpy() == ref["flags"]).all()
    g.close()
    return float(np.max(np.abs(v2 - ref["v2map"]) / np.abs(ref["v2map"])))


def test_widest_tcgen05_map_256x200(glad_mod, oracle):
    """256 x 200 mirror-symmetric sky grid = GLAD_MAX_SKY columns: folded 128 x 100 -> ny8 = 104 (ragged last 8-block, two-MMA
    mode), nxp = 128, N = 256 accumulator columns, 32 accumulator registers per thread: jam_quad_tc_kernel<2,32,16>."""
    case = dyn_case(11, centred(256, 0.008), centred(200, 0.011), nu=24)
    err = compare(glad_mod, oracle, case)
    assert err < 1e-4


def test_three_bf16_terms_one_mma_and_multi_mma(glad_mod, oracle):
    """NT = 3 (24 mantissa bits per operand): 33 x 18 grid (folded 17 x 9: the three row blocks fit one M = 128 tile) and
    120 x 100 (folded 60 x 50: 3 x 56 rows > 128, three MMAs per K-step, N = 192).  The 3-term result must also be at least
    as close to the oracle as the 2-term one up to the accumulator's own rounding."""
    small = dyn_case(12, centred(33, 0.07), centred(18, 0.09))
    e3 = compare(glad_mod, oracle, small, terms=3)
    e2 = compare(glad_mod, oracle, small, terms=2)
    assert e3 < 5e-6 and e3 <= e2 + 2e-6, (e3, e2)
    big = dyn_case(13, centred(120, 0.017), centred(100, 0.02), nu=32)
    assert compare(glad_mod, oracle, big, terms=3) < 1e-5


def test_simt_kernel_at_the_sizes_production_routes_to_it(glad_mod, oracle):
    """With GLAD_MAX_SKY = 256 a mirror-symmetric grid never has more than 128 folded rows, so the sizes that reach the SIMT
    kernel without being asked for are the asymmetric (unfoldable) ones: 40 x 150 irregular coordinates -> 150 rows > 128 -> the
    tcgen05 plan declines and jam_quad_kernel (FP32 SIMT) runs by default (no option set)."""
    rng = np.random.default_rng(14)
    xs = np.sort(rng.uniform(-0.9, 1.1, 40))
    ys = np.sort(rng.uniform(-0.8, 1.4, 150))
    case = dyn_case(14, xs, ys, nu=32)
    assert compare(glad_mod, oracle, case) < 1e-4
    # asymmetric in x only, 130 folded columns: N = 2 * 136 > 256 also declines
    case = dyn_case(15, np.sort(rng.uniform(-1.0, 1.2, 130)), centred(24, 0.08), nu=32)
    assert compare(glad_mod, oracle, case) < 1e-4


def test_explicit_slices_and_flush_lengths(glad_mod, oracle):
    """K-slices and the accumulator group length are context options now (they were environment knobs): every setting gives
    the oracle's map; one chunk per group (flush = 1) is the most accurate."""
    case = dyn_case(16, centred(48, 0.04), centred(40, 0.05), B=2, nu=64)
    errs = {(s, f): compare(glad_mod, oracle, case, slices=s, flush=f) for s in (1, 3) for f in (0, 1, 8)}
    assert max(errs.values()) < 2e-5, errs


def test_binning_kernel_shared_memory_limit_is_an_eshape_at_setup(glad_mod):
    """176 x 176 asymmetric grid: 484 thread tiles pass the tile limit, but jam_post_kernel would need 2*176*176*4 = 248 KB of
    shared memory: glad_set_kin_data says so (it used to surface as an opaque CUDA error inside the first batch call)."""
    rng = np.random.default_rng(17)
    case = dyn_case(17, np.sort(rng.uniform(-1, 1.2, 176)), np.sort(rng.uniform(-1, 1.2, 176)), B=1, nu=8)
    g = glad_mod.Glad(0)
    with pytest.raises(glad_mod.GladError, match="shared memory"):
        g.set_kin_data(case[4])
    g.close()


def test_lens_image_shared_memory_limit_is_an_eshape_at_setup(glad_mod):
    """A 1 x 40000 image passes GLAD_MAX_IMAGE_PIXELS, but with the halo of a 31 x 31 PSF it has 40001 padded rows of 55 floats
    = 8.8 MB of shared memory: GLAD_ESHAPE from glad_set_image_data, not a CUDA error at the first launch."""
    g = glad_mod.Glad(0)
    grid = dict(nx=1, ny=40000, supersample=1, pix=0.05, x0=0.0, y0=-1000.0)
    psf = np.full((31, 31), 1.0 / 961, np.float32)
    with pytest.raises(glad_mod.GladError, match="shared memory"):
        g.set_image_data(grid, psf, None, None)
    g.close()


def test_two_contexts_on_two_devices_in_one_process(glad_mod, oracle):
    """The opt-in to > 48 KB of dynamic shared memory is per function AND per device: a second context on another GPU must
    launch the large-shared-memory kernels too, and a call must leave the caller's current device alone."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    case = dyn_case(18, centred(48, 0.04), centred(40, 0.05), B=2, nu=32)
    dyn, lum, mass, beta, kin = case
    ref = oracle.jam_vrms_batch(dyn, lum, mass, beta, kin)
    torch.cuda.set_device(0)
    for dev in (0, 1):
        g = glad_mod.Glad(dev)
        g.set_kin_data(kin)
        out = g.jam_vrms_batch(dyn, lum, mass, beta)
        assert torch.cuda.current_device() == 0
        np.testing.assert_allclose(out["vrms"].cpu().numpy(), ref["vrms"], rtol=1e-4)
        g.close()
