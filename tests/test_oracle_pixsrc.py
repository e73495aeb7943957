"""Pins of the pixelated-source oracle (oracle/pixsrc.py; paper Eq. 37-43) against things other than itself."""
import numpy as np
import pytest
import scipy.linalg
import scipy.signal

import oracle
from oracle import pixsrc


def _lens(thetaE=1.0, gamma=2.0, q=0.8, pa=0.5, gext=0.05, phiext=1.0, bh=0.0):
    p = np.zeros(26, np.float32)
    p[0:9] = [0.01, -0.02, thetaE, gamma, q, pa, gext, phiext, bh]
    p[9:16] = [0.05, -0.03, 0.2, 0.2, 2.0, 0.8, 0.7]
    return p


def _setup(n=14, k=5, nsx=7, nsy=6, seed=0):
    rng = np.random.default_rng(seed)
    pix = 0.2
    grid = dict(nx=n, ny=n - 2, supersample=1, pix=pix, x0=-(n - 1) / 2 * pix, y0=-(n - 3) / 2 * pix)
    psf = rng.uniform(0.1, 1.0, (k, k))
    psf /= psf.sum()                                   # asymmetric on purpose: a flipped kernel must fail
    data = rng.normal(0.0, 1.0, (grid["ny"], grid["nx"])).astype(np.float32)
    ivar = rng.uniform(0.5, 2.0, data.shape).astype(np.float32)
    ivar[0, :3] = 0.0                                  # masked pixels
    src = dict(nx=nsx, ny=nsy, pix=0.25, x0=-0.75, y0=-0.625)   # float32-exact: the batch wrapper takes float32
    return grid, psf.astype(np.float32), data, ivar, src


def test_mapping_rows_reproduce_linear_source():
    """Bilinear interpolation is exact for s(beta) = a + b beta_x + c beta_y: L s equals that plane at the oracle's own
    (separately pinned) ray-shot beta; rows sum to 1 inside, 0 outside (surface brightness conserved)."""
    grid, _, _, _, src = _setup()
    p = _lens()
    L, beta = pixsrc.mapping_matrix(p, grid, src)
    rs = L.sum(axis=1)
    inside = rs > 0
    assert 10 < inside.sum() < inside.size             # both kinds of rows are present
    assert np.allclose(rs[inside], 1.0, atol=1e-13)
    assert np.all(L >= 0) and np.all((L > 0).sum(axis=1) <= 4)
    sx = src["x0"] + src["pix"] * np.arange(src["nx"])
    sy = src["y0"] + src["pix"] * np.arange(src["ny"])
    s = (0.3 + 1.7 * sx[None, :] - 0.9 * sy[:, None]).reshape(-1)
    want = 0.3 + 1.7 * beta[:, 0] - 0.9 * beta[:, 1]
    assert np.allclose((L @ s)[inside], want[inside], atol=1e-12)
    # the inside test is the rectangle of source-pixel centres
    bx, by = beta[:, 0], beta[:, 1]
    rect = (bx >= sx[0]) & (bx < sx[-1]) & (by >= sy[0]) & (by < sy[-1])
    assert np.array_equal(rect, inside)
    # beta really is theta - alpha of the pinned deflection
    ix, iy = 3, 5
    ax, ay = oracle.deflection(p.astype(np.float64), grid["x0"] + ix * grid["pix"], grid["y0"] + iy * grid["pix"])
    assert np.allclose(beta[iy * grid["nx"] + ix], [grid["x0"] + ix * grid["pix"] - ax, grid["y0"] + iy * grid["pix"] - ay])


def test_no_lens_identity_mapping():
    """theta_E -> 0, no shear, no point mass, source grid = image grid: L is the identity on the interior."""
    n, pix = 8, 0.1
    grid = dict(nx=n, ny=n, supersample=1, pix=pix, x0=0.05, y0=0.05)      # away from the lens centre at (0.01,-0.02)
    p = _lens(thetaE=1e-12, gext=0.0)
    L, _ = pixsrc.mapping_matrix(p, grid, dict(nx=n, ny=n, pix=pix, x0=0.05 - 1e-9, y0=0.05 - 1e-9))
    Lin = L.reshape(n, n, n, n)[: n - 1, : n - 1]
    for iy in range(n - 1):
        for ix in range(n - 1):
            assert abs(Lin[iy, ix, iy, ix] - 1.0) < 1e-6


def test_blurring_matrix_is_scipy_convolution():
    grid, psf, _, _, _ = _setup()
    nx, ny = grid["nx"], grid["ny"]
    Bm = pixsrc.blurring_matrix(psf, nx, ny)
    v = np.random.default_rng(1).normal(size=(ny, nx))
    want = scipy.signal.convolve2d(v, psf.astype(np.float64), mode="same", boundary="fill")
    assert np.allclose((Bm @ v.reshape(-1)).reshape(ny, nx), want, atol=1e-13)


def test_curvature_logdet_closed_form():
    """Second difference with zero boundaries has eigenvalues -2 + 2 cos(k pi/(n+1)); g's are mu_i^2 + mu_j^2."""
    nsx, nsy = 7, 5
    g = pixsrc.curvature_g(nsx, nsy)
    mx = -2 + 2 * np.cos(np.arange(1, nsx + 1) * np.pi / (nsx + 1))
    my = -2 + 2 * np.cos(np.arange(1, nsy + 1) * np.pi / (nsy + 1))
    ev = np.sort((mx[None, :] ** 2 + my[:, None] ** 2).reshape(-1))
    assert np.allclose(np.sort(np.linalg.eigvalsh(g)), ev, atol=1e-11)
    # and it is the Hessian of E_S written out pixel by pixel with s = 0 outside
    s = np.random.default_rng(2).normal(size=(nsy, nsx))
    sp = np.pad(s, 1)
    es = 0.0
    for j in range(1, nsy + 1):
        for i in range(1, nsx + 1):
            es += 0.5 * ((sp[j, i - 1] - 2 * sp[j, i] + sp[j, i + 1]) ** 2 + (sp[j - 1, i] - 2 * sp[j, i] + sp[j + 1, i]) ** 2)
    assert np.isclose(0.5 * s.reshape(-1) @ g @ s.reshape(-1), es, rtol=1e-13)


def test_s_mp_is_regularised_least_squares():
    """Eq. 40 is the minimiser of E_D + lambda E_S: solve the stacked least-squares problem with LAPACK's lstsq."""
    grid, psf, data, ivar, src = _setup()
    lam = float(np.float32(0.37))                     # the oracle takes lambda as the float32 the GPU reads
    r = pixsrc.pixsrc_evidence(_lens(), grid, psf, data, ivar, src, lam)
    assert r["flag"] == 0
    L, _ = pixsrc.mapping_matrix(_lens(), grid, src)
    f = pixsrc.blurring_matrix(psf, grid["nx"], grid["ny"]) @ L
    w = ivar.astype(np.float64).reshape(-1)
    Dx = np.kron(np.eye(src["ny"]), pixsrc.second_difference(src["nx"]))
    Dy = np.kron(pixsrc.second_difference(src["ny"]), np.eye(src["nx"]))
    M = np.vstack([np.sqrt(w)[:, None] * f, np.sqrt(lam) * Dx, np.sqrt(lam) * Dy])
    rhs = np.concatenate([np.sqrt(w) * data.astype(np.float64).reshape(-1), np.zeros(2 * Dx.shape[0])])
    s, *_ = scipy.linalg.lstsq(M, rhs)
    assert np.allclose(r["s_mp"].reshape(-1), s, rtol=1e-8, atol=1e-10)
    assert np.isclose(r["chi2"], float(np.sum(w * (f @ s - data.reshape(-1)) ** 2)), rtol=1e-10)
    assert np.allclose(r["model"].reshape(-1), f @ s, atol=1e-10)


@pytest.mark.parametrize("lam", [0.05, 1.0, 30.0])
def test_evidence_is_gaussian_marginal_likelihood(lam):
    """Eq. 43 integrates s out of N(d; f s, C_d) N(s; 0, (lambda g)^-1): the result is N(d; 0, C_d + f (lambda g)^-1 f^T),
    evaluated here directly on the unmasked pixels (no s_MP, no det(F + lambda g)): any wrong sign, missing
    log-determinant or missing N/2 ln(..) term of R-P5 fails."""
    grid, psf, data, ivar, src = _setup()
    r = pixsrc.pixsrc_evidence(_lens(), grid, psf, data, ivar, src, lam)
    L, _ = pixsrc.mapping_matrix(_lens(), grid, src)
    f = pixsrc.blurring_matrix(psf, grid["nx"], grid["ny"]) @ L
    w = ivar.astype(np.float64).reshape(-1)
    m = w > 0
    fm, dm = f[m], data.astype(np.float64).reshape(-1)[m]
    g = pixsrc.curvature_g(src["nx"], src["ny"])
    S = np.diag(1.0 / w[m]) + fm @ np.linalg.inv(np.float64(np.float32(lam)) * g) @ fm.T
    sign, ld = np.linalg.slogdet(S)
    want = -0.5 * dm @ np.linalg.solve(S, dm) - 0.5 * ld - 0.5 * m.sum() * np.log(2 * np.pi)
    assert sign > 0
    assert np.isclose(r["logev"], want, rtol=1e-10)


def test_noise_free_data_recovered_and_batch_wrapper():
    """Data made from a smooth source through the same operator, tiny lambda: the model reproduces the data; the batch
    wrapper returns the per-vector results; lambda <= 0 is flagged."""
    grid, psf, _, ivar, src = _setup()
    p = _lens()
    L, _ = pixsrc.mapping_matrix(p, grid, src)
    f = pixsrc.blurring_matrix(psf, grid["nx"], grid["ny"]) @ L
    jj, ii = np.mgrid[0:src["ny"], 0:src["nx"]]
    s_true = np.exp(-0.5 * ((ii - 3.0) ** 2 + (jj - 2.5) ** 2) / 1.5 ** 2).reshape(-1)
    data = (f @ s_true).reshape(grid["ny"], grid["nx"]).astype(np.float32)
    r = pixsrc.pixsrc_evidence(p, grid, psf, data, ivar, src, 1e-6)
    assert np.max(np.abs(r["model"] - data)) < 1e-4 and r["chi2"] < 1e-5
    lens = np.stack([p, _lens(thetaE=1.1, q=0.7)])
    sg = np.array([[src["x0"], src["y0"], src["pix"]]] * 2, np.float32)
    out = pixsrc.pixsrc_batch(lens, grid, psf, data, ivar, sg, np.array([1e-6, -1.0], np.float32), src["nx"], src["ny"])
    assert np.isclose(out["logev"][0], r["logev"], rtol=1e-12) and out["flag"][0] == 0
    assert out["flag"][1] == 1 and out["logev"][1] == -np.inf


def test_lambda_hat_satisfies_the_stationarity_condition():
    """lambda_hat of Eq. 43.  At the maximum of the evidence over lambda, with s_MP the minimiser of chi2/2 + lambda E_S
    (envelope theorem): d ln P / d lambda = -E_S(s_MP) - 1/2 tr[(F + lambda g)^-1 g] + N_s / (2 lambda) = 0, i.e.
    2 lambda_hat E_S = N_s - lambda_hat tr[(F + lambda_hat g)^-1 g]  (the condition Suyu et al. 2006 give for the optimal lambda).
    Evaluated here from F, g and s_MP rebuilt in numpy, beside the finite-difference slope of ln P itself."""
    grid, psf, _, ivar, src = _setup()
    for seed, p in ((1, _lens()), (2, _lens(thetaE=0.9, gamma=2.2, q=0.7))):
        # data = a smooth source through the operator + noise, so that the evidence has an interior maximum in lambda
        rng = np.random.default_rng(seed)
        Lm, _ = pixsrc.mapping_matrix(p, grid, src)
        f = pixsrc.blurring_matrix(psf, grid["nx"], grid["ny"]) @ Lm
        jj, ii = np.mgrid[0:src["ny"], 0:src["nx"]]
        s_true = 3.0 * np.exp(-((ii - 3.0) ** 2 + (jj - 2.5) ** 2) / 4.0).reshape(-1)
        data = (f @ s_true + rng.normal(0.0, 0.05, f.shape[0])).reshape(grid["ny"], grid["nx"]).astype(np.float32)
        w = np.full(data.shape, 400.0, np.float32)
        w[0, :3] = 0.0
        r = pixsrc.pixsrc_lambda_opt(p, grid, psf, data, w, src, 1e-6, 1e6)
        lam = r["lam_hat"]
        assert 1e-5 < lam < 1e5 and r["flag"] == 0
        wv = w.astype(np.float64).reshape(-1)
        F = f.T @ (wv[:, None] * f)
        g = pixsrc.curvature_g(src["nx"], src["ny"])
        tr = np.trace(np.linalg.solve(F + lam * g, g))
        ns = src["nx"] * src["ny"]
        assert 2 * lam * r["reg"] == pytest.approx(ns - lam * tr, rel=1e-4)
        ev = lambda x: pixsrc.pixsrc_evidence(p, grid, psf, data, w, src, np.exp(x))["logev"]
        x0, h = np.log(lam), 1e-3
        slope = (ev(x0 + h) - ev(x0 - h)) / (2 * h)
        curv = (ev(x0 + h) - 2 * ev(x0) + ev(x0 - h)) / h**2
        assert curv < 0 and abs(slope / curv) < 1e-4                      # distance to the stationary point in ln(lambda)
        assert ev(x0) >= max(ev(x0 + 0.05), ev(x0 - 0.05))
