"""fp64 CPU oracle of the pixelated-source extended-image likelihood (paper Eq. 37-43).

TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rule as oracle/__init__.py): only tests/, smoke() and bench.py's
cpu_baseline leg may import it; it shares nothing with paper_2504_01302_b200.

Every matrix of Table 1 is built DENSE, exactly as the paper writes it, and the linear algebra is
numpy.linalg in fp64 - no sparsity, no blocking, no reuse of the banded structure:

  L  [N_pix, N_s]  source plane -> image plane (Eq. 33 P:246 + bilinear interpolation, "following Suyu et al. 2006" P:269)
  B  [N_pix, N_pix] blurring matrix of the PSF (Eq. 38), the same "same"-size zero-padded convolution as row a4
  f  = B L                                            (Eq. 38)
  C_d^-1 = diag(ivar)                                 (the noise covariance of Eq. 37; ivar = 0 masks a pixel out)
  F  = f^T C_d^-1 f,  D = f^T C_d^-1 d_esr            (Eq. 41, 42)
  s_MP = (F + lambda g)^-1 D                          (Eq. 40)
  ln P(d_esr | f, lambda, g)                          (Eq. 43; "explicit expression ... Suyu et al. (2006), Eq. (19)" P:304)

Readings (DESIGN.md R-P1..5):
  R-P1  image-plane points are the pixel centres of the L1 grid (no supersampling inside the operator).
  R-P2  the source grid is regular, n_sx x n_sy pixels of size p_s, pixel (0,0) centred at (x_s0, y_s0); it is an INPUT
        per parameter vector (the caller may adapt it to the mapped arc).  A ray landing outside the rectangle spanned
        by the source-pixel centres gives an all-zero row of L.
  R-P3  "g" in Eq. 40 is the Hessian of the curvature regulariser E_S = 1/2 sum_pixels [(d2/dx2 s)^2 + (d2/dy2 s)^2] with
        second differences (1,-2,1) and s = 0 outside the grid (so g = Dx^T Dx + Dy^T Dy is positive definite).
  R-P4  lambda is an input per vector (the optimisation of lambda-hat, is a 1-D search over this function).
  R-P5  the evidence is  -E_D(s_MP) - lambda E_S(s_MP) - 1/2 ln det(F + lambda g) + N_s/2 ln lambda + 1/2 ln det g
        - N_d/2 ln 2 pi + 1/2 sum_{ivar>0} ln ivar,  E_D = 1/2 (f s - d)^T C_d^-1 (f s - d),  E_S = 1/2 s^T g s,
        N_d = number of pixels with ivar > 0.  (It is pinned in tests/test_oracle_pixsrc.py against the marginal
        likelihood N(d; 0, C_d + f (lambda g)^-1 f^T) evaluated directly.)
"""
from __future__ import annotations

import numpy as np

from . import NLENS, deflection


def mapping_matrix(params, grid, src_grid):
    """L [ny*nx, n_sy*n_sx] of one parameter vector.  params: the 26 lens numbers (only the mass part is used);
    grid: dict(nx, ny, pix, x0, y0); src_grid: dict(nx, ny, pix, x0, y0) (R-P2).  Returns (L, beta [ny*nx, 2])."""
    nx, ny, pix = int(grid["nx"]), int(grid["ny"]), float(grid["pix"])
    nsx, nsy, ps = int(src_grid["nx"]), int(src_grid["ny"]), float(src_grid["pix"])
    L = np.zeros((ny * nx, nsy * nsx))
    beta = np.zeros((ny * nx, 2))
    p = np.asarray(params, dtype=np.float32).astype(np.float64)
    for iy in range(ny):
        for ix in range(nx):
            thx = float(grid["x0"]) + ix * pix
            thy = float(grid["y0"]) + iy * pix
            ax, ay = deflection(p, thx, thy)
            bx, by = thx - ax, thy - ay                      # Eq. 33
            beta[iy * nx + ix] = (bx, by)
            tx = (bx - float(src_grid["x0"])) / ps
            ty = (by - float(src_grid["y0"])) / ps
            if not (np.isfinite(tx) and np.isfinite(ty)):
                continue
            i0, j0 = int(np.floor(tx)), int(np.floor(ty))
            if i0 < 0 or j0 < 0 or i0 + 1 > nsx - 1 or j0 + 1 > nsy - 1:
                continue                                     # R-P2: outside the source grid
            fx, fy = tx - i0, ty - j0
            r = iy * nx + ix
            L[r, j0 * nsx + i0] = (1 - fx) * (1 - fy)
            L[r, j0 * nsx + i0 + 1] = fx * (1 - fy)
            L[r, (j0 + 1) * nsx + i0] = (1 - fx) * fy
            L[r, (j0 + 1) * nsx + i0 + 1] = fx * fy
    return L, beta


def blurring_matrix(psf, nx, ny):
    """B [ny*nx, ny*nx]: (B v)[iy,ix] = sum_{dy,dx} psf[dy,dx] v[iy-(dy-c), ix-(dx-c)], zero outside (row a4's rule)."""
    psf = np.asarray(psf, dtype=np.float32).astype(np.float64)
    k = psf.shape[0]
    c = k // 2
    Bm = np.zeros((ny * nx, ny * nx))
    for iy in range(ny):
        for ix in range(nx):
            for dy in range(k):
                sy = iy - (dy - c)
                if sy < 0 or sy >= ny:
                    continue
                for dx in range(k):
                    sx = ix - (dx - c)
                    if sx < 0 or sx >= nx:
                        continue
                    Bm[iy * nx + ix, sy * nx + sx] += psf[dy, dx]
    return Bm


def second_difference(n):
    """[n, n] matrix of (1, -2, 1) with zeros outside (R-P3)."""
    return -2.0 * np.eye(n) + np.eye(n, k=1) + np.eye(n, k=-1)


def curvature_g(nsx, nsy):
    """g = Dx^T Dx + Dy^T Dy on the row-major (j, i) source grid (R-P3)."""
    Dx = np.kron(np.eye(nsy), second_difference(nsx))
    Dy = np.kron(second_difference(nsy), np.eye(nsx))
    return Dx.T @ Dx + Dy.T @ Dy


def pixsrc_evidence(params, grid, psf, data, ivar, src_grid, lam, Bm=None):
    """One parameter vector.  Returns dict(logev, chi2, reg, s_mp [n_sy,n_sx], model [ny,nx], logdetA, flag).
    flag = 1 (logev = -inf) if F + lambda g is not positive definite or lambda <= 0."""
    nx, ny = int(grid["nx"]), int(grid["ny"])
    nsx, nsy = int(src_grid["nx"]), int(src_grid["ny"])
    ns = nsx * nsy
    d = np.asarray(data, dtype=np.float32).astype(np.float64).reshape(-1)
    w = np.asarray(ivar, dtype=np.float32).astype(np.float64).reshape(-1)
    lam = float(np.float32(lam))
    out = dict(logev=-np.inf, chi2=np.inf, reg=np.nan, s_mp=np.full((nsy, nsx), np.nan), model=np.full((ny, nx), np.nan),
               logdetA=np.nan, flag=1)
    if not (lam > 0.0 and np.isfinite(lam)):
        return out
    L, _ = mapping_matrix(params, grid, src_grid)
    if Bm is None:
        Bm = blurring_matrix(psf, nx, ny)
    f = Bm @ L                                                # Eq. 38
    F = f.T @ (w[:, None] * f)                                # Eq. 41
    D = f.T @ (w * d)                                         # Eq. 42
    g = curvature_g(nsx, nsy)
    A = F + lam * g
    try:
        ch = np.linalg.cholesky(A)
    except np.linalg.LinAlgError:
        return out
    s = np.linalg.solve(A, D)                                 # Eq. 40
    r = f @ s - d
    ED = 0.5 * float(r @ (w * r))
    ES = 0.5 * float(s @ (g @ s))
    logdetA = 2.0 * float(np.sum(np.log(np.diag(ch))))
    _, logdetg = np.linalg.slogdet(g)
    nd = int(np.count_nonzero(w > 0))
    logev = (-ED - lam * ES - 0.5 * logdetA + 0.5 * ns * np.log(lam) + 0.5 * logdetg
             - 0.5 * nd * np.log(2.0 * np.pi) + 0.5 * float(np.sum(np.log(w[w > 0]))))
    return dict(logev=logev, chi2=2.0 * ED, reg=ES, s_mp=s.reshape(nsy, nsx), model=(f @ s).reshape(ny, nx),
                logdetA=logdetA, flag=0)


def pixsrc_batch(lens, grid, psf, data, ivar, src_grids, lam, nsx, nsy):
    """lens [B,26] float32, src_grids [B,3] float32 = {x_s0, y_s0, p_s} per vector, lam [B] float32."""
    lens = np.ascontiguousarray(lens, dtype=np.float32).reshape(-1, NLENS)
    B = lens.shape[0]
    sg = np.ascontiguousarray(src_grids, dtype=np.float32).reshape(B, 3)
    lam = np.ascontiguousarray(lam, dtype=np.float32).reshape(B)
    Bm = blurring_matrix(psf, int(grid["nx"]), int(grid["ny"]))
    # the mass part must be a valid model (theta_E >= 0, 1 < gamma < 3, 0 < q <= 1, theta_E,BH^2 >= 0: the GLAD_FLAG_LENS_INVALID
    # conditions on lens[2..4], lens[8]); the light slots lens[9..25] do not enter Eq. 37-43
    bad = ~((lens[:, 2] >= 0) & (lens[:, 3] > 1) & (lens[:, 3] < 3) & (lens[:, 4] > 0) & (lens[:, 4] <= 1) & (lens[:, 8] >= 0))
    res = [pixsrc_evidence(lens[b], grid, psf, data, ivar,
                           dict(nx=nsx, ny=nsy, pix=float(sg[b, 2]), x0=float(sg[b, 0]), y0=float(sg[b, 1])),
                           np.float32(-1.0) if (bad[b] or not sg[b, 2] > 0) else lam[b], Bm) for b in range(B)]
    return {k: np.array([r[k] for r in res]) for k in res[0]}


def pixsrc_lambda_opt(params, grid, psf, data, ivar, src_grid, lam_lo, lam_hi, Bm=None):
    """Eq. 43: the evidence "at the optimal regularisation constant" -- lambda_hat = argmax over
    [lam_lo, lam_hi] of ln P(d | f, lambda, g), by scipy's bounded scalar minimiser on x = ln(lambda) applied to pixsrc_evidence
    as it stands (F, D do not depend on lambda; they are rebuilt per call all the same: no reuse, no shortcut).
    Returns dict(lam_hat, and pixsrc_evidence(lam_hat)'s fields).  lam_hat is rounded to float32 (the type the batch call takes)
    and the evidence is evaluated at that rounded value."""
    from scipy.optimize import minimize_scalar
    if Bm is None:
        Bm = blurring_matrix(psf, int(grid["nx"]), int(grid["ny"]))
    neg = lambda x: -pixsrc_evidence(params, grid, psf, data, ivar, src_grid, np.exp(x), Bm)["logev"]
    r = minimize_scalar(neg, bounds=(np.log(lam_lo), np.log(lam_hi)), method="bounded", options=dict(xatol=1e-9, maxiter=200))
    lam_hat = float(np.float32(np.exp(r.x)))
    out = pixsrc_evidence(params, grid, psf, data, ivar, src_grid, lam_hat, Bm)
    out["lam_hat"] = lam_hat
    return out

