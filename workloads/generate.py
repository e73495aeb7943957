"""Seeded synthetic workloads for BASELINE.json:configs.

One numpy default_rng(seed) per config; the draw order below is fixed.  All arrays
handed to either side are float32 / int32; nothing here evaluates the lens model,
the Jeans quadrature, a convolution or a chi-square.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.optimize import nnls
from scipy.special import erf, gamma as gamma_fn, gammaincinv

NLENS, NDYN = 26, 4
Z_D = 0.295
G_NEWTON = 0.004301              # (km/s)^2 pc / Msun
C_KMS = 299792.458
ARCSEC_PER_RAD = 648000.0 / math.pi

# name -> recipe.  "lens"/"dyn" = None switches that half off.
CONFIGS = {
    "C1": dict(seed=0, B=8,
               lens=dict(n=40, pix=0.08, s=1, psf=("gauss", 5), noise=0.01, thetaE=(0.8, 1.2), sie=True,
                         bh=False, n_lens_light=0),
               dyn=dict(n_lum=10, n_mass=10, beta="iso", grid=20, nbins=16, nu=64, per_vector_lum=False),
               fixed_dist=True),
    "C2": dict(seed=1, B=1024,
               lens=dict(n=100, pix=0.05, s=2, psf=("moffat", 21), noise=0.01, thetaE=(1.6, 1.9), sie=False,
                         bh=True, n_lens_light=1),
               dyn=dict(n_lum=20, n_mass=20, beta="scalar", grid=80, nbins=60, nu=128, per_vector_lum=False),
               fixed_dist=False),
    "C4": dict(seed=3, B=8192,
               lens=dict(n=120, pix=0.05, s=3, psf=("moffat", 31), noise=0.02, thetaE=(1.6, 1.9), sie=False,
                         bh=True, n_lens_light=2),
               dyn=None, fixed_dist=False),
    "C5": dict(seed=4, B=4096,
               lens=dict(n=200, pix=0.04, s=3, psf=("moffat", 31), noise=0.02, thetaE=(1.6, 1.9), sie=False,
                         bh=True, n_lens_light=1),
               dyn=dict(n_lum=30, n_mass=30, beta="per_gaussian", grid=160, nbins=100, nu=256,
                        per_vector_lum=True),
               fixed_dist=False),
}
# C3: dynamics-only sweep, 18 cells "C3-<nG>-<grid>-<B>"
for _ng in (10, 20, 40):
    for _g in (40, 80, 160):
        for _b in (256, 4096):
            CONFIGS[f"C3-{_ng}-{_g}-{_b}"] = dict(
                seed=2, B=_b, lens=None,
                dyn=dict(n_lum=_ng, n_mass=_ng, beta="per_gaussian", grid=_g, nbins=100, nu=128,
                         per_vector_lum=False),
                fixed_dist=True)

FOV = 1.0          # kinematic field of view +-1"
KIN_FWHM = 0.1     # BASELINE.json "seeing FWHM 0.1"" (paper: 0.14")
IMG_FWHM = 0.1


def gauss_legendre_u(n: int):
    """n-point Gauss-Legendre on t in [0,1] mapped by u = t^2, w_u = 2 t w_t (reading R-D4)."""
    t, w = np.polynomial.legendre.leggauss(n)
    t = 0.5 * (t + 1.0)
    w = 0.5 * w
    return (t * t).astype(np.float32), (2.0 * t * w).astype(np.float32)


# 7-point Kronrod extension of the 3-point Gauss rule on [-1, 1] (the pair Shampine's TwoD uses): nodes, weights
_K7_X = np.array([-0.9604912687080203, -0.7745966692414834, -0.4342437493468026, 0.0,
                  0.4342437493468026, 0.7745966692414834, 0.9604912687080203])
_K7_W = np.array([0.1046562260264673, 0.2684880898683334, 0.4013974147759622, 0.4509165386584741,
                  0.4013974147759622, 0.2684880898683334, 0.1046562260264673])


def kronrod_composite(panels: int):
    """Composite 7-point Kronrod rule on (0,1): `panels` equal sub-intervals.  The paper's fixed mesh (the region cut into
    64 sub-regions, each into four rectangles, Gauss-Kronrod in each) is 16 x 16 rectangles = this rule with panels = 16 in each
    of the two directions (112 x 112 nodes)."""
    h = 1.0 / panels
    x = np.concatenate([(p + 0.5 * (_K7_X + 1.0)) * h for p in range(panels)])
    w = np.concatenate([0.5 * h * _K7_W for _ in range(panels)])
    return x, w


def jam_sph_rules(kin: dict, panels: int = 16, nr: int = 20, nth: int = 10, nz: int = 96, u_decades: float = 5.0,
                  sigma_max: float = 0.0) -> dict:
    """Inputs of the JAM_sph path (readings R-SPH1..4) for the sky grid of `kin`: polar grid (20 x 10 = "over 200
    points in polar coordinates") log-spaced in r from half the smallest pixel radius to the larger of 3 x the largest pixel
    radius and 4 x sigma_max (the widest luminous Gaussian: the LOS integral reaches that far), uniform in theta
    on [0, pi/2]; radial rule tau on (0,1) and potential rule u = 10^(-u_decades (1 - t)) (log-spaced: the u^2 exp(-a u^2) peaks
    of a sigma = 0.01" black hole seen from r' ~ 60" sit at u ~ 1e-4), both from the composite Kronrod mesh; LOS rule = nz-point
    Gauss-Legendre on (-1,1)."""
    xs, ys = np.asarray(kin["xs"], np.float64), np.asarray(kin["ys"], np.float64)
    rad = np.hypot(*np.meshgrid(xs, ys))
    rmin = max(0.5 * float(rad[rad > 0].min()) if (rad > 0).any() else 1e-3, 1e-4)
    rmax = max(3.0 * float(rad.max()) if rad.max() > 0 else 1.0, 4.0 * float(sigma_max))
    t, w = kronrod_composite(panels)
    L = u_decades * np.log(10.0)
    u = np.exp(-L * (1.0 - t))
    z, wz = np.polynomial.legendre.leggauss(nz)
    f = np.float32
    return dict(rgrid=np.geomspace(rmin, rmax, nr).astype(f), thgrid=np.linspace(0.0, 0.5 * np.pi, nth).astype(f),
                tau=t.astype(f), wtau=w.astype(f), un=u.astype(f), uw=(L * u * w).astype(f), zeta=z.astype(f), wz=wz.astype(f))


def cse_table():
    """(A_i, s_i) of the CSE expansion of the NFW convergence (Eq. A.3-A.5): the table workloads/fit_cse_nfw.py wrote.  An input of
    the method ("predetermined"): this repository's fit, not Oguri (2021)'s 44 pairs (not available, not printed)."""
    import os
    t = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cse_nfw.txt"))
    return t[:, 0].copy(), t[:, 1].copy()


def enfw_params(B: int, seed: int = 11) -> np.ndarray:
    """Per-vector halo {rho_s, r_s [arcsec], q, phi}: a dark-matter halo that carries roughly half the convergence at the Einstein
    radius of the C2 truth (kappa_enfw(1.65") ~ 0.2-0.35), r_s ~ U(8, 20) arcsec (the RXJ1131 class), q ~ U(0.6, 1)."""
    rng = np.random.default_rng(seed)
    out = np.stack([rng.uniform(0.15, 0.3, B), rng.uniform(8.0, 20.0, B), rng.uniform(0.6, 1.0, B), rng.uniform(0.0, np.pi, B)], 1)
    return out.astype(np.float32)


def _psf(kind: str, k: int, pix: float, fwhm: float) -> np.ndarray:
    c = k // 2
    yy, xx = np.mgrid[0:k, 0:k]
    r2 = ((xx - c) ** 2 + (yy - c) ** 2) * pix * pix
    if kind == "gauss":
        sig = fwhm / 2.3548
        p = np.exp(-r2 / (2 * sig * sig))
    else:  # Moffat beta=3: not separable, so a separable shortcut is never the only thing tested
        bm = 3.0
        a = fwhm / (2.0 * math.sqrt(2.0 ** (1.0 / bm) - 1.0))
        p = (1.0 + r2 / (a * a)) ** (-bm)
    return (p / p.sum()).astype(np.float32)


def _kin_kernel(pix: float, fwhm: float) -> np.ndarray:
    """Gaussian of the given FWHM integrated over the square pixel, +-4 sigma, unit sum."""
    sig = fwhm / 2.3548
    hw = int(math.ceil(4.0 * sig / pix))
    e = (np.arange(-hw, hw + 2) - 0.5) * pix
    cdf = 0.5 * (1.0 + erf(e / (sig * math.sqrt(2.0))))
    w1 = np.diff(cdf)
    k = np.outer(w1, w1)
    return (k / k.sum()).astype(np.float32)


def _sigma_crit(ddt_mpc, dd_mpc):
    """Eq. 13, Msun/pc^2."""
    return C_KMS ** 2 / (4 * math.pi * G_NEWTON) * (ddt_mpc * 1e6) / ((1 + Z_D) * (dd_mpc * 1e6) ** 2)


def bh_theta2(mbh, ddt_mpc):
    """theta_E,BH^2 [arcsec^2] = 4 G M (1+z_d)/(c^2 D_dt) (from Eq. 4)."""
    return 4 * G_NEWTON * mbh * (1 + Z_D) / (C_KMS ** 2 * ddt_mpc * 1e6) * ARCSEC_PER_RAD ** 2


def _mass_mge_epl(thetaE, gam, q, ddt, dd, n):
    """Closed-form 1-D MGE of the EPL power law, sigma log-spaced 0.02"-50" (paper decomposes
    to 50"): Sigma_0n = Sigma_crit (3-g)/2 b^t 2^(1-t/2)/Gamma(t/2) sigma_n^-t dln(sigma)."""
    t = gam - 1.0
    b = (2.0 / (1.0 + q)) ** (1.0 / t) * thetaE
    sig = np.geomspace(0.02, 50.0, n)
    dln = math.log(50.0 / 0.02) / (n - 1)
    amp = _sigma_crit(ddt, dd) * (3 - gam) / 2 * b ** t * 2 ** (1 - t / 2) / gamma_fn(t / 2) * sig ** (-t) * dln
    return np.stack([amp, sig, np.full(n, q)], axis=1)


def _lum_mge_sersic(n_ser, re, qp, n, scale=1000.0):
    """1-D MGE (same q' for all Gaussians, footnote P:234) of a Sersic profile by NNLS on a
    log-radial grid; sigma log-spaced 0.02"-10".  Fidelity is irrelevant to parity."""
    bn = gammaincinv(2 * n_ser, 0.5)
    r = np.geomspace(0.01, 20.0, 240)
    prof = np.exp(-bn * ((r / re) ** (1.0 / n_ser) - 1.0))
    sig = np.geomspace(0.02, 10.0, n)
    basis = np.exp(-r[:, None] ** 2 / (2 * sig[None, :] ** 2)) / prof[:, None]
    try:
        amp, _ = nnls(basis, np.ones_like(r), maxiter=200 * n)
    except RuntimeError:                       # scipy's active-set NNLS may cycle; any non-negative table will do
        amp = np.maximum(np.linalg.lstsq(basis, np.ones_like(r), rcond=1e-8)[0], 0.0)
    amp = np.maximum(amp, 1e-4 * amp.max())
    return np.stack([scale * amp, sig, np.full(n, qp)], axis=1)


def _bins(rng, xs, ys, nbins):
    """'Voronoi-like' labels: seeds with radial density ~ 1/r inside the FoV, nearest seed."""
    X, Y = np.meshgrid(xs, ys)
    for _ in range(200):
        r = rng.uniform(0.0, FOV, nbins)
        a = rng.uniform(0.0, 2 * math.pi, nbins)
        sx, sy = r * np.cos(a), r * np.sin(a)
        d2 = (X[..., None] - sx) ** 2 + (Y[..., None] - sy) ** 2
        lab = np.argmin(d2, axis=-1).astype(np.int32)
        if np.unique(lab).size == nbins:
            return lab
    raise RuntimeError("could not draw non-empty bins")


def make_workload(name: str, data_model=None, B: int | None = None) -> dict:
    """Build config `name`.  `data_model(wl) -> (image[ny,nx] or None, vrms[nbins] or None)` returns the
    noise-free model of batch element 0 (the truth vector); None leaves data at zero / unit ivar."""
    cfg = CONFIGS[name]
    rng = np.random.default_rng(cfg["seed"])
    B = cfg["B"] if B is None else int(B)
    L, D = cfg["lens"], cfg["dyn"]
    U = lambda lo, hi: rng.uniform(lo, hi, B)

    # ---- per-vector physical parameters (draw order fixed) ----
    thetaE = U(*(L["thetaE"] if L else (1.6, 1.9)))
    gam = np.full(B, 2.0) if (L and L["sie"]) else U(1.8, 2.2)
    q = U(0.6, 1.0)
    g_ext, phi_ext = U(0.0, 0.1), U(0.0, math.pi)
    has_bh = (L["bh"] if L else True)
    mbh = 10.0 ** U(8.0, 10.0) if has_bh else np.zeros(B)
    xl, yl, pa = U(-0.025, 0.025), U(-0.025, 0.025), U(0.0, math.pi)
    xs_, ys_ = U(-0.2, 0.2), U(-0.2, 0.2)
    Ie_s, Re_s, n_s, q_s, phi_s = U(0.1, 0.3), U(0.1, 0.4), U(1.0, 4.0), U(0.6, 1.0), U(0.0, math.pi)
    Ie_1, Re_1, n_1, q_1 = U(0.01, 0.03), U(1.0, 2.5), U(2.0, 5.0), U(0.6, 1.0)
    Ie_2, Re_2, n_2, q_2 = U(0.02, 0.06), U(0.3, 0.8), U(1.0, 2.5), U(0.6, 1.0)
    inc = np.deg2rad(U(60.0, 90.0))
    if cfg["fixed_dist"]:
        dd, ddt = np.full(B, 775.0), np.full(B, 1823.0)          # Table 3
    else:
        dd, ddt = U(600.0, 1000.0), U(1000.0, 4000.0)
    ups = U(0.9, 1.1)
    # truth = element 0 (Table 3)
    thetaE[0] = 1.0 if name == "C1" else 1.65
    gam[0], q[0], g_ext[0], phi_ext[0] = 2.0, 0.8, 0.09, 1.42
    mbh[0] = 5e9 if has_bh else 0.0
    xl[0], yl[0], pa[0] = 0.0, 0.0, math.radians(30.0)
    xs_[0], ys_[0], Ie_s[0], Re_s[0], n_s[0], q_s[0], phi_s[0] = 0.08, -0.05, 0.2, 0.2, 2.0, 0.8, 0.7
    Ie_1[0], Re_1[0], n_1[0], q_1[0] = 0.02, 1.85, 4.0, 0.8
    inc[0], dd[0], ddt[0], ups[0] = math.radians(84.3), 775.0, 1823.0, 1.0

    wl = {"name": name, "B": B, "lens": None, "dyn": None, "ddt": ddt.astype(np.float32), "z_d": Z_D}

    if L:
        p = np.zeros((B, NLENS))
        p[:, 0], p[:, 1], p[:, 2], p[:, 3], p[:, 4], p[:, 5] = xl, yl, thetaE, gam, q, pa
        p[:, 6], p[:, 7] = g_ext, phi_ext
        p[:, 8] = bh_theta2(mbh, ddt)
        p[:, 9:16] = np.stack([xs_, ys_, Ie_s, Re_s, n_s, q_s, phi_s], axis=1)
        if L["n_lens_light"] >= 1:
            p[:, 16:21] = np.stack([Ie_1, Re_1, n_1, q_1, pa], axis=1)
        if L["n_lens_light"] >= 2:
            p[:, 21:26] = np.stack([Ie_2, Re_2, n_2, q_2, pa], axis=1)
        # the C ABI takes the grid as fp32: the numbers are made fp32-representable HERE so that the fp64 oracle and the library get
        # the same grid (0.05 and -2.475 are not: rays 1e-7 arcsec apart move the peak of a magnified n = 3.8 source by 1.4e-4)
        n, pix = L["n"], float(np.float32(L["pix"]))
        x0 = float(np.float32(-(n - 1) / 2 * pix))
        grid = dict(nx=n, ny=n, supersample=L["s"], pix=pix, x0=x0, y0=x0)
        wl["lens"] = dict(params=p.astype(np.float32), grid=grid,
                          psf=_psf(L["psf"][0], L["psf"][1], pix, IMG_FWHM), noise=L["noise"],
                          data=np.zeros((n, n), np.float32), ivar=np.ones((n, n), np.float32))

    if D:
        dp = np.stack([inc, dd, mbh, ups], axis=1).astype(np.float32)
        g = D["grid"]
        spix = 2 * FOV / g
        ax = ((np.arange(g) - (g - 1) / 2) * spix).astype(np.float32)     # exactly antisymmetric
        mass = np.stack([_mass_mge_epl(thetaE[b], gam[b], q[b], ddt[b], dd[b], D["n_mass"]) for b in range(B)])
        if D["per_vector_lum"]:
            lum = np.stack([_lum_mge_sersic(n_1[b], Re_1[b], q_1[b], D["n_lum"]) for b in range(B)])
        else:
            lum = _lum_mge_sersic(4.0, 1.85, 0.8, D["n_lum"])
        if D["beta"] == "iso":
            beta = np.zeros(B)
        elif D["beta"] == "scalar":
            beta = U(-0.3, 0.5)
            beta[0] = 0.15
        else:
            beta = rng.uniform(-0.3, 0.5, (B, D["n_lum"]))
            beta[0, :] = 0.15
        un, uw = gauss_legendre_u(D["nu"])
        kin = dict(xs=ax, ys=ax.copy(), bin_id=_bins(rng, ax, ax, D["nbins"]), nbins=D["nbins"],
                   kernel=_kin_kernel(spix, KIN_FWHM), vrms_obs=np.zeros(D["nbins"], np.float32),
                   vrms_ivar=np.ones(D["nbins"], np.float32), u_nodes=un, u_weights=uw)
        wl["dyn"] = dict(params=dp, lum_mge=lum.astype(np.float32), mass_mge=mass.astype(np.float32),
                         beta=beta.astype(np.float32), kin=kin)

    if data_model is not None:
        img, vr = data_model(subset(wl, [0]))
        nrng = np.random.default_rng(cfg["seed"] + 1000)
        if L and img is not None:
            sig = L["noise"]
            wl["lens"]["data"] = (np.asarray(img, np.float64) + nrng.normal(0.0, sig, img.shape)).astype(np.float32)
            wl["lens"]["ivar"] = np.full(img.shape, 1.0 / sig ** 2, np.float32)
        if D and vr is not None:
            vr = np.asarray(vr, np.float64)
            wl["dyn"]["kin"]["vrms_obs"] = (vr * (1.0 + nrng.normal(0.0, 0.02, vr.shape))).astype(np.float32)  # Eq. 60
            wl["dyn"]["kin"]["vrms_ivar"] = (1.0 / (0.02 * vr) ** 2).astype(np.float32)
    return wl


# Synthetic lensed-quasar observations (Eq. 35-36): an RXJ1131-like quad for the truth vector (batch element 0) of each config
# family.  These are DATA: image positions [arcsec] and delays [days] of a point source at the truth source centre
# (0.08, -0.05), written once by tests/quasar_util.mock_quasar (oracle deflection + MINPACK, seed 0: positions + N(0, 0.004"),
# delays x (1 + N(0, 0.03))) and rounded to the digits below; tests/test_oracle_quasar.py checks that the oracle finds them
# consistent with the truth vector (chi2 of the order of the number of data points).
_QUASAR = {
    "C1": dict(theta=[[0.3763, -1.0949], [0.8562, 0.4753], [0.2470, 1.0287], [-0.8162, 0.0215]], ref=0,
               dt_obs=[0.0, 7.2228, 6.3046, 13.7051], sigma_dt=[0.0, 0.25, 0.25, 0.4112]),
    "C2": dict(theta=[[-1.4223, -0.0663], [0.4798, -1.8253], [1.4803, 0.5375], [0.1286, 1.7884]], ref=1,
               dt_obs=[28.9663, 0.0, 18.6398, 10.9334], sigma_dt=[0.8690, 0.0, 0.5592, 0.3280]),
}


def quasar_data(name: str) -> dict:
    """Quasar observations for config `name` (C4, C5 share C2's truth mass model): dict(theta [4,2], sigma_theta [4], ref,
    dt_obs [4] days relative to image ref, sigma_dt [4]; 0 = the reference image itself), float64."""
    q = _QUASAR["C1" if name == "C1" else "C2"]
    th = np.asarray(q["theta"], np.float64)
    return dict(theta=th, sigma_theta=np.full(len(th), 0.004), ref=int(q["ref"]),
                dt_obs=np.asarray(q["dt_obs"], np.float64), sigma_dt=np.asarray(q["sigma_dt"], np.float64))


def subset(wl: dict, idx) -> dict:
    """Same static data, only the batch elements `idx` (for parity sub-batches)."""
    idx = np.asarray(idx, dtype=np.int64)
    out = {"name": wl["name"], "B": int(idx.size), "lens": None, "dyn": None,
           "ddt": np.ascontiguousarray(wl["ddt"][idx]), "z_d": wl["z_d"]}
    if wl["lens"]:
        out["lens"] = dict(wl["lens"])
        out["lens"]["params"] = np.ascontiguousarray(wl["lens"]["params"][idx])
    if wl["dyn"]:
        d = dict(wl["dyn"])
        d["params"] = np.ascontiguousarray(d["params"][idx])
        d["beta"] = np.ascontiguousarray(d["beta"][idx])
        if d["mass_mge"].ndim == 3:
            d["mass_mge"] = np.ascontiguousarray(d["mass_mge"][idx])
        if d["lum_mge"].ndim == 3:
            d["lum_mge"] = np.ascontiguousarray(d["lum_mge"][idx])
        out["dyn"] = d
    return out


def pixsrc_inputs(wl: dict, nsx: int, nsy: int, seed: int = 7) -> dict:
    """Inputs of the pixelated-source likelihood (Eq. 37-43) for the lens vectors of `wl`: a source grid per vector
    centred on that vector's source position (half-width ~U(0.5, 0.8) arcsec, "O(10^3)" source pixels at 32 x 32)
    and a regularisation constant lambda = 10^U(-1, 1).  Only seeded draws; none of the method's arithmetic."""
    rng = np.random.default_rng(seed)
    p = wl["lens"]["params"]
    B = p.shape[0]
    hw = rng.uniform(0.5, 0.8, B)
    ps = 2.0 * hw / (max(nsx, nsy) - 1)
    sg = np.stack([p[:, 9] - (nsx - 1) / 2 * ps, p[:, 10] - (nsy - 1) / 2 * ps, ps], axis=1).astype(np.float32)
    lam = (10.0 ** rng.uniform(-1.0, 1.0, B)).astype(np.float32)
    return dict(src_grids=sg, lam=lam, nsx=int(nsx), nsy=int(nsy))
