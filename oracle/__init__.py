"""ctypes loader for the fp64 CPU oracle (oracle/glad_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It
shares nothing with paper_2504_01302_b200 (no import in either direction).

`build()` compiles the C file with gcc (-O2, no fast-math, OpenMP over the batch).
All array arguments are numpy; float32 inputs are the very arrays the CUDA path
reads (the C code promotes them to double), outputs are float64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "glad_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "jam_sph_oracle.c")]
_LIB = os.path.join(_HERE, "libglad_oracle.so")
_lib = None

NLENS = 26
NDYN = 4
FLAG_LENS_INVALID, FLAG_DYN_INVALID, FLAG_BIN_INVALID = 1, 2, 4


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, *_SRCS, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        d, i, fp, dp, ip = C.c_double, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(C.c_int32)
        L.glad_oracle_num_threads.restype = i
        L.glad_oracle_sersic_bn.restype = d
        L.glad_oracle_sersic_bn.argtypes = [d]
        L.glad_oracle_sersic.restype = d
        L.glad_oracle_sersic.argtypes = [d] * 8
        L.glad_oracle_epl_alpha.restype = None
        L.glad_oracle_epl_alpha.argtypes = [d] * 5 + [dp, dp]
        L.glad_oracle_deflection.restype = None
        L.glad_oracle_deflection.argtypes = [dp, d, d, dp, dp]
        L.glad_oracle_lens_image_batch.restype = i
        L.glad_oracle_lens_image_batch.argtypes = [fp, i, i, i, i, d, d, d, fp, i, fp, fp, dp, dp, ip]
        L.glad_oracle_lens_image_batch_kinds.restype = i
        L.glad_oracle_lens_image_batch_kinds.argtypes = [fp, i, i, i, i, d, d, d, fp, i, fp, fp, ip, dp, dp, ip]
        L.glad_oracle_chameleon.restype = d
        L.glad_oracle_chameleon.argtypes = [d] * 7
        L.glad_oracle_jam_sigv2_point.restype = d
        L.glad_oracle_jam_sigv2_point.argtypes = [d, d, d, i, dp, dp, dp, dp, i, dp, dp, dp, i, dp, dp]
        L.glad_oracle_jam_vrms_batch.restype = i
        L.glad_oracle_jam_vrms_batch.argtypes = [fp, i, fp, i, C.c_long, fp, i, C.c_long, fp, i, i, i, fp, fp,
                                                 ip, i, fp, i, fp, fp, fp, fp, i, dp, dp, dp, dp, ip]
        L.glad_oracle_kin_bins.restype = i
        L.glad_oracle_kin_bins.argtypes = [dp, dp, i, i, ip, i, fp, i, fp, fp, dp, dp]
        L.glad_oracle_joint.restype = None
        L.glad_oracle_joint.argtypes = [dp, dp, i, dp]
        L.glad_oracle_bh_theta2.restype = d
        L.glad_oracle_bh_theta2.argtypes = [d, d, d]
        L.glad_oracle_mge_f_sigma.restype = d
        L.glad_oracle_mge_f_sigma.argtypes = [i, dp, d, i]
        L.glad_oracle_mge1d.restype = i
        L.glad_oracle_mge1d.argtypes = [i, dp, i, d, d, i, dp]
        L.glad_oracle_sigma_crit.restype = d
        L.glad_oracle_sigma_crit.argtypes = [d, d, d]
        L.glad_oracle_deflection_sheet.restype = None
        L.glad_oracle_deflection_sheet.argtypes = [dp, d, d, d, d, d, dp, dp]
        L.glad_oracle_potential_sheet.restype = d
        L.glad_oracle_potential_sheet.argtypes = [dp, d, d, d, d, d]
        L.glad_oracle_hessian_sheet.restype = None
        L.glad_oracle_hessian_sheet.argtypes = [dp, d, d, d, d, d, dp]
        L.glad_oracle_sheet_kappa.restype = d
        L.glad_oracle_sheet_kappa.argtypes = [d] * 5
        L.glad_oracle_lens_image_batch_sheet.restype = i
        L.glad_oracle_lens_image_batch_sheet.argtypes = [fp, i, i, i, i, d, d, d, fp, i, fp, fp, ip, fp, d, d, dp, dp, ip]
        L.glad_oracle_quasar_batch_sheet.restype = i
        L.glad_oracle_quasar_batch_sheet.argtypes = [fp, fp, fp, d, d, i, i, dp, dp, i, dp, dp, dp, dp, dp, dp, dp, dp]
        L.glad_oracle_potential.restype = d
        L.glad_oracle_potential.argtypes = [dp, d, d]
        L.glad_oracle_hessian.restype = None
        L.glad_oracle_hessian.argtypes = [dp, d, d, dp]
        L.glad_oracle_tdelay_const.restype = d
        L.glad_oracle_quasar_batch.restype = i
        L.glad_oracle_quasar_batch.argtypes = [fp, fp, i, i, dp, dp, i, dp, dp, dp, dp, dp, dp, dp, dp]
        L.glad_oracle_set_cse_table.restype = i
        L.glad_oracle_set_cse_table.argtypes = [i, dp, dp]
        L.glad_oracle_nfw_kappa.restype = d
        L.glad_oracle_nfw_kappa.argtypes = [d]
        L.glad_oracle_enfw.restype = None
        L.glad_oracle_enfw.argtypes = [dp, d, d, dp, dp, dp, dp, dp]
        L.glad_oracle_lens_image_batch_halo.restype = i
        L.glad_oracle_lens_image_batch_halo.argtypes = [fp, i, i, i, i, d, d, d, fp, i, fp, fp, ip, fp, d, d, fp, dp, dp, ip]
        L.glad_oracle_quasar_batch_halo.restype = i
        L.glad_oracle_quasar_batch_halo.argtypes = [fp, fp, fp, d, d, fp, i, i, dp, dp, i, dp, dp, dp, dp, dp, dp, dp, dp]
        L.glad_oracle_jam_sph_intrinsic.restype = None
        L.glad_oracle_jam_sph_intrinsic.argtypes = [d, d, i, dp, dp, dp, dp, i, dp, dp, dp, d, i, dp, dp, i, dp, dp, dp]
        L.glad_oracle_jam_sph_los.restype = d
        L.glad_oracle_jam_sph_los.argtypes = [d, d, d, i, dp, dp, dp, i, dp, i, dp, dp, d, i, dp, dp]
        L.glad_oracle_jam_sph_vrms_batch.restype = i
        L.glad_oracle_jam_sph_vrms_batch.argtypes = [fp, i, fp, i, C.c_long, fp, i, C.c_long, fp, i, i, i, fp, fp, ip, i, fp, i,
                                                     fp, fp, i, fp, i, fp, i, fp, fp, i, fp, fp, i, fp, fp, dp, dp, dp, dp, ip]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().glad_oracle_num_threads())


def sersic_bn(n: float) -> float:
    return float(lib().glad_oracle_sersic_bn(float(n)))


def sersic(dx, dy, Ie, Re, n, q, phi, bn=None) -> float:
    bn = sersic_bn(n) if bn is None else bn
    return float(lib().glad_oracle_sersic(dx, dy, Ie, Re, n, q, phi, bn))


def epl_alpha(x, y, thetaE, gamma, q):
    ax, ay = C.c_double(), C.c_double()
    lib().glad_oracle_epl_alpha(x, y, thetaE, gamma, q, C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def deflection(params, thx, thy, lam=1.0, sheet=None):
    """sheet = (r_core, r_tr) switches the internal mass sheet on (Eq. 6, 50; readings R-S1..3) with constant lam."""
    p = np.ascontiguousarray(params, dtype=np.float64)
    assert p.size == NLENS
    ax, ay = C.c_double(), C.c_double()
    rc, rt = sheet if sheet is not None else (0.0, 0.0)
    lib().glad_oracle_deflection_sheet(_ptr(p, C.c_double), float(lam), float(rc), float(rt), thx, thy, C.byref(ax), C.byref(ay))
    return ax.value, ay.value


def sheet_kappa(lam, rc, rt, dx, dy) -> float:
    """(1 - lam) S(R) of Eq. 50 normalised to S(0) = 1."""
    return float(lib().glad_oracle_sheet_kappa(float(lam), float(rc), float(rt), float(dx), float(dy)))


def bh_theta2(Mbh, Ddt_mpc, zd) -> float:
    return float(lib().glad_oracle_bh_theta2(float(Mbh), float(Ddt_mpc), float(zd)))


LIGHT_SERSIC, LIGHT_CHAMELEON = 0, 1


def chameleon(dx, dy, I0, wc, wt, q, phi) -> float:
    """Eq. 47."""
    return float(lib().glad_oracle_chameleon(dx, dy, I0, wc, wt, q, phi))


def lens_image_batch(lens, grid, psf, data=None, ivar=None, want_images=True, kinds=None, lam=None, sheet=None, enfw=None):
    """grid = dict(nx, ny, supersample, pix, x0, y0). kinds = None (all Sersic) or 3 ints (source, lens light 1, 2):
    0 Sersic, 1 Chameleon (slot = {I_0, w_c, w_t, q, phi}). lam [B] + sheet = (r_core, r_tr): internal mass sheet.
    Returns dict(images, chi2, flags)."""
    lens = _f32(lens).reshape(-1, NLENS)
    B = lens.shape[0]
    nx, ny = int(grid["nx"]), int(grid["ny"])
    psf = _f32(psf)
    k = psf.shape[0]
    data, ivar = _f32(data), _f32(ivar)
    images = np.empty((B, ny, nx), np.float64) if want_images else None
    chi2 = np.empty(B, np.float64)
    flags = np.zeros(B, np.int32)
    kk = None if kinds is None else np.ascontiguousarray(kinds, dtype=np.int32).reshape(3)
    lm = None if lam is None else _f32(lam).reshape(-1)
    assert lm is None or (lm.size == B and sheet is not None)
    src, srt = sheet if (sheet is not None and lm is not None) else (0.0, 0.0)
    nf = None if enfw is None else _f32(enfw).reshape(B, 4)          # eNFW halo {rho_s, r_s, q, phi} per vector (set_cse_table first)
    rc = lib().glad_oracle_lens_image_batch_halo(
        _ptr(lens, C.c_float), B, nx, ny, int(grid["supersample"]), float(grid["pix"]), float(grid["x0"]),
        float(grid["y0"]), _ptr(psf, C.c_float), k, _ptr(data, C.c_float), _ptr(ivar, C.c_float), _ptr(kk, C.c_int32),
        _ptr(lm, C.c_float), float(src), float(srt), _ptr(nf, C.c_float), _ptr(images, C.c_double), _ptr(chi2, C.c_double),
        _ptr(flags, C.c_int32))
    if rc != 0:
        raise ValueError("oracle: bad lens arguments")
    return {"images": images, "chi2": chi2, "flags": flags}


def jam_vrms_batch(dyn, lum_mge, mass_mge, beta, kin, want_maps=False):
    """kin = dict(xs, ys, bin_id, nbins, kernel, vrms_obs, vrms_ivar, u_nodes, u_weights).
    lum_mge / mass_mge: [n,3] (shared) or [B,n,3] (per vector). beta: [B] or [B,n_lum].
    Returns dict(vrms, chi2, flags[, v2map, sbmap])."""
    dyn = _f32(dyn).reshape(-1, NDYN)
    B = dyn.shape[0]
    lum, mass, beta = _f32(lum_mge), _f32(mass_mge), _f32(beta)
    n_lum, n_mass = lum.shape[-2], mass.shape[-2]
    lum_stride = 0 if lum.ndim == 2 else n_lum * 3
    mass_stride = 0 if mass.ndim == 2 else n_mass * 3
    per_g = 1 if beta.ndim == 2 else 0
    xs, ys = _f32(kin["xs"]), _f32(kin["ys"])
    nx, ny = xs.size, ys.size
    bin_id = np.ascontiguousarray(kin["bin_id"], dtype=np.int32)
    nbins = int(kin["nbins"])
    kern = _f32(kin["kernel"])
    vo, vi = _f32(kin.get("vrms_obs")), _f32(kin.get("vrms_ivar"))
    un, uw = _f32(kin["u_nodes"]), _f32(kin["u_weights"])
    vrms = np.empty((B, nbins), np.float64)
    chi2 = np.empty(B, np.float64)
    flags = np.zeros(B, np.int32)
    v2map = np.empty((B, ny, nx), np.float64) if want_maps else None
    sbmap = np.empty((B, ny, nx), np.float64) if want_maps else None
    rc = lib().glad_oracle_jam_vrms_batch(
        _ptr(dyn, C.c_float), B, _ptr(lum, C.c_float), n_lum, lum_stride, _ptr(mass, C.c_float), n_mass,
        mass_stride, _ptr(beta, C.c_float), per_g, nx, ny, _ptr(xs, C.c_float), _ptr(ys, C.c_float),
        _ptr(bin_id, C.c_int32), nbins, _ptr(kern, C.c_float), kern.shape[0], _ptr(vo, C.c_float),
        _ptr(vi, C.c_float), _ptr(un, C.c_float), _ptr(uw, C.c_float), un.size, _ptr(vrms, C.c_double),
        _ptr(chi2, C.c_double), _ptr(v2map, C.c_double), _ptr(sbmap, C.c_double), _ptr(flags, C.c_int32))
    if rc != 0:
        raise ValueError("oracle: bad jam arguments")
    out = {"vrms": vrms, "chi2": chi2, "flags": flags}
    if want_maps:
        out["v2map"], out["sbmap"] = v2map, sbmap
    return out


def jam_sigv2_point(xp, yp, inc, sig_k, q_k, nu0_k, b_k, sig_j, q_j, rho0_j, u_nodes, u_weights) -> float:
    """Raw quadrature at one sky point, all lengths pc, intrinsic (deprojected) tables."""
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    sig_k, q_k, nu0_k, b_k, sig_j, q_j, rho0_j, un, uw = map(
        f, (sig_k, q_k, nu0_k, b_k, sig_j, q_j, rho0_j, u_nodes, u_weights))
    P = lambda a: _ptr(a, C.c_double)
    return float(lib().glad_oracle_jam_sigv2_point(
        xp, yp, inc, sig_k.size, P(sig_k), P(q_k), P(nu0_k), P(b_k), sig_j.size, P(sig_j), P(q_j), P(rho0_j),
        un.size, P(un), P(uw)))


def kin_bins(sv2, sb, bin_id, nbins, kernel, vrms_obs=None, vrms_ivar=None):
    """Rows a7+a8 on given fp64 maps [ny,nx]. Returns (vrms[nbins], chi2, bad)."""
    sv2 = np.ascontiguousarray(sv2, dtype=np.float64)
    sb = np.ascontiguousarray(sb, dtype=np.float64)
    ny, nx = sv2.shape
    bin_id = np.ascontiguousarray(bin_id, dtype=np.int32)
    kern = _f32(kernel)
    vo, vi = _f32(vrms_obs), _f32(vrms_ivar)
    vr = np.empty(nbins, np.float64)
    x2 = C.c_double(0.0)
    bad = lib().glad_oracle_kin_bins(_ptr(sv2, C.c_double), _ptr(sb, C.c_double), nx, ny, _ptr(bin_id, C.c_int32),
                                     nbins, _ptr(kern, C.c_float), kern.shape[0], _ptr(vo, C.c_float),
                                     _ptr(vi, C.c_float), _ptr(vr, C.c_double), C.byref(x2))
    return vr, x2.value, int(bad)


def joint_loglike(chi2_lens, chi2_dyn):
    a = np.ascontiguousarray(chi2_lens, dtype=np.float64)
    b = np.ascontiguousarray(chi2_dyn, dtype=np.float64)
    out = np.empty_like(a)
    lib().glad_oracle_joint(_ptr(a, C.c_double), _ptr(b, C.c_double), a.size, _ptr(out, C.c_double))
    return out


# ---- 1-D MGE of a radial profile (Eq. 44-46) ----
PROFILE_SERSIC, PROFILE_EPL, PROFILE_CHAMELEON = 0, 1, 2
MGE_EULER_P = 12          # reading R-M1 (the paper does not print P)


def mge_f_sigma(kind, prof, sigma, P=MGE_EULER_P) -> float:
    """Eq. 45 at one sigma.  prof = [I_e, R_e, n, q'] (Sersic) or [scale, theta_E, gamma, q] (EPL)."""
    pr = np.ascontiguousarray(prof, dtype=np.float64)
    assert pr.size == 4
    return float(lib().glad_oracle_mge_f_sigma(int(kind), _ptr(pr, C.c_double), float(sigma), int(P)))


def mge1d(kind, prof, n_gauss, sigma_lo, sigma_hi, P=MGE_EULER_P):
    """Eq. 46: rows {A_n, sigma_n, q'} [n_gauss,3] (fp64) of one profile."""
    pr = np.ascontiguousarray(prof, dtype=np.float64)
    assert pr.size == 4
    out = np.empty((int(n_gauss), 3), np.float64)
    rc = lib().glad_oracle_mge1d(int(kind), _ptr(pr, C.c_double), int(n_gauss), float(sigma_lo), float(sigma_hi),
                                 int(P), _ptr(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle: bad mge1d arguments")
    return out


def mge1d_batch(kind, prof, n_gauss, sigma_lo, sigma_hi, P=MGE_EULER_P):
    """prof [B,4] float32 (the array the CUDA path reads) -> [B,n_gauss,3] fp64."""
    prof = _f32(prof).reshape(-1, 4)
    return np.stack([mge1d(kind, prof[b].astype(np.float64), n_gauss, sigma_lo, sigma_hi, P) for b in range(prof.shape[0])])


def sigma_crit(Ddt_mpc, Dd_mpc, zd) -> float:
    return float(lib().glad_oracle_sigma_crit(float(Ddt_mpc), float(Dd_mpc), float(zd)))


def model_tables(lens, dyn, ddt, zd, n_lum, n_mass, lum_range, mass_range, P=MGE_EULER_P, tracer_kind=PROFILE_SERSIC,
                 lam=None, sheet=None, enfw=None, halo=None):
    """The self-consistent joint model of P:406 / Fig. 2 (reading R-M3): from the lens vector and the distances
    derive (a) the luminous MGE = Eq. 46 of lens-light component #1 (lens[16:20]; Sersic, or Chameleon with tracer_kind), (b) the mass MGE = Eq. 46 of
    Sigma_crit * kappa_epl (Eq. 13, B.1-B.3), (c) lens[8] = theta_E,BH^2 from M_BH = dyn[2] (Eq. 4).
    Returns (lens' [B,26] float32, lum [B,n_lum,3] float32, mass [B,n_mass,3] float32): tables rounded to the
    float32 the batch calls take.  lam [B] + sheet = dict(rc, rt, n, sigma_lo, sigma_hi): internal mass sheet; the mass
    table then has n_mass + sheet["n"] rows (lam x the EPL rows, then the sheet's round Gaussians).  enfw [B,4] + halo =
    dict(n, sigma_lo, sigma_hi): the eNFW halo's rows (Eq. 46 of Sigma_crit lam kappa_enfw, profile kind 3, q' = the halo's q)
    come last (set_cse_table first); a halo with rho_s = 0 gives rows of zero amplitude."""
    lens = _f32(lens).reshape(-1, NLENS).copy()
    dyn = _f32(dyn).reshape(-1, NDYN)
    ddt = _f32(ddt).reshape(-1)
    B = lens.shape[0]
    lum = np.empty((B, n_lum, 3), np.float32)
    mass = None
    for b in range(B):
        Ie, Re, n, q = (float(v) for v in lens[b, 16:20])
        lum[b] = mge1d(tracer_kind, [Ie, Re, n, q], n_lum, *lum_range, P=P)   # Chameleon tracer: the slots are {I_0, w_c, w_t, q}
        sc = sigma_crit(float(ddt[b]), float(dyn[b, 1]), zd)
        m = mge1d(PROFILE_EPL, [sc, float(lens[b, 2]), float(lens[b, 3]), float(lens[b, 4])], n_mass, *mass_range, P=P)
        if lam is not None:
            # Sigma_int = Sigma_crit [lam kappa_epl + (1 - lam) S(R)] (Eq. 6, 12, 50; readings R-S1..3).  The sheet is round
            # (q' = 1), the EPL is not, so it gets rows of its own: a round Chameleon-shaped profile (Eq. 47 at q = 1:
            # I_0/2 (1/sqrt(R^2+w_c^2) - 1/sqrt(R^2+w_t^2))) expanded by Eq. 46 on sheet_n sigmas in [sheet_lo, sheet_hi]
            lb, rc, rt = float(np.float32(lam[b])), float(sheet["rc"]), float(sheet["rt"])
            i0 = 2.0 * sc * (1.0 - lb) / (1.0 / rc - 1.0 / rt)
            sh = mge1d(PROFILE_CHAMELEON, [i0, rc, rt, 1.0], int(sheet["n"]), float(sheet["sigma_lo"]), float(sheet["sigma_hi"]), P=P)
            m[:, 0] *= lb
            m = np.concatenate([m, sh])
        if enfw is not None:
            nf = [float(np.float32(v)) for v in np.asarray(enfw)[b]]
            lb = 1.0 if lam is None else float(np.float32(lam[b]))
            hr = mge1d(3, [sc * nf[0], nf[1], 0.0, nf[2]], int(halo["n"]), float(halo["sigma_lo"]), float(halo["sigma_hi"]), P=P)
            hr[:, 0] *= lb
            m = np.concatenate([m, hr])
        if mass is None:
            mass = np.empty((B, m.shape[0], 3), np.float32)
        mass[b] = m
        lens[b, 8] = bh_theta2(float(dyn[b, 2]), float(ddt[b]), zd)
    return lens, lum, mass


# ---- SURVEY.md 8(f) rank 4 (quasar part): image-position and time-delay chi^2 (Eq. 35-36) ----
def potential(params, thx, thy, lam=1.0, sheet=None) -> float:
    """psi(theta) of EPL + shear + point mass (readings R-Q4) [+ internal mass sheet]."""
    p = np.ascontiguousarray(params, dtype=np.float64)
    assert p.size == NLENS
    rc, rt = sheet if sheet is not None else (0.0, 0.0)
    return float(lib().glad_oracle_potential_sheet(_ptr(p, C.c_double), float(lam), float(rc), float(rt), float(thx), float(thy)))


def hessian(params, thx, thy, lam=1.0, sheet=None):
    """(psi_xx, psi_xy, psi_yy) at theta."""
    p = np.ascontiguousarray(params, dtype=np.float64)
    assert p.size == NLENS
    h = np.empty(3, np.float64)
    rc, rt = sheet if sheet is not None else (0.0, 0.0)
    lib().glad_oracle_hessian_sheet(_ptr(p, C.c_double), float(lam), float(rc), float(rt), float(thx), float(thy), _ptr(h, C.c_double))
    return h


def tdelay_const() -> float:
    """days per (Mpc arcsec^2)."""
    return float(lib().glad_oracle_tdelay_const())


def quasar_batch(lens, ddt, qso, lam=None, sheet=None, enfw=None):
    """qso = dict(theta [n_img,2], sigma_theta [n_img], ref, dt_obs [n_img], sigma_dt [n_img]) (float64).
    lam [B] + sheet = (r_core, r_tr): internal mass sheet.
    Returns dict(chi2_img, chi2_tmd [B]; theta_pre [B,n_img,2]; dt_pre [B,n_img]; beta [B,2]; last_step [B,n_img])."""
    lens = _f32(lens).reshape(-1, NLENS)
    ddt = _f32(ddt).reshape(-1)
    B = lens.shape[0]
    assert ddt.size == B
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    th, st, dt, sd = f(qso["theta"]).reshape(-1, 2), f(qso["sigma_theta"]), f(qso["dt_obs"]), f(qso["sigma_dt"])
    n = th.shape[0]
    assert st.size == n and dt.size == n and sd.size == n
    out = {"chi2_img": np.empty(B), "chi2_tmd": np.empty(B), "theta_pre": np.empty((B, n, 2)),
           "dt_pre": np.empty((B, n)), "beta": np.empty((B, 2)), "last_step": np.empty((B, n))}
    P = lambda a: _ptr(a, C.c_double)
    lm = None if lam is None else _f32(lam).reshape(-1)
    assert lm is None or (lm.size == B and sheet is not None)
    src, srt = sheet if (sheet is not None and lm is not None) else (0.0, 0.0)
    nf = None if enfw is None else _f32(enfw).reshape(B, 4)
    rc = lib().glad_oracle_quasar_batch_halo(_ptr(lens, C.c_float), _ptr(ddt, C.c_float), _ptr(lm, C.c_float), float(src),
                                              float(srt), _ptr(nf, C.c_float), B, n, P(th), P(st), int(qso["ref"]), P(dt), P(sd),
                                              P(out["chi2_img"]), P(out["chi2_tmd"]), P(out["theta_pre"]),
                                              P(out["dt_pre"]), P(out["beta"]), P(out["last_step"]))
    if rc != 0:
        raise ValueError("oracle: bad quasar arguments")
    return out


# ------------------------------------------------------------------------------------------------
# JAM_sph (oracle/jam_sph_oracle.c)
# ------------------------------------------------------------------------------------------------
def jam_sph_intrinsic(r, theta, sig_k, q_k, nu0_k, beta_k, sig_j, q_j, mass_j, rcut, tau, wtau, un, uw):
    """(nu v_r^2, nu v_theta^2, nu v_phi^2, nu) at one point (r [pc], theta), intrinsic tables in pc / Msun."""
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    sig_k, q_k, nu0_k, beta_k, sig_j, q_j, mass_j, tau, wtau, un, uw = map(
        f, (sig_k, q_k, nu0_k, beta_k, sig_j, q_j, mass_j, tau, wtau, un, uw))
    out = np.zeros(4)
    P = lambda a: _ptr(a, C.c_double)
    lib().glad_oracle_jam_sph_intrinsic(float(r), float(theta), sig_k.size, P(sig_k), P(q_k), P(nu0_k), P(beta_k),
                                        sig_j.size, P(sig_j), P(q_j), P(mass_j), float(rcut), tau.size, P(tau), P(wtau),
                                        un.size, P(un), P(uw), P(out))
    return out


def jam_sph_los(xp, yp, inc, sig_k, q_k, nu0_k, rgrid, thgrid, ratios, rcut, zeta, wz) -> float:
    """int nu v_z'^2 dz' at one sky point (pc), ratios [3,nr,nth] on the polar grid (pc, rad)."""
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    sig_k, q_k, nu0_k, rgrid, thgrid, ratios, zeta, wz = map(f, (sig_k, q_k, nu0_k, rgrid, thgrid, ratios, zeta, wz))
    P = lambda a: _ptr(a, C.c_double)
    return float(lib().glad_oracle_jam_sph_los(float(xp), float(yp), float(inc), sig_k.size, P(sig_k), P(q_k), P(nu0_k),
                                               rgrid.size, P(rgrid), thgrid.size, P(thgrid), P(ratios), float(rcut),
                                               zeta.size, P(zeta), P(wz)))


def jam_sph_vrms_batch(dyn, lum_mge, mass_mge, beta, kin, sph, want_maps=False):
    """kin as jam_vrms_batch (u_nodes unused); sph = dict(rgrid, thgrid, tau, wtau, un, uw, zeta, wz); beta = beta_ani.
    Returns dict(vrms, chi2, flags[, v2map, moments [B,3,nr,nth]])."""
    dyn = _f32(dyn).reshape(-1, NDYN)
    B = dyn.shape[0]
    lum, mass, beta = _f32(lum_mge), _f32(mass_mge), _f32(beta)
    n_lum, n_mass = lum.shape[-2], mass.shape[-2]
    lum_stride = 0 if lum.ndim == 2 else n_lum * 3
    mass_stride = 0 if mass.ndim == 2 else n_mass * 3
    per_g = 1 if beta.ndim == 2 else 0
    xs, ys = _f32(kin["xs"]), _f32(kin["ys"])
    nx, ny = xs.size, ys.size
    bin_id = np.ascontiguousarray(kin["bin_id"], dtype=np.int32)
    nbins = int(kin["nbins"])
    kern = _f32(kin["kernel"])
    vo, vi = _f32(kin.get("vrms_obs")), _f32(kin.get("vrms_ivar"))
    a = {k: _f32(sph[k]) for k in ("rgrid", "thgrid", "tau", "wtau", "un", "uw", "zeta", "wz")}
    nr, nth = a["rgrid"].size, a["thgrid"].size
    vrms = np.empty((B, nbins), np.float64)
    chi2 = np.empty(B, np.float64)
    flags = np.zeros(B, np.int32)
    v2map = np.empty((B, ny, nx), np.float64) if want_maps else None
    mom = np.empty((B, 3, nr, nth), np.float64) if want_maps else None
    F = C.c_float
    rc = lib().glad_oracle_jam_sph_vrms_batch(
        _ptr(dyn, F), B, _ptr(lum, F), n_lum, lum_stride, _ptr(mass, F), n_mass, mass_stride, _ptr(beta, F), per_g, nx, ny,
        _ptr(xs, F), _ptr(ys, F), _ptr(bin_id, C.c_int32), nbins, _ptr(kern, F), kern.shape[0], _ptr(vo, F), _ptr(vi, F),
        nr, _ptr(a["rgrid"], F), nth, _ptr(a["thgrid"], F), a["tau"].size, _ptr(a["tau"], F), _ptr(a["wtau"], F),
        a["un"].size, _ptr(a["un"], F), _ptr(a["uw"], F), a["zeta"].size, _ptr(a["zeta"], F), _ptr(a["wz"], F),
        _ptr(vrms, C.c_double), _ptr(chi2, C.c_double), _ptr(v2map, C.c_double), _ptr(mom, C.c_double), _ptr(flags, C.c_int32))
    if rc != 0:
        raise ValueError("oracle: bad jam_sph arguments")
    out = {"vrms": vrms, "chi2": chi2, "flags": flags}
    if want_maps:
        out["v2map"], out["moments"] = v2map, mom
    return out


# ------------------------------------------------------------------------------------------------
# eNFW halo through core-steep ellipsoids (mass part; Appendix A)
# ------------------------------------------------------------------------------------------------
def set_cse_table(A, s):
    """The (A_i, s_i) table of Eq. A.3 -- an input of the method (workloads.cse_table()); also used by MGE profile kind 3."""
    A, s = np.ascontiguousarray(A, dtype=np.float64), np.ascontiguousarray(s, dtype=np.float64)
    assert A.size == s.size
    if lib().glad_oracle_set_cse_table(int(A.size), _ptr(A, C.c_double), _ptr(s, C.c_double)) != 0:
        raise ValueError("oracle: CSE table too long")


def nfw_kappa(u) -> float:
    """Eq. A.1 with rho_s = 1."""
    return float(lib().glad_oracle_nfw_kappa(float(u)))


def enfw(nf, dx, dy):
    """dict(kappa, ax, ay, h [3] = (xx, xy, yy), psi) of the halo nf = {rho_s, r_s, q, phi} at offset (dx, dy) from its centre."""
    nf = np.ascontiguousarray(nf, dtype=np.float64)
    k, ax, ay, ps = C.c_double(), C.c_double(), C.c_double(), C.c_double()
    h = np.empty(3)
    lib().glad_oracle_enfw(_ptr(nf, C.c_double), float(dx), float(dy), C.byref(k), C.byref(ax), C.byref(ay), _ptr(h, C.c_double), C.byref(ps))
    return {"kappa": k.value, "ax": ax.value, "ay": ay.value, "h": h, "psi": ps.value}
