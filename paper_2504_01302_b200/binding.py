"""Thin ctypes binding of libglad (include/glad.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels.  PyTorch supplies device memory and the stream, nothing else.
There is no fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from .build import LIB, build

NLENS, NDYN, NPROF = 26, 4, 4
PROFILE_SERSIC, PROFILE_EPL, PROFILE_CHAMELEON, PROFILE_NFW_CSE = 0, 1, 2, 3
LENS_NOALLOC_MAX_B = 4096          # GLAD_LENS_NOALLOC_MAX_B
LIGHT_SERSIC, LIGHT_CHAMELEON = 0, 1
FLAG_LENS_INVALID, FLAG_DYN_INVALID, FLAG_BIN_INVALID = 1, 2, 4
FLAG_PIXSRC_NOT_PD = 8

_lib = None
EXPORTS = ["glad_create", "glad_destroy", "glad_last_error", "glad_version", "glad_set_image_data",
           "glad_set_kin_data", "glad_lens_image_batch", "glad_jam_vrms_batch", "glad_joint_loglike_batch",
           "glad_joint_loglike_host", "glad_bh_theta2", "glad_launch_count", "glad_profile_enable",
           "glad_profile_read", "glad_mge1d_batch", "glad_joint_loglike_model_batch", "glad_set_overlap", "glad_set_light_profiles",
           "glad_set_quasar_data", "glad_quasar_chi2_batch", "glad_joint_loglike_full_batch", "glad_set_mass_sheet",
           "glad_pixsrc_evidence_batch", "glad_set_jam_options", "glad_set_jam_sph_rules", "glad_jam_sph_vrms_batch", "glad_set_enfw", "glad_pixsrc_lambda_opt_batch",
           "glad_lens_image_noalloc"]


class GladError(RuntimeError):
    pass


class ImageGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("supersample", C.c_int),
                ("pix", C.c_float), ("x0", C.c_float), ("y0", C.c_float)]


class SkyGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("d_xs", C.c_void_p), ("d_ys", C.c_void_p)]


def load(rebuild: bool = False):
    """Load libglad.so (building it in-tree if it is missing or stale and nvcc is present)."""
    global _lib
    if _lib is not None and not rebuild:
        return _lib
    if rebuild or not os.path.exists(LIB):
        build(force=rebuild)
    if not os.path.exists(LIB):
        raise GladError(f"libglad.so not found at {LIB}: run __graft_entry__.build()")
    L = C.CDLL(LIB)
    vp, i, l = C.c_void_p, C.c_int, C.c_long
    L.glad_create.restype = i
    L.glad_create.argtypes = [C.POINTER(vp), i, vp]
    L.glad_destroy.restype = None
    L.glad_destroy.argtypes = [vp]
    L.glad_last_error.restype = C.c_char_p
    L.glad_last_error.argtypes = [vp]
    L.glad_version.restype = C.c_char_p
    L.glad_set_image_data.restype = i
    L.glad_set_image_data.argtypes = [vp, C.POINTER(ImageGrid), vp, vp, vp, i]
    L.glad_set_kin_data.restype = i
    L.glad_set_kin_data.argtypes = [vp, C.POINTER(SkyGrid), vp, i, vp, i, vp, vp, vp, vp, i]
    L.glad_lens_image_batch.restype = i
    L.glad_lens_image_batch.argtypes = [vp, vp, i, vp, vp, vp]
    L.glad_lens_image_noalloc.restype = i
    L.glad_lens_image_noalloc.argtypes = [vp, vp, i, vp, vp, vp]
    L.glad_jam_vrms_batch.restype = i
    L.glad_jam_vrms_batch.argtypes = [vp, vp, i, vp, i, l, vp, i, l, vp, i, vp, vp, vp, vp]
    L.glad_joint_loglike_batch.restype = i
    L.glad_joint_loglike_batch.argtypes = [vp, vp, vp, i, vp, i, l, vp, i, l, vp, i, vp, vp, vp, vp]
    L.glad_joint_loglike_host.restype = i
    L.glad_joint_loglike_host.argtypes = [vp, vp, vp, i, vp, i, l, vp, i, l, vp, i, vp, vp, vp, vp]
    L.glad_bh_theta2.restype = C.c_double
    L.glad_bh_theta2.argtypes = [C.c_double] * 3
    L.glad_profile_enable.restype = i
    L.glad_profile_enable.argtypes = [vp, i]
    L.glad_profile_read.restype = i
    L.glad_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_long)]
    L.glad_mge1d_batch.restype = i
    L.glad_mge1d_batch.argtypes = [vp, i, vp, i, i, C.c_float, C.c_float, i, vp]
    L.glad_joint_loglike_model_batch.restype = i
    L.glad_joint_loglike_model_batch.argtypes = [vp, vp, vp, vp, C.c_float, i, i, C.c_float, C.c_float, i, C.c_float,
                                                 C.c_float, vp, i, vp, vp, vp, vp, vp, vp]
    L.glad_set_light_profiles.restype = i
    L.glad_set_light_profiles.argtypes = [vp, i, i, i]
    L.glad_set_overlap.restype = i
    L.glad_set_overlap.argtypes = [vp, i]
    dp = C.POINTER(C.c_double)
    L.glad_set_quasar_data.restype = i
    L.glad_set_quasar_data.argtypes = [vp, i, dp, dp, i, dp, dp]
    L.glad_quasar_chi2_batch.restype = i
    L.glad_quasar_chi2_batch.argtypes = [vp, vp, vp, i, vp, vp, vp, vp, vp]
    L.glad_joint_loglike_full_batch.restype = i
    L.glad_joint_loglike_full_batch.argtypes = [vp, vp, vp, vp, C.c_float, i, i, C.c_float, C.c_float, i, C.c_float,
                                                C.c_float, vp, i, vp, vp, vp, vp, vp, vp]
    L.glad_set_mass_sheet.restype = i
    L.glad_set_mass_sheet.argtypes = [vp, vp, i, C.c_float, C.c_float, i, C.c_float, C.c_float]
    L.glad_pixsrc_evidence_batch.restype = i
    L.glad_pixsrc_evidence_batch.argtypes = [vp, vp, vp, vp, i, i, i, i, vp, vp, vp, vp, vp, vp]
    L.glad_set_jam_sph_rules.restype = i
    L.glad_set_jam_sph_rules.argtypes = [vp, vp, i, vp, i, vp, vp, i, vp, vp, i, vp, vp, i]
    L.glad_jam_sph_vrms_batch.restype = i
    L.glad_jam_sph_vrms_batch.argtypes = [vp, vp, i, vp, i, l, vp, i, l, vp, i, vp, vp, vp, vp, vp]
    L.glad_pixsrc_lambda_opt_batch.restype = i
    L.glad_pixsrc_lambda_opt_batch.argtypes = [vp, vp, vp, C.c_float, C.c_float, i, i, i, i, vp, vp, vp, vp, vp, vp, vp]
    L.glad_set_enfw.restype = i
    L.glad_set_enfw.argtypes = [vp, vp, i, i, C.POINTER(C.c_double), C.POINTER(C.c_double), i, C.c_float, C.c_float]
    L.glad_set_jam_options.restype = i
    L.glad_set_jam_options.argtypes = [vp, i, i, i, i]
    L.glad_launch_count.restype = l
    L.glad_launch_count.argtypes = [vp]
    _lib = L
    return L


def bh_theta2(mbh_msun: float, ddt_mpc: float, z_d: float) -> float:
    return float(load().glad_bh_theta2(mbh_msun, ddt_mpc, z_d))


def _dev(t, dtype, device):
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        t = torch.from_numpy(np.ascontiguousarray(t))
    return t.to(device=device, dtype=dtype).contiguous()


def _p(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Glad:
    """One libglad context bound to torch's current stream on `device`."""

    DEFAULT_JAM_PATH = "auto"      # tests flip this class attribute to run every case on the FP32 SIMT form of row a6 as well

    def __init__(self, device: int | str = 0):
        if not torch.cuda.is_available():
            raise GladError("libglad needs a CUDA device (sm_100); there is no CPU path")
        self.device = torch.device("cuda", device) if isinstance(device, int) else torch.device(device)
        self.lib = load()
        self._keep = {}
        ctx = C.c_void_p()
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream()
            st = self.lib.glad_create(C.byref(ctx), self.device.index or 0, C.c_void_p(self.stream.cuda_stream))
        if st != 0:
            raise GladError(f"glad_create failed with status {st} (device is not sm_100?)")
        self.ctx = ctx
        if self.DEFAULT_JAM_PATH != "auto":
            self.set_jam_options(path=self.DEFAULT_JAM_PATH)
        self.n_halo_rows = 0
        self.image_shape = None
        self.sky_shape = None
        self.nbins = 0

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.glad_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != 0:
            raise GladError(f"libglad status {st}: {self.lib.glad_last_error(self.ctx).decode()}")

    @property
    def launch_count(self) -> int:
        return int(self.lib.glad_launch_count(self.ctx))

    KERNELS = ("lens_prep", "lens_image", "jam_prep", "jam_quad", "jam_post", "joint", "mge", "quasar",
               "pixsrc_map", "pixsrc_blur", "pixsrc_syrk", "pixsrc_rhs", "pixsrc_chol", "pixsrc_model", "jam_sph", "jam_sph_los")

    def set_light_profiles(self, source=0, lens1=0, lens2=0):
        """0 = Sersic, 1 = Chameleon (Eq. 47) per light component, for the batch calls that follow."""
        self._check(self.lib.glad_set_light_profiles(self.ctx, int(source), int(lens1), int(lens2)))

    def set_jam_options(self, path: str = "auto", terms: int = 0, flush: int = 0, slices: int = 0):
        """Row a6 options: path "auto" (tcgen05 where the grid fits) or "simt"; bf16 terms 2/3; 0 = default."""
        self._check(self.lib.glad_set_jam_options(self.ctx, {"auto": 0, "tc": 0, "simt": 1}[path], int(terms), int(flush), int(slices)))

    def set_enfw(self, enfw, cse_A=None, cse_s=None, n_gauss=16, sigma_range=(0.05, 300.0)):
        """eNFW halo per vector: enfw [n,4] = {rho_s, r_s, q, phi} (None switches it off); (cse_A, cse_s) = the CSE table."""
        if enfw is None:
            self._check(self.lib.glad_set_enfw(self.ctx, None, 0, 0, None, None, 0, 0.0, 0.0))
            self._keep.pop("enfw", None)
            self.n_halo_rows = 0
            return
        t = _dev(enfw, torch.float32, self.device).reshape(-1, 4)
        A = np.ascontiguousarray(cse_A, dtype=np.float64)
        s = np.ascontiguousarray(cse_s, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        self._check(self.lib.glad_set_enfw(self.ctx, _p(t), int(t.shape[0]), int(A.size), A.ctypes.data_as(dp), s.ctypes.data_as(dp),
                                           int(n_gauss), float(sigma_range[0]), float(sigma_range[1])))
        self._keep["enfw"] = t
        self.n_halo_rows = int(n_gauss)

    def set_overlap(self, on: bool):
        self._check(self.lib.glad_set_overlap(self.ctx, 1 if on else 0))

    def profile_enable(self, on: bool = True):
        self._check(self.lib.glad_profile_enable(self.ctx, 1 if on else 0))

    def profile_read(self) -> dict:
        """{kernel: (total ms, launches)} since the last read (synchronises the stream)."""
        ms = (C.c_double * len(self.KERNELS))()
        cnt = (C.c_long * len(self.KERNELS))()
        self._check(self.lib.glad_profile_read(self.ctx, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.KERNELS)}

    # ---- static data -------------------------------------------------------------------------
    def set_image_data(self, grid: dict, psf, data=None, ivar=None):
        f = torch.float32
        k = {"psf": _dev(psf, f, self.device), "data": _dev(data, f, self.device), "ivar": _dev(ivar, f, self.device)}
        g = ImageGrid(int(grid["nx"]), int(grid["ny"]), int(grid["supersample"]), float(grid["pix"]),
                      float(grid["x0"]), float(grid["y0"]))
        self._check(self.lib.glad_set_image_data(self.ctx, C.byref(g), _p(k["data"]), _p(k["ivar"]), _p(k["psf"]),
                                                 int(k["psf"].shape[0])))
        self._keep["image"] = k
        self.image_shape = (g.ny, g.nx)

    def set_kin_data(self, kin: dict):
        f = torch.float32
        k = {n: _dev(kin.get(n), f, self.device) for n in ("xs", "ys", "kernel", "vrms_obs", "vrms_ivar", "u_nodes", "u_weights")}
        k["bin_id"] = _dev(kin["bin_id"], torch.int32, self.device)
        g = SkyGrid(int(k["xs"].numel()), int(k["ys"].numel()), k["xs"].data_ptr(), k["ys"].data_ptr())
        self._check(self.lib.glad_set_kin_data(self.ctx, C.byref(g), _p(k["bin_id"]), int(kin["nbins"]), _p(k["kernel"]),
                                               int(k["kernel"].shape[0]), _p(k["vrms_obs"]), _p(k["vrms_ivar"]),
                                               _p(k["u_nodes"]), _p(k["u_weights"]), int(k["u_nodes"].numel())))
        self._keep["kin"] = k
        self.sky_shape = (g.ny, g.nx)
        self.nbins = int(kin["nbins"])

    # ---- batch calls (device tensors in, device tensors out; enqueue only) --------------------
    def lens_image_batch(self, lens_params, want_images=True, want_chi2=True, out=None):
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        B = p.shape[0]
        out = out or {}
        img = out.get("images") if want_images else None
        if want_images and img is None:
            img = torch.empty((B,) + (self.image_shape or (0, 0)), dtype=torch.float32, device=self.device)
        chi2 = (out.get("chi2") if out.get("chi2") is not None else torch.empty(B, dtype=torch.float32, device=self.device)) if want_chi2 else None
        flags = out.get("flags") if out.get("flags") is not None else torch.empty(B, dtype=torch.int32, device=self.device)
        self._check(self.lib.glad_lens_image_batch(self.ctx, _p(p), B, _p(img), _p(chi2), _p(flags)))
        return {"images": img, "chi2": chi2, "flags": flags}

    def lens_image_noalloc(self, lens_params, out):
        """glad_lens_image_noalloc: lens_params a device float32 tensor [B, NLENS], out = dict(images, chi2, flags) of preallocated
        device tensors (any may be None): nothing is allocated here or in the library; B <= LENS_NOALLOC_MAX_B."""
        B = lens_params.shape[0]
        self._check(self.lib.glad_lens_image_noalloc(self.ctx, _p(lens_params), B, _p(out.get("images")), _p(out.get("chi2")),
                                                     _p(out.get("flags"))))
        return out

    def _tables(self, lum_mge, mass_mge, beta):
        f = torch.float32
        lum, mass, beta = _dev(lum_mge, f, self.device), _dev(mass_mge, f, self.device), _dev(beta, f, self.device)
        n_lum, n_mass = lum.shape[-2], mass.shape[-2]
        ls = 0 if lum.dim() == 2 else n_lum * 3
        ms = 0 if mass.dim() == 2 else n_mass * 3
        return lum, n_lum, ls, mass, n_mass, ms, beta, (1 if beta.dim() == 2 else 0)

    def jam_vrms_batch(self, dyn_params, lum_mge, mass_mge, beta, want_chi2=True, want_map=False):
        d = _dev(dyn_params, torch.float32, self.device).reshape(-1, NDYN)
        B = d.shape[0]
        lum, nl, ls, mass, nm, ms, bt, pg = self._tables(lum_mge, mass_mge, beta)
        vrms = torch.empty((B, self.nbins), dtype=torch.float32, device=self.device)
        chi2 = torch.empty(B, dtype=torch.float32, device=self.device) if want_chi2 else None
        v2map = torch.empty((B,) + (self.sky_shape or (0, 0)), dtype=torch.float32, device=self.device) if want_map else None
        flags = torch.empty(B, dtype=torch.int32, device=self.device)
        self._check(self.lib.glad_jam_vrms_batch(self.ctx, _p(d), B, _p(lum), nl, ls, _p(mass) if nm else None, nm, ms,
                                                 _p(bt), pg, _p(vrms), _p(chi2), _p(v2map), _p(flags)))
        return {"vrms": vrms, "chi2": chi2, "v2map": v2map, "flags": flags}

    def set_jam_sph_rules(self, sph: dict):
        """sph = dict(rgrid, thgrid, tau, wtau, un, uw, zeta, wz): polar grid and the three rules of the JAM_sph path."""
        k = {n: _dev(sph[n], torch.float32, self.device) for n in ("rgrid", "thgrid", "tau", "wtau", "un", "uw", "zeta", "wz")}
        self._check(self.lib.glad_set_jam_sph_rules(self.ctx, _p(k["rgrid"]), int(k["rgrid"].numel()), _p(k["thgrid"]),
                                                    int(k["thgrid"].numel()), _p(k["tau"]), _p(k["wtau"]), int(k["tau"].numel()),
                                                    _p(k["un"]), _p(k["uw"]), int(k["un"].numel()), _p(k["zeta"]), _p(k["wz"]),
                                                    int(k["zeta"].numel())))
        self._keep["sph"] = k
        self.sph_shape = (int(k["rgrid"].numel()), int(k["thgrid"].numel()))

    def jam_sph_vrms_batch(self, dyn_params, lum_mge, mass_mge, beta, want_chi2=True, want_map=False, want_moments=False):
        """JAM_sph (the paper's dynamics): beta = beta_ani; outputs as jam_vrms_batch plus moments [B,3,nr,nth]."""
        d = _dev(dyn_params, torch.float32, self.device).reshape(-1, NDYN)
        B = d.shape[0]
        lum, nl, ls, mass, nm, ms, bt, pg = self._tables(lum_mge, mass_mge, beta)
        vrms = torch.empty((B, self.nbins), dtype=torch.float32, device=self.device)
        chi2 = torch.empty(B, dtype=torch.float32, device=self.device) if want_chi2 else None
        v2map = torch.empty((B,) + (self.sky_shape or (0, 0)), dtype=torch.float32, device=self.device) if want_map else None
        mom = torch.empty((B, 3) + self.sph_shape, dtype=torch.float32, device=self.device) if want_moments else None
        flags = torch.empty(B, dtype=torch.int32, device=self.device)
        self._check(self.lib.glad_jam_sph_vrms_batch(self.ctx, _p(d), B, _p(lum), nl, ls, _p(mass) if nm else None, nm, ms,
                                                     _p(bt), pg, _p(vrms), _p(chi2), _p(v2map), _p(mom), _p(flags)))
        return {"vrms": vrms, "chi2": chi2, "v2map": v2map, "moments": mom, "flags": flags}

    def joint_loglike_batch(self, lens_params, dyn_params, lum_mge, mass_mge, beta, out=None):
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        d = _dev(dyn_params, torch.float32, self.device).reshape(-1, NDYN)
        B = p.shape[0]
        if d.shape[0] != B:
            raise GladError("lens and dyn batches differ")
        lum, nl, ls, mass, nm, ms, bt, pg = self._tables(lum_mge, mass_mge, beta)
        out = out or {}
        mk = lambda n, dt: out.get(n) if out.get(n) is not None else torch.empty(B, dtype=dt, device=self.device)
        ll, c2l, c2d, fl = mk("loglike", torch.float32), mk("chi2_lens", torch.float32), mk("chi2_dyn", torch.float32), mk("flags", torch.int32)
        self._check(self.lib.glad_joint_loglike_batch(self.ctx, _p(p), _p(d), B, _p(lum), nl, ls, _p(mass) if nm else None,
                                                      nm, ms, _p(bt), pg, _p(ll), _p(c2l), _p(c2d), _p(fl)))
        return {"loglike": ll, "chi2_lens": c2l, "chi2_dyn": c2d, "flags": fl}

    def joint_loglike_host(self, lens_params, dyn_params, lum_mge, mass_mge, beta, loglike_out):
        """Host (CPU, ideally pinned) tensors in, host tensor out; copies + sync inside the C call."""
        for t in (lens_params, dyn_params, lum_mge, mass_mge, beta, loglike_out):
            if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
                raise GladError("joint_loglike_host wants contiguous float32 CPU tensors")
        B = lens_params.shape[0]
        nl, nm = lum_mge.shape[-2], mass_mge.shape[-2]
        ls = 0 if lum_mge.dim() == 2 else nl * 3
        ms = 0 if mass_mge.dim() == 2 else nm * 3
        self._check(self.lib.glad_joint_loglike_host(self.ctx, _p(lens_params), _p(dyn_params), B, _p(lum_mge), nl, ls,
                                                     _p(mass_mge) if nm else None, nm, ms, _p(beta), 1 if beta.dim() == 2 else 0,
                                                     _p(loglike_out), None, None, None))
        return loglike_out

    # ---- on-device 1-D MGE and the self-consistent joint model ----------------
    def mge1d_batch(self, kind, prof, n_gauss, sigma_lo, sigma_hi, euler_order=0):
        pr = _dev(prof, torch.float32, self.device).reshape(-1, NPROF)
        B = pr.shape[0]
        mge = torch.empty((B, int(n_gauss), 3), dtype=torch.float32, device=self.device)
        self._check(self.lib.glad_mge1d_batch(self.ctx, int(kind), _p(pr), B, int(n_gauss), float(sigma_lo), float(sigma_hi),
                                              int(euler_order), _p(mge)))
        return mge

    def joint_loglike_model_batch(self, lens_params, dyn_params, ddt, z_d, n_lum, lum_range, n_mass, mass_range, beta,
                                  want_tables=False, out=None):
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        d = _dev(dyn_params, torch.float32, self.device).reshape(-1, NDYN)
        dt = _dev(ddt, torch.float32, self.device).reshape(-1)
        bt = _dev(beta, torch.float32, self.device)
        B = p.shape[0]
        if d.shape[0] != B or dt.shape[0] != B:
            raise GladError("lens, dyn and ddt batches differ")
        out = out or {}
        mk = lambda n, ty: out.get(n) if out.get(n) is not None else torch.empty(B, dtype=ty, device=self.device)
        ll, c2l, c2d, fl = mk("loglike", torch.float32), mk("chi2_lens", torch.float32), mk("chi2_dyn", torch.float32), mk("flags", torch.int32)
        lum = torch.empty((B, int(n_lum), 3), dtype=torch.float32, device=self.device) if want_tables else None
        n_tot = int(n_mass) + (self._n_sheet if "lambda" in self._keep else 0) + (self.n_halo_rows if "enfw" in self._keep else 0)
        mass = torch.empty((B, n_tot, 3), dtype=torch.float32, device=self.device) if want_tables else None
        self._check(self.lib.glad_joint_loglike_model_batch(
            self.ctx, _p(p), _p(d), _p(dt), float(z_d), B, int(n_lum), float(lum_range[0]), float(lum_range[1]), int(n_mass),
            float(mass_range[0]), float(mass_range[1]), _p(bt), 1 if bt.dim() == 2 else 0, _p(ll), _p(c2l), _p(c2d), _p(fl),
            _p(lum), _p(mass)))
        return {"loglike": ll, "chi2_lens": c2l, "chi2_dyn": c2d, "flags": fl, "lum_mge": lum, "mass_mge": mass}

    # ---- internal mass sheet (Eq. 6, 50) -------------------------------------------------------
    def set_mass_sheet(self, lam, r_core=45.0, r_tr=45.09, n_sheet=8, sigma_lo=6.0, sigma_hi=2000.0):
        """lam [B] (kept alive here) switches the sheet on for the batch calls that follow; None switches it off."""
        if lam is None:
            self._keep.pop("lambda", None)
            self._check(self.lib.glad_set_mass_sheet(self.ctx, None, 0, 0.0, 0.0, 0, 0.0, 0.0))
            return
        t = _dev(lam, torch.float32, self.device).reshape(-1)
        self._check(self.lib.glad_set_mass_sheet(self.ctx, _p(t), int(t.numel()), float(r_core), float(r_tr), int(n_sheet), float(sigma_lo), float(sigma_hi)))
        self._keep["lambda"] = t
        self._n_sheet = int(n_sheet)

    # ---- quasar terms (Eq. 35-36) --------------------------------------------------------------
    def set_quasar_data(self, qso: dict | None):
        """qso = dict(theta [n_img,2], sigma_theta [n_img], ref, dt_obs [n_img] days, sigma_dt [n_img]) host arrays; None clears."""
        if qso is None:
            self._check(self.lib.glad_set_quasar_data(self.ctx, 0, None, None, 0, None, None))
            self.n_img = 0
            return
        f = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        th, st, dt, sd = f(qso["theta"]), f(qso["sigma_theta"]), f(qso.get("dt_obs")), f(qso.get("sigma_dt"))
        n = th.size // 2
        if st.size != n or (dt is not None and (dt.size != n or sd is None or sd.size != n)):
            raise GladError("quasar arrays differ in length")
        P = lambda a: None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))
        self._check(self.lib.glad_set_quasar_data(self.ctx, n, P(th), P(st), int(qso["ref"]), P(dt), P(sd)))
        self.n_img = n

    def quasar_chi2_batch(self, lens_params, ddt, want_details=True):
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        dt = _dev(ddt, torch.float32, self.device).reshape(-1)
        B = p.shape[0]
        if dt.shape[0] != B:
            raise GladError("lens and ddt batches differ")
        n = getattr(self, "n_img", 0)
        c2i = torch.empty(B, dtype=torch.float32, device=self.device)
        c2t = torch.empty(B, dtype=torch.float32, device=self.device)
        mk = lambda *shape: torch.empty(shape, dtype=torch.float64, device=self.device) if want_details else None
        tp, dp, bb = mk(B, n, 2), mk(B, n), mk(B, 2)
        self._check(self.lib.glad_quasar_chi2_batch(self.ctx, _p(p), _p(dt), B, _p(c2i), _p(c2t), _p(tp), _p(dp), _p(bb)))
        return {"chi2_img": c2i, "chi2_tmd": c2t, "theta_pre": tp, "dt_pre": dp, "beta": bb}

    def pixsrc_evidence_batch(self, lens_params, src_grids, lam, nsx, nsy, want_source=True, want_model=True, scratch_mib=0):
        """Pixelated-source evidence (Eq. 37-43): lens [B,26], src_grids [B,3] = {x_s0, y_s0, p_s}, lam [B]."""
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        sg = _dev(src_grids, torch.float32, self.device).reshape(-1, 3)
        lm = _dev(lam, torch.float32, self.device).reshape(-1)
        B = p.shape[0]
        if sg.shape[0] != B or lm.shape[0] != B:
            raise GladError("lens, source-grid and lambda batches differ")
        if getattr(self, "image_shape", None) is None:
            raise GladError("set_image_data has not been called")
        f32 = lambda *shape: torch.empty(shape, dtype=torch.float32, device=self.device)
        ev, c2, rg = f32(B), f32(B), f32(B)
        fl = torch.empty(B, dtype=torch.int32, device=self.device)
        s = f32(B, int(nsy), int(nsx)) if want_source else None
        m = f32(B, *self.image_shape) if want_model else None
        self._check(self.lib.glad_pixsrc_evidence_batch(self.ctx, _p(p), _p(sg), _p(lm), int(nsx), int(nsy), B, int(scratch_mib),
                                                        _p(ev), _p(c2), _p(rg), _p(s), _p(m), _p(fl)))
        return {"logev": ev, "chi2": c2, "reg": rg, "s_mp": s, "model": m, "flags": fl}

    def pixsrc_lambda_opt_batch(self, lens_params, src_grids, lam_range, nsx, nsy, want_source=True, want_model=True, scratch_mib=0):
        """Eq. 43: lambda_hat on [lam_range] per vector and the evidence (and everything pixsrc_evidence_batch returns) at it."""
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        sg = _dev(src_grids, torch.float32, self.device).reshape(-1, 3)
        B = p.shape[0]
        if sg.shape[0] != B:
            raise GladError("lens and source-grid batches differ")
        if getattr(self, "image_shape", None) is None:
            raise GladError("set_image_data has not been called")
        f32 = lambda *shape: torch.empty(shape, dtype=torch.float32, device=self.device)
        lh, ev, c2, rg = f32(B), f32(B), f32(B), f32(B)
        fl = torch.empty(B, dtype=torch.int32, device=self.device)
        s = f32(B, int(nsy), int(nsx)) if want_source else None
        m = f32(B, *self.image_shape) if want_model else None
        self._check(self.lib.glad_pixsrc_lambda_opt_batch(self.ctx, _p(p), _p(sg), float(lam_range[0]), float(lam_range[1]), int(nsx), int(nsy),
                                                          B, int(scratch_mib), _p(lh), _p(ev), _p(c2), _p(rg), _p(s), _p(m), _p(fl)))
        return {"lam_hat": lh, "logev": ev, "chi2": c2, "reg": rg, "s_mp": s, "model": m, "flags": fl}

    def joint_loglike_full_batch(self, lens_params, dyn_params, ddt, z_d, n_lum, lum_range, n_mass, mass_range, beta, out=None):
        p = _dev(lens_params, torch.float32, self.device).reshape(-1, NLENS)
        d = _dev(dyn_params, torch.float32, self.device).reshape(-1, NDYN)
        dt = _dev(ddt, torch.float32, self.device).reshape(-1)
        bt = _dev(beta, torch.float32, self.device)
        B = p.shape[0]
        if d.shape[0] != B or dt.shape[0] != B:
            raise GladError("lens, dyn and ddt batches differ")
        out = out or {}
        mk = lambda n, ty: out.get(n) if out.get(n) is not None else torch.empty(B, dtype=ty, device=self.device)
        ll, c2l, c2d, fl = mk("loglike", torch.float32), mk("chi2_lens", torch.float32), mk("chi2_dyn", torch.float32), mk("flags", torch.int32)
        c2i, c2t = mk("chi2_img", torch.float32), mk("chi2_tmd", torch.float32)
        self._check(self.lib.glad_joint_loglike_full_batch(
            self.ctx, _p(p), _p(d), _p(dt), float(z_d), B, int(n_lum), float(lum_range[0]), float(lum_range[1]), int(n_mass),
            float(mass_range[0]), float(mass_range[1]), _p(bt), 1 if bt.dim() == 2 else 0, _p(ll), _p(c2l), _p(c2d), _p(c2i),
            _p(c2t), _p(fl)))
        return {"loglike": ll, "chi2_lens": c2l, "chi2_dyn": c2d, "chi2_img": c2i, "chi2_tmd": c2t, "flags": fl}
