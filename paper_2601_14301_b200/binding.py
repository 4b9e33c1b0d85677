"""Thin ctypes binding of the C ABI in include/trimeg.h (argument marshalling only).

Same names as the C entry points.  PyTorch supplies device memory and the stream; every
step of the path runs in the library's CUDA kernels.  If libtrimeg.so is missing or cannot
be loaded this module raises: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtrimeg.so")

EXPORTS = (
    "trimeg_mesh_create", "trimeg_mesh_create_unstructured", "trimeg_mesh_locality_order", "trimeg_mesh_destroy", "trimeg_mesh_info", "trimeg_set_params",
    "trimeg_mesh_download_geom", "trimeg_equilibrium_upload", "trimeg_field_upload", "trimeg_field_upload_spline", "trimeg_field_download_coeffs",
    "trimeg_locate", "trimeg_gather", "trimeg_rhs", "trimeg_field_upload_aux", "trimeg_rhs_em", "trimeg_pullback", "trimeg_scatter", "trimeg_scatter_static", "trimeg_sort", "trimeg_compact",
    "trimeg_push", "trimeg_set_push_kernel", "trimeg_get_push_kernel", "trimeg_push_host", "trimeg_release_host_buffers", "trimeg_get_stats", "trimeg_reset_stats", "trimeg_get_tile_counters", "trimeg_measure_fp64_peak_operands",
    "trimeg_measure_fp64_peak", "trimeg_measure_gather_peak", "trimeg_strerror", "trimeg_version",
)

OK, ERR_INVALID_ARG, ERR_MESH, ERR_NO_FIELD, ERR_CUDA, ERR_ALLOC, ERR_UNSUPPORTED, ERR_CAPACITY = 0, -1, -2, -3, -4, -5, -6, -7
SCATTER_STATIC_BYTES = 16 * 1024 * 1024      # TRIMEG_SCATTER_STATIC_BYTES
# TRIMEG_PUSH_KERNEL_* of include/trimeg.h
FIELD_AS, FIELD_AH = 1, 2      # TRIMEG_FIELD_AS / _AH
PUSH_KERNEL_AUTO, PUSH_KERNEL_THREAD, PUSH_KERNEL_LANE, PUSH_KERNEL_WCACHE = -1, 0, 1, 2
PUSH_KERNELS = (PUSH_KERNEL_THREAD, PUSH_KERNEL_LANE, PUSH_KERNEL_WCACHE)


class TrimegError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} ({code})")
        self.code = code


class trimeg_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("R0", "a", "B0", "q0", "q2", "rho0", "qs_over_ms", "T", "kappa_n", "kappa_T")] + \
               [("eom_variant", C.c_int), ("weight_mode", C.c_int)]


class trimeg_markers(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("R", "Z", "phi", "vpar", "mu", "w", "cell")]


_lib = None


def load() -> C.CDLL:
    """Load libtrimeg.so (built by paper_2601_14301_b200.build).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build the CUDA library first "
            "(python -m paper_2601_14301_b200.build or __graft_entry__.build()). No CPU fallback exists.")
    L = C.CDLL(LIB_PATH)
    vp, sz, dbl, i32 = C.c_void_p, C.c_size_t, C.c_double, C.c_int
    dp = C.POINTER(C.c_double)
    L.trimeg_mesh_create.argtypes = [C.POINTER(vp), i32, i32, dp, dp, dp, C.POINTER(trimeg_params)]
    L.trimeg_mesh_create_unstructured.argtypes = [C.POINTER(vp), i32, dp, dp, i32, C.POINTER(C.c_int32), i32, i32, C.POINTER(trimeg_params)]
    L.trimeg_mesh_locality_order.argtypes = [i32, dp, dp, i32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.trimeg_mesh_destroy.argtypes = [vp]
    L.trimeg_mesh_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32)]
    L.trimeg_set_params.argtypes = [vp, C.POINTER(trimeg_params)]
    L.trimeg_mesh_download_geom.argtypes = [vp, vp, vp]
    L.trimeg_equilibrium_upload.argtypes = [vp, i32, i32, dbl, dbl, dbl, dbl, dp, i32, dbl, dbl, dp]
    L.trimeg_field_upload.argtypes = [vp, i32, C.POINTER(i32), vp, i32, vp]
    L.trimeg_field_upload_spline.argtypes = [vp, i32, vp, i32, vp]
    L.trimeg_field_download_coeffs.argtypes = [vp, vp, vp]
    L.trimeg_locate.argtypes = [vp, sz, vp, vp, vp, vp]
    L.trimeg_gather.argtypes = [vp, sz, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.trimeg_rhs.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, vp, vp, vp, vp, vp]
    L.trimeg_scatter.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, vp]
    L.trimeg_scatter_static.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, vp]
    L.trimeg_field_upload_aux.argtypes = [vp, i32, vp, i32, vp]
    L.trimeg_rhs_em.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, vp, vp, vp, vp, vp]
    L.trimeg_pullback.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp]
    L.trimeg_sort.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, vp]
    L.trimeg_compact.argtypes = [vp, C.POINTER(trimeg_markers), sz, vp, C.POINTER(sz), vp]
    L.trimeg_push.argtypes = [vp, C.POINTER(trimeg_markers), sz, dbl, i32, vp]
    L.trimeg_set_push_kernel.argtypes = [vp, i32]
    L.trimeg_push_host.argtypes = [vp, C.POINTER(trimeg_markers), sz, dbl, i32, i32]
    L.trimeg_release_host_buffers.argtypes = [vp]
    L.trimeg_get_stats.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.trimeg_reset_stats.argtypes = [vp]
    L.trimeg_get_tile_counters.argtypes = [vp, C.POINTER(C.c_int64)]
    L.trimeg_get_push_kernel.argtypes = [vp]
    L.trimeg_measure_fp64_peak.argtypes = [vp, dp]
    L.trimeg_measure_fp64_peak_operands.argtypes = [vp, i32, dp]
    L.trimeg_measure_gather_peak.argtypes = [vp, sz, i32, dp]
    L.trimeg_strerror.argtypes = [i32]
    L.trimeg_strerror.restype = C.c_char_p
    L.trimeg_version.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("trimeg_strerror", "trimeg_version"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def strerror(code: int) -> str:
    return load().trimeg_strerror(int(code)).decode()


def version() -> str:
    return load().trimeg_version().decode()


def _check(rc: int, what: str):
    if rc != OK:
        raise TrimegError(rc, what)


def _stream(stream) -> C.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _ptr(t: Optional[torch.Tensor], dtype, n: Optional[int] = None, device: str = "cuda") -> C.c_void_p:
    if t is None:
        return C.c_void_p(0)
    if t.dtype != dtype or not t.is_contiguous() or t.device.type != device:
        raise TypeError(f"expected contiguous {device} tensor of {dtype}, got {t.dtype} on {t.device}")
    if n is not None and t.numel() < n:
        raise ValueError(f"tensor too small: {t.numel()} < {n}")
    return C.c_void_p(t.data_ptr())


def _markers(m: Dict[str, torch.Tensor], n: int, device: str = "cuda") -> trimeg_markers:
    s = trimeg_markers()
    for k in ("R", "Z", "phi", "vpar", "mu", "w"):
        setattr(s, k, _ptr(m[k], torch.float64, n, device).value)
    s.cell = _ptr(m["cell"], torch.int32, n, device).value
    return s


class Context:
    """Owner of one trimeg_ctx (mesh + field tables on the current CUDA device)."""

    def __init__(self, n_r: int, n_theta: int, r_nodes, params: Dict, vert_R=None, vert_Z=None):
        import numpy as np
        self.L = load()
        self.h = C.c_void_p(0)
        r = np.ascontiguousarray(r_nodes, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        vR = vZ = None
        if vert_R is not None:
            vR = np.ascontiguousarray(vert_R, dtype=np.float64)
            vZ = np.ascontiguousarray(vert_Z, dtype=np.float64)
        p = trimeg_params(**params)
        rc = self.L.trimeg_mesh_create(C.byref(self.h), int(n_r), int(n_theta), r.ctypes.data_as(dp),
                                       vR.ctypes.data_as(dp) if vR is not None else None,
                                       vZ.ctypes.data_as(dp) if vZ is not None else None, C.byref(p))
        _check(rc, "trimeg_mesh_create")
        nv, nt = C.c_int(0), C.c_int(0)
        _check(self.L.trimeg_mesh_info(self.h, C.byref(nv), C.byref(nt)), "trimeg_mesh_info")
        self.n_r, self.n_theta, self.n_vert, self.n_tri = int(n_r), int(n_theta), nv.value, nt.value
        self.n_modes = 0
        self.n_phi = 0

    @classmethod
    def unstructured(cls, vert_R, vert_Z, tri, params: Dict, nbx: int = 0, nby: int = 0) -> "Context":
        """Row f4: any conforming triangulation (trimeg_mesh_create_unstructured)."""
        import numpy as np
        self = cls.__new__(cls)
        self.L = load()
        self.h = C.c_void_p(0)
        vR = np.ascontiguousarray(vert_R, dtype=np.float64)
        vZ = np.ascontiguousarray(vert_Z, dtype=np.float64)
        tr = np.ascontiguousarray(tri, dtype=np.int32)
        if tr.ndim != 2 or tr.shape[1] != 3 or vR.shape != vZ.shape:
            raise ValueError("tri must be [n_tri][3], vert_R and vert_Z of one length")
        dp = C.POINTER(C.c_double)
        p = trimeg_params(**params)
        rc = self.L.trimeg_mesh_create_unstructured(C.byref(self.h), int(vR.size), vR.ctypes.data_as(dp), vZ.ctypes.data_as(dp),
                                                    int(tr.shape[0]), tr.ctypes.data_as(C.POINTER(C.c_int32)), int(nbx), int(nby),
                                                    C.byref(p))
        _check(rc, "trimeg_mesh_create_unstructured")
        nv, nt = C.c_int(0), C.c_int(0)
        _check(self.L.trimeg_mesh_info(self.h, C.byref(nv), C.byref(nt)), "trimeg_mesh_info")
        self.n_r, self.n_theta, self.n_vert, self.n_tri = 0, 0, nv.value, nt.value
        self.n_modes = 0
        self.n_phi = 0
        return self

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.trimeg_mesh_destroy(self.h)
            self.h = C.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- mesh / field
    def set_params(self, params: Dict):
        p = trimeg_params(**params)
        _check(self.L.trimeg_set_params(self.h, C.byref(p)), "trimeg_set_params")

    def equilibrium_upload(self, tab: Optional[Dict]):
        """Row f4: tab = dict(C [nR][nZ], Ra, Za, hR, hZ, D [nF], pa, hp) of B-spline coefficients; None: analytic equilibrium."""
        import numpy as np
        dp = C.POINTER(C.c_double)
        if tab is None:
            _check(self.L.trimeg_equilibrium_upload(self.h, 0, 0, 0.0, 0.0, 0.0, 0.0, None, 0, 0.0, 0.0, None), "trimeg_equilibrium_upload")
            return
        Cc = np.ascontiguousarray(tab["C"], dtype=np.float64)
        D = np.ascontiguousarray(tab["D"], dtype=np.float64)
        _check(self.L.trimeg_equilibrium_upload(self.h, Cc.shape[0], Cc.shape[1], float(tab["Ra"]), float(tab["Za"]), float(tab["hR"]),
                                                float(tab["hZ"]), Cc.ctypes.data_as(dp), D.size, float(tab["pa"]), float(tab["hp"]),
                                                D.ctypes.data_as(dp)), "trimeg_equilibrium_upload")

    def mesh_download_geom(self, stream=None) -> torch.Tensor:
        out = torch.empty((self.n_tri, 6), dtype=torch.float64, device="cuda")
        _check(self.L.trimeg_mesh_download_geom(self.h, _ptr(out, torch.float64), _stream(stream)),
               "trimeg_mesh_download_geom")
        return out

    def field_upload(self, mode_n: Sequence[int], data: Optional[torch.Tensor], kind: int, stream=None):
        modes = (C.c_int * max(1, len(mode_n)))(*[int(n) for n in mode_n])
        M = len(mode_n)
        if M > 0:
            want = (M, self.n_vert, 6) if kind == 0 else (self.n_tri, M, 21)
            if tuple(data.shape) != want:
                raise ValueError(f"field data shape {tuple(data.shape)} != {want}")
        ptr = _ptr(data, torch.complex128) if M > 0 else C.c_void_p(0)
        _check(self.L.trimeg_field_upload(self.h, M, modes, ptr, int(kind), _stream(stream)), "trimeg_field_upload")
        self.n_modes = M
        self.n_phi = 0

    def field_upload_spline(self, data: torch.Tensor, kind: int, stream=None):
        """Row f3: real nodal DOFs [n_phi][n_vert][6] (kind 0) or coefficients [n_tri][n_phi][21] (kind 1)."""
        n_phi = int(data.shape[0] if kind == 0 else data.shape[1])
        want = (n_phi, self.n_vert, 6) if kind == 0 else (self.n_tri, n_phi, 21)
        if tuple(data.shape) != want:
            raise ValueError(f"field data shape {tuple(data.shape)} != {want}")
        _check(self.L.trimeg_field_upload_spline(self.h, n_phi, _ptr(data, torch.float64), int(kind), _stream(stream)),
               "trimeg_field_upload_spline")
        self.n_modes = 0
        self.n_phi = n_phi

    def field_download_coeffs(self, stream=None) -> torch.Tensor:
        if getattr(self, "n_phi", 0):
            out = torch.empty((self.n_tri, self.n_phi, 21), dtype=torch.float64, device="cuda")
            _check(self.L.trimeg_field_download_coeffs(self.h, _ptr(out, torch.float64), _stream(stream)),
                   "trimeg_field_download_coeffs")
            return out
        out = torch.empty((self.n_tri, self.n_modes, 21), dtype=torch.complex128, device="cuda")
        if self.n_modes:
            _check(self.L.trimeg_field_download_coeffs(self.h, _ptr(out, torch.complex128), _stream(stream)),
                   "trimeg_field_download_coeffs")
        return out

    # -- kernels
    def locate(self, R: torch.Tensor, Z: torch.Tensor, cell: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        n = R.numel()
        if cell is None:
            cell = torch.empty(n, dtype=torch.int32, device=R.device)
        _check(self.L.trimeg_locate(self.h, n, _ptr(R, torch.float64, n), _ptr(Z, torch.float64, n),
                                    _ptr(cell, torch.int32, n), _stream(stream)), "trimeg_locate")
        return cell

    def gather(self, R, Z, phi, cell_hint=None, want_dphi=True, stream=None, out=None) -> Dict[str, torch.Tensor]:
        """out: optional dict of preallocated outputs (dphi, dphi_dR, dphi_dZ[, dphi_dphi]) to write into."""
        n = R.numel()
        if out is None:
            out = {k: torch.empty(n, dtype=torch.float64, device=R.device) for k in ("dphi", "dphi_dR", "dphi_dZ")}
            fp = torch.empty(n, dtype=torch.float64, device=R.device) if want_dphi else None
        else:
            fp = out.get("dphi_dphi") if want_dphi else None
        _check(self.L.trimeg_gather(self.h, n, _ptr(R, torch.float64, n), _ptr(Z, torch.float64, n),
                                    _ptr(phi, torch.float64, n), _ptr(cell_hint, torch.int32, n),
                                    _ptr(out["dphi"], torch.float64), _ptr(out["dphi_dR"], torch.float64),
                                    _ptr(out["dphi_dZ"], torch.float64), _ptr(fp, torch.float64), _stream(stream)),
               "trimeg_gather")
        if want_dphi:
            out["dphi_dphi"] = fp
        return out

    def rhs(self, m: Dict[str, torch.Tensor], stream=None) -> Dict[str, torch.Tensor]:
        n = m["R"].numel()
        ms = _markers(m, n)
        out = {k: torch.empty(n, dtype=torch.float64, device=m["R"].device)
               for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt")}
        _check(self.L.trimeg_rhs(self.h, C.byref(ms), n, *[_ptr(out[k], torch.float64) for k in
                                                             ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt")],
                                 _stream(stream)), "trimeg_rhs")
        return out

    def field_upload_aux(self, which: int, data: Optional[torch.Tensor], kind: int, stream=None):
        """which: FIELD_AS (dA^s) or FIELD_AH (dA^h); data None drops the table."""
        if data is not None and self.n_modes > 0:
            want = (self.n_modes, self.n_vert, 6) if kind == 0 else (self.n_tri, self.n_modes, 21)
            if tuple(data.shape) != want:
                raise ValueError(f"field data shape {tuple(data.shape)} != {want}")
        _check(self.L.trimeg_field_upload_aux(self.h, int(which), _ptr(data, torch.complex128), int(kind), _stream(stream)),
               "trimeg_field_upload_aux")

    def rhs_em(self, m: Dict[str, torch.Tensor], stream=None) -> Dict[str, torch.Tensor]:
        n = m["R"].numel()
        ms = _markers(m, n)
        out = {k: torch.empty(n, dtype=torch.float64, device=m["R"].device) for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt")}
        _check(self.L.trimeg_rhs_em(self.h, C.byref(ms), n, *[_ptr(out[k], torch.float64) for k in
                                                                ("dRdt", "dZdt", "dphidt", "dudt", "dwdt")], _stream(stream)),
               "trimeg_rhs_em")
        return out

    def pullback(self, m: Dict[str, torch.Tensor], n: Optional[int] = None, stream=None):
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        _check(self.L.trimeg_pullback(self.h, C.byref(ms), n, _stream(stream)), "trimeg_pullback")

    def scatter(self, m: Dict[str, torch.Tensor], n: Optional[int] = None, out: Optional[torch.Tensor] = None,
                stream=None) -> torch.Tensor:
        """rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p}: complex128 [n_modes][n_vert][6]."""
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        if out is None:
            out = torch.empty((self.n_modes, self.n_vert, 6), dtype=torch.complex128, device=m["R"].device)
        _check(self.L.trimeg_scatter(self.h, C.byref(ms), n, _ptr(out, torch.complex128) if self.n_modes else C.c_void_p(0),
                                     _stream(stream)), "trimeg_scatter")
        return out

    def scatter_static(self, m: Dict[str, torch.Tensor], out: torch.Tensor, n: Optional[int] = None, stream=None) -> torch.Tensor:
        """trimeg_scatter_static: the projection with all scratch in the library's static device array -- no allocation
        anywhere, so `out` (complex128 [n_modes][n_vert][6]) is the caller's."""
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        _check(self.L.trimeg_scatter_static(self.h, C.byref(ms), n, _ptr(out, torch.complex128) if self.n_modes else C.c_void_p(0),
                                            _stream(stream)), "trimeg_scatter_static")
        return out

    def sort(self, m: Dict[str, torch.Tensor], want_perm: bool = False, n: Optional[int] = None,
             stream=None) -> Optional[torch.Tensor]:
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        perm = torch.empty(n, dtype=torch.int64, device=m["R"].device) if want_perm else None
        _check(self.L.trimeg_sort(self.h, C.byref(ms), n, _ptr(perm, torch.int64), _stream(stream)), "trimeg_sort")
        return perm

    def compact(self, m: Dict[str, torch.Tensor], want_perm: bool = False, n: Optional[int] = None, stream=None):
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        perm = torch.empty(n, dtype=torch.int64, device=m["R"].device) if want_perm else None
        na = C.c_size_t(0)
        _check(self.L.trimeg_compact(self.h, C.byref(ms), n, _ptr(perm, torch.int64), C.byref(na), _stream(stream)),
               "trimeg_compact")
        return int(na.value), perm

    def push(self, m: Dict[str, torch.Tensor], dt: float, nsteps: int, n: Optional[int] = None, stream=None):
        n = m["R"].numel() if n is None else int(n)
        ms = _markers(m, n)
        _check(self.L.trimeg_push(self.h, C.byref(ms), n, float(dt), int(nsteps), _stream(stream)), "trimeg_push")

    def get_push_kernel(self) -> int:
        return int(self.L.trimeg_get_push_kernel(self.h))

    def set_push_kernel(self, variant: int):
        _check(self.L.trimeg_set_push_kernel(self.h, int(variant)), "trimeg_set_push_kernel")

    def push_host(self, m_host: Dict[str, torch.Tensor], dt: float, nsteps: int, locate_first: bool = True):
        n = m_host["R"].numel()
        ms = _markers(m_host, n, device="cpu")
        _check(self.L.trimeg_push_host(self.h, C.byref(ms), n, float(dt), int(nsteps), int(bool(locate_first))),
               "trimeg_push_host")

    def release_host_buffers(self):
        _check(self.L.trimeg_release_host_buffers(self.h), "trimeg_release_host_buffers")

    def get_stats(self) -> Dict[str, int]:
        a, b, c = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        _check(self.L.trimeg_get_stats(self.h, C.byref(a), C.byref(b), C.byref(c)), "trimeg_get_stats")
        return dict(n_lost=a.value, n_relocated=b.value, n_launches=c.value)

    def measure_fp64_peak(self) -> float:
        v = C.c_double(0.0)
        _check(self.L.trimeg_measure_fp64_peak(self.h, C.byref(v)), "trimeg_measure_fp64_peak")
        return float(v.value)

    def measure_gather_peak(self, table_bytes: int, record_bytes: int) -> float:
        v = C.c_double(0.0)
        _check(self.L.trimeg_measure_gather_peak(self.h, int(table_bytes), int(record_bytes), C.byref(v)),
               "trimeg_measure_gather_peak")
        return float(v.value)

    def measure_fp64_peak_operands(self, n_reg_operands: int) -> float:
        v = C.c_double(0.0)
        _check(self.L.trimeg_measure_fp64_peak_operands(self.h, int(n_reg_operands), C.byref(v)),
               "trimeg_measure_fp64_peak_operands")
        return float(v.value)

    def get_tile_counters(self) -> Dict[str, int]:
        a = (C.c_int64 * 8)()
        _check(self.L.trimeg_get_tile_counters(self.h, a), "trimeg_get_tile_counters")
        names = ("cyc_group", "n_regroup", "unused", "cyc_eval", "cyc_noslot", "n_fallback", "n_records", "n_stages")
        return {k: int(v) for k, v in zip(names, a)}

    def reset_stats(self):
        _check(self.L.trimeg_reset_stats(self.h), "trimeg_reset_stats")


def context_for(wl, inputs_module=None, eom_variant: int = 0, weight_mode: int = 0) -> Context:
    """Context on the mesh of a workload, with the generator's vertex coordinates so that the
    geometry is bit-identical to any other consumer of the same inputs."""
    if inputs_module is None:
        from . import inputs as inputs_module
    r, Rv, Zv = inputs_module.mesh_nodes(wl)
    return Context(wl.n_r, wl.n_theta, r, wl.params(eom_variant, weight_mode), Rv, Zv)


def mesh_locality_order(vert_R, vert_Z, tri):
    """trimeg_mesh_locality_order: int32 permutation `order`; use tri[order] as the triangle list (host only, no GPU needed)."""
    import numpy as np
    L = load()
    vR = np.ascontiguousarray(vert_R, dtype=np.float64)
    vZ = np.ascontiguousarray(vert_Z, dtype=np.float64)
    tr = np.ascontiguousarray(tri, dtype=np.int32)
    order = np.empty(tr.shape[0], dtype=np.int32)
    dp = C.POINTER(C.c_double)
    ip = C.POINTER(C.c_int32)
    _check(L.trimeg_mesh_locality_order(int(vR.size), vR.ctypes.data_as(dp), vZ.ctypes.data_as(dp), int(tr.shape[0]),
                                        tr.ctypes.data_as(ip), order.ctypes.data_as(ip)), "trimeg_mesh_locality_order")
    return order


def markers_to_device(m, device="cuda") -> Dict[str, torch.Tensor]:
    """numpy marker dict -> torch tensors on `device` ('cell' added as -1 if absent)."""
    import numpy as np
    out = {k: torch.from_numpy(np.ascontiguousarray(m[k], dtype=np.float64)).to(device)
           for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    if "cell" in m:
        out["cell"] = torch.from_numpy(np.ascontiguousarray(m["cell"], dtype=np.int32)).to(device)
    else:
        out["cell"] = torch.full((out["R"].numel(),), -1, dtype=torch.int32, device=device)
    return out
