"""ctypes front-end of the CPU oracle (oracle/trimeg_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It never
imports the CUDA package's binding or extension; the only module it shares
with the CUDA path is the seeded input generator (which is passed in by the
caller, not imported here).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np

from .build import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))


class _Params(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("R0", "a", "B0", "q0", "q2", "rho0", "qs_over_ms", "T", "kappa_n", "kappa_T")] + \
               [("eom_variant", C.c_int), ("weight_mode", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, dp, dp, dp, C.POINTER(_Params)]
        L.orc_create_unstructured.restype = C.c_void_p
        L.orc_create_unstructured.argtypes = [C.c_int, dp, dp, C.c_int, ip, C.c_int, C.c_int, C.POINTER(_Params)]
        L.orc_box_count.argtypes = [C.c_void_p]
        L.orc_set_equilibrium_table.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, dp,
                                                C.c_int, C.c_double, C.c_double, dp]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_n_tri.argtypes = [C.c_void_p]
        L.orc_n_vert.argtypes = [C.c_void_p]
        L.orc_get_tri.argtypes = [C.c_void_p, ip]
        L.orc_get_geom.argtypes = [C.c_void_p, dp]
        L.orc_get_rin2.argtypes = [C.c_void_p]
        L.orc_get_rin2.restype = C.c_double
        L.orc_set_params.argtypes = [C.c_void_p, C.POINTER(_Params)]
        L.orc_set_modes.argtypes = [C.c_void_p, C.c_int, ip]
        L.orc_set_coef.argtypes = [C.c_void_p, dp]
        L.orc_get_coef.argtypes = [C.c_void_p, dp]
        L.orc_bell_from_dofs.argtypes = [C.c_void_p, dp]
        L.orc_bell_from_dofs.restype = C.c_int
        L.orc_locate_brute.argtypes = [C.c_void_p, C.c_size_t, dp, dp, ip]
        L.orc_locate.argtypes = [C.c_void_p, C.c_size_t, dp, dp, ip]
        L.orc_bary.argtypes = [C.c_void_p, C.c_size_t, ip, dp, dp, dp]
        L.orc_gather.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, ip, dp, dp, dp, dp]
        L.orc_equilibrium.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp]
        L.orc_rhs.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, dp, ip, dp, dp, dp, dp, dp]
        L.orc_rhs_point.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, dp, dp]
        L.orc_push.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, dp, ip,
                               C.c_double, C.c_int, C.c_int]
        L.orc_rhs_point_em.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, dp, dp]
        L.orc_set_aux_coef.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_rhs_em.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, dp, ip, dp, dp, dp, dp, dp]
        L.orc_pullback.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, dp, ip]
        L.orc_set_spline.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_get_spline.argtypes = [C.c_void_p, dp]
        L.orc_bell_spline_from_dofs.argtypes = [C.c_void_p, C.c_int, dp]
        L.orc_bell_spline_from_dofs.restype = C.c_int
        L.orc_scatter.argtypes = [C.c_void_p, C.c_size_t, dp, dp, dp, dp, ip, dp]
        L.orc_scatter.restype = C.c_long
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


EQ_FIELDS = ("B", "BR", "BZ", "Bphi", "bR", "bZ", "bphi", "dBdR", "dBdZ",
             "dbR_dZ", "dbZ_dR", "dbphi_dR", "dbphi_dZ", "psi")


class Oracle:
    """One mesh + parameter set + (optional) field."""

    def __init__(self, n_r: int, n_theta: int, r_nodes, Rv, Zv, params: Dict):
        self.L = lib()
        self.n_r, self.n_theta = int(n_r), int(n_theta)
        self._r = _f64(r_nodes)
        self._Rv, self._Zv = _f64(Rv), _f64(Zv)
        self._p = _Params(**params)
        self.h = self.L.orc_create(self.n_r, self.n_theta, _d(self._r), _d(self._Rv), _d(self._Zv),
                                   C.byref(self._p))
        if not self.h:
            raise ValueError("orc_create failed")
        self.n_tri = self.L.orc_n_tri(self.h)
        self.n_vert = self.L.orc_n_vert(self.h)
        self.n_modes = 0
        self.mode_n = np.zeros(0, dtype=np.int32)

    @classmethod
    def unstructured(cls, Rv, Zv, tri, params: Dict, nbx: int = 0, nby: int = 0) -> "Oracle":
        """O13: any conforming triangulation (vertex coordinates, int32 [n_tri][3]); nbx x nby boxes (default: about one
        triangle's area per box)."""
        self = cls.__new__(cls)
        self.L = lib()
        self.n_r = self.n_theta = 0
        self._Rv, self._Zv = _f64(Rv), _f64(Zv)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        if nbx <= 0 or nby <= 0:
            nbx = nby = max(1, int(np.sqrt(tri.shape[0] / 2.0)))
        self._p = _Params(**params)
        self.h = self.L.orc_create_unstructured(self._Rv.size, _d(self._Rv), _d(self._Zv), tri.shape[0], _i(tri), int(nbx), int(nby),
                                                C.byref(self._p))
        if not self.h:
            raise ValueError("orc_create_unstructured failed (degenerate triangle or bad index)")
        self.n_tri = self.L.orc_n_tri(self.h)
        self.n_vert = self.L.orc_n_vert(self.h)
        self.n_modes = 0
        self.mode_n = np.zeros(0, dtype=np.int32)
        return self

    def set_equilibrium_table(self, tab: Optional[Dict]):
        """O14: tab = dict(C [nR][nZ], Ra, Za, hR, hZ, D [nF], pa, hp) (inputs.equilibrium_table); None: analytic equilibrium."""
        if tab is None:
            self.L.orc_set_equilibrium_table(self.h, 0, 0, 0.0, 0.0, 0.0, 0.0, None, 0, 0.0, 0.0, None)
            return
        Cc, D = _f64(tab["C"]), _f64(tab["D"])
        self.L.orc_set_equilibrium_table(self.h, Cc.shape[0], Cc.shape[1], float(tab["Ra"]), float(tab["Za"]), float(tab["hR"]),
                                         float(tab["hZ"]), _d(Cc), D.size, float(tab["pa"]), float(tab["hp"]), _d(D))

    def box_entries(self) -> int:
        return int(self.L.orc_box_count(self.h))

    def __del__(self):
        try:
            if getattr(self, "h", None):
                self.L.orc_destroy(self.h)
                self.h = None
        except Exception:
            pass

    # ---- mesh
    def set_params(self, params: Dict):
        self._p = _Params(**params)
        self.L.orc_set_params(self.h, C.byref(self._p))

    def triangles(self) -> np.ndarray:
        out = np.empty((self.n_tri, 3), dtype=np.int32)
        self.L.orc_get_tri(self.h, _i(out))
        return out

    def geom(self) -> np.ndarray:
        out = np.empty((self.n_tri, 6), dtype=np.float64)
        self.L.orc_get_geom(self.h, _d(out))
        return out

    def rin2(self) -> float:
        return float(self.L.orc_get_rin2(self.h))

    # ---- field
    def set_modes(self, mode_n):
        self.mode_n = np.ascontiguousarray(mode_n, dtype=np.int32)
        self.n_modes = int(self.mode_n.size)
        self.L.orc_set_modes(self.h, self.n_modes, _i(self.mode_n))

    def bell_from_dofs(self, mode_n, dofs: np.ndarray) -> np.ndarray:
        """dofs [M][n_vert][6] complex128 -> coefficients [n_tri][M][21] complex128."""
        self.set_modes(mode_n)
        dofs = np.ascontiguousarray(dofs, dtype=np.complex128)
        assert dofs.shape == (self.n_modes, self.n_vert, 6), dofs.shape
        rc = self.L.orc_bell_from_dofs(self.h, _d(dofs.view(np.float64)))
        if rc != 0:
            raise RuntimeError("singular Bell system")
        return self.coeffs()

    def set_coeffs(self, mode_n, coef: np.ndarray):
        self.set_modes(mode_n)
        coef = np.ascontiguousarray(coef, dtype=np.complex128)
        assert coef.shape == (self.n_tri, self.n_modes, 21), coef.shape
        self.L.orc_set_coef(self.h, _d(coef.view(np.float64)))

    def coeffs(self) -> np.ndarray:
        out = np.empty((self.n_tri, self.n_modes, 21), dtype=np.complex128)
        if out.size:
            self.L.orc_get_coef(self.h, _d(out.view(np.float64)))
        return out

    # ---- locator
    def locate_brute(self, R, Z) -> np.ndarray:
        R, Z = _f64(R), _f64(Z)
        cell = np.empty(R.size, dtype=np.int32)
        self.L.orc_locate_brute(self.h, R.size, _d(R), _d(Z), _i(cell))
        return cell

    def locate(self, R, Z) -> np.ndarray:
        R, Z = _f64(R), _f64(Z)
        cell = np.empty(R.size, dtype=np.int32)
        self.L.orc_locate(self.h, R.size, _d(R), _d(Z), _i(cell))
        return cell

    def bary(self, t, R, Z) -> np.ndarray:
        t = np.ascontiguousarray(t, dtype=np.int32)
        R, Z = _f64(R), _f64(Z)
        out = np.empty((R.size, 3), dtype=np.float64)
        self.L.orc_bary(self.h, R.size, _i(t), _d(R), _d(Z), _d(out))
        return out

    # ---- gather / equilibrium / rhs / push
    def gather(self, R, Z, phi):
        R, Z, phi = _f64(R), _f64(Z), _f64(phi)
        n = R.size
        cell = np.empty(n, dtype=np.int32)
        f, fR, fZ, fp = (np.empty(n) for _ in range(4))
        self.L.orc_gather(self.h, n, _d(R), _d(Z), _d(phi), _i(cell), _d(f), _d(fR), _d(fZ), _d(fp))
        return dict(cell=cell, dphi=f, dphi_dR=fR, dphi_dZ=fZ, dphi_dphi=fp)

    def equilibrium(self, R, Z) -> Dict[str, np.ndarray]:
        R, Z = _f64(R), _f64(Z)
        out = np.empty((R.size, 14), dtype=np.float64)
        self.L.orc_equilibrium(self.h, R.size, _d(R), _d(Z), _d(out))
        return {k: out[:, i].copy() for i, k in enumerate(EQ_FIELDS)}

    def rhs(self, R, Z, phi, vpar, mu, w):
        a = [_f64(x) for x in (R, Z, phi, vpar, mu, w)]
        n = a[0].size
        cell = np.empty(n, dtype=np.int32)
        o = [np.empty(n) for _ in range(5)]
        self.L.orc_rhs(self.h, n, *[_d(x) for x in a], _i(cell), *[_d(x) for x in o])
        return dict(cell=cell, dRdt=o[0], dZdt=o[1], dphidt=o[2], dvpardt=o[3], dwdt=o[4])

    def rhs_point(self, R, Z, vpar, mu, w, fld) -> np.ndarray:
        """RHS with field values (dphi, d/dR, d/dZ, d/dphi) handed in: [n][5]."""
        a = [_f64(x) for x in (R, Z, vpar, mu, w)]
        fld = np.ascontiguousarray(fld, dtype=np.float64)
        n = a[0].size
        assert fld.shape == (n, 4)
        out = np.empty((n, 5), dtype=np.float64)
        self.L.orc_rhs_point(self.h, n, *[_d(x) for x in a], _d(fld), _d(out))
        return out

    def push(self, m: Dict[str, np.ndarray], dt: float, nsteps: int, cell: Optional[np.ndarray] = None,
             nthreads: int = 0) -> Dict[str, np.ndarray]:
        """Returns a NEW marker dict (inputs untouched) with 'cell' added."""
        out = {k: np.array(m[k], dtype=np.float64, copy=True, order="C") for k in ("R", "Z", "phi", "vpar", "mu", "w")}
        if cell is None:
            cell = self.locate(out["R"], out["Z"])
        cell = np.array(cell, dtype=np.int32, copy=True, order="C")
        n = out["R"].size
        self.L.orc_push(self.h, n, _d(out["R"]), _d(out["Z"]), _d(out["phi"]), _d(out["vpar"]),
                        _d(out["mu"]), _d(out["w"]), _i(cell), float(dt), int(nsteps), int(nthreads))
        out["cell"] = cell
        return out

    # ---- cubic B-spline toroidal basis (O11): the field of gather / rhs / push becomes sum_j N_j(phi) P_j(xi, eta)
    def set_spline_coeffs(self, n_phi: int, coef: Optional[np.ndarray]):
        """coef real [n_tri][n_phi][21] (None: zeros); n_phi = 0 returns to the harmonic field."""
        self.n_phi = int(n_phi)
        if n_phi > 0 and coef is not None:
            coef = np.ascontiguousarray(coef, dtype=np.float64)
            assert coef.shape == (self.n_tri, n_phi, 21), coef.shape
            self.L.orc_set_spline(self.h, int(n_phi), _d(coef))
        else:
            self.L.orc_set_spline(self.h, int(n_phi), None)

    def bell_spline_from_dofs(self, dofs: np.ndarray) -> np.ndarray:
        """dofs real [n_phi][n_vert][6] -> coefficients real [n_tri][n_phi][21]; the field becomes the spline field."""
        dofs = np.ascontiguousarray(dofs, dtype=np.float64)
        n_phi = dofs.shape[0]
        assert dofs.shape == (n_phi, self.n_vert, 6), dofs.shape
        if self.L.orc_bell_spline_from_dofs(self.h, n_phi, _d(dofs)) != 0:
            raise RuntimeError("singular Bell system")
        self.n_phi = n_phi
        out = np.empty((self.n_tri, n_phi, 21), dtype=np.float64)
        self.L.orc_get_spline(self.h, _d(out))
        return out

    # ---- electromagnetic terms (O9, O10): dA^s = aux 0, dA^h = aux 1, on the mode list of the main field
    # (set_modes / bell_from_dofs / set_coeffs drop the aux tables: set them afterwards)
    def set_aux_coeffs(self, which: int, coef: Optional[np.ndarray]):
        if coef is None:
            self.L.orc_set_aux_coef(self.h, int(which), None)
            return
        coef = np.ascontiguousarray(coef, dtype=np.complex128)
        assert coef.shape == (self.n_tri, self.n_modes, 21), coef.shape
        self.L.orc_set_aux_coef(self.h, int(which), _d(coef.view(np.float64)))

    def rhs_point_em(self, R, Z, upar, mu, w, fld) -> np.ndarray:
        """EM right-hand side with the field values handed in: fld [n][3][4] = (value, d/dR, d/dZ, d/dphi) of dPhi, dA^s, dA^h."""
        a = [_f64(x) for x in (R, Z, upar, mu, w)]
        fld = np.ascontiguousarray(fld, dtype=np.float64)
        n = a[0].size
        assert fld.shape == (n, 3, 4)
        out = np.empty((n, 5), dtype=np.float64)
        self.L.orc_rhs_point_em(self.h, n, *[_d(x) for x in a], _d(fld), _d(out))
        return out

    def rhs_em(self, R, Z, phi, upar, mu, w):
        a = [_f64(x) for x in (R, Z, phi, upar, mu, w)]
        n = a[0].size
        cell = np.empty(n, dtype=np.int32)
        o = [np.empty(n) for _ in range(5)]
        self.L.orc_rhs_em(self.h, n, *[_d(x) for x in a], _i(cell), *[_d(x) for x in o])
        return dict(cell=cell, dRdt=o[0], dZdt=o[1], dphidt=o[2], dudt=o[3], dwdt=o[4])

    def pullback(self, R, Z, phi, upar, w, cell=None):
        """Returns (u_new, w_new); inputs untouched."""
        R, Z, phi = _f64(R), _f64(Z), _f64(phi)
        u = np.array(upar, dtype=np.float64, copy=True, order="C")
        ww = np.array(w, dtype=np.float64, copy=True, order="C")
        cf = None if cell is None else np.ascontiguousarray(cell, dtype=np.int32)
        self.L.orc_pullback(self.h, R.size, _d(R), _d(Z), _d(phi), _d(u), _d(ww), _i(cf) if cf is not None else None)
        return u, ww

    def scatter(self, R, Z, phi, w, cell=None) -> np.ndarray:
        """p2g projection (O8): rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p} for the modes of set_modes /
        bell_from_dofs / set_coeffs; complex128 [M][n_vert][6].  cell: optional int32 flags, markers with cell < 0 are skipped."""
        R, Z, phi, w = _f64(R), _f64(Z), _f64(phi), _f64(w)
        out = np.zeros((self.n_modes, self.n_vert, 6), dtype=np.complex128)
        cf = None if cell is None else np.ascontiguousarray(cell, dtype=np.int32)
        rc = self.L.orc_scatter(self.h, R.size, _d(R), _d(Z), _d(phi), _d(w), _i(cf) if cf is not None else None,
                                _d(out.view(np.float64)))
        if rc < 0:
            raise RuntimeError("singular Bell system")
        self.last_scatter_count = int(rc)
        return out

    def max_threads(self) -> int:
        return int(self.L.orc_max_threads())


def from_workload(wl, inputs_module, eom_variant: int = 0, weight_mode: int = 0) -> Oracle:
    """Oracle on the mesh of a workload; `inputs_module` is the shared seeded generator
    (paper_2601_14301_b200.inputs), passed in so that this package imports nothing of the
    CUDA package."""
    r, Rv, Zv = inputs_module.mesh_nodes(wl)
    return Oracle(wl.n_r, wl.n_theta, r, Rv, Zv, wl.params(eom_variant, weight_mode))
