"""Seeded synthetic inputs for the TRIMEG marker-push hot path.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2601_14301_b200.binding`).  It holds none of the method's
arithmetic: no locator, no Bell expansion, no field evaluation, no equations
of motion.  It only lays out the inputs the five workloads of BASELINE.json
describe (mesh node positions, nodal degrees of freedom of a seeded analytic
function, marker phase-space samples) with numpy, bit-identically for both
consumers.  Recipes: SURVEY.md §8(d) "Synthetic inputs" and readings G8-G16,
restated in DESIGN.md §4.

Nothing here touches a GPU; importing it never loads the CUDA extension.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional, Tuple

import numpy as np

TWO_PI = 2.0 * math.pi


@dataclasses.dataclass(frozen=True)
class Workload:
    """One of BASELINE.json's configs (1-based names cfg1..cfg5)."""

    name: str
    n_r: int
    n_theta: int
    radial: str  # "uniform" | "tanh"
    modes: Tuple[int, ...]
    n_markers: int
    dt: float
    nsteps: int
    seed: int
    kappa_n: float = 1.0
    kappa_T: float = 6.9
    sigma_w: float = 0.0
    marker_recipe: str = "volume"  # "linear_r" | "volume" | "edge10"
    field_recipe: str = "q_window"  # "m123" | "q_window"
    # equilibrium / normalisation common to all configs
    R0: float = 10.0
    a: float = 1.0
    B0: float = 1.0
    q0: float = 1.4
    q2: float = 2.0
    rho0: float = 1.0 / 60.0
    qs_over_ms: float = 1.0
    T: float = 2.0
    tanh_beta: float = 1.5

    @property
    def n_vert(self) -> int:
        return 1 + self.n_r * self.n_theta

    @property
    def n_tri(self) -> int:
        return (2 * self.n_r - 1) * self.n_theta

    def params(self, eom_variant: int = 0, weight_mode: int = 0) -> Dict[str, float]:
        return dict(
            R0=self.R0, a=self.a, B0=self.B0, q0=self.q0, q2=self.q2,
            rho0=self.rho0, qs_over_ms=self.qs_over_ms, T=self.T,
            kappa_n=self.kappa_n, kappa_T=self.kappa_T,
            eom_variant=int(eom_variant), weight_mode=int(weight_mode),
        )


WORKLOADS: Dict[str, Workload] = {
    # BASELINE.json configs[0]: tiny plumbing case
    "cfg1": Workload("cfg1", 8, 32, "uniform", (0, 1), 4096, 0.05, 20, seed=0,
                     kappa_n=1.0, kappa_T=6.9, sigma_w=0.0,
                     marker_recipe="linear_r", field_recipe="m123"),
    # configs[1]: medium ITG-like
    "cfg2": Workload("cfg2", 64, 256, "uniform", (0, 5, 10), 1 << 22, 0.02, 100, seed=2,
                     sigma_w=1e-4),
    # configs[2]: large ITG, table > L2, unsorted markers
    "cfg3": Workload("cfg3", 128, 512, "tanh", (0, 4, 8, 12), 1 << 26, 0.02, 20, seed=3,
                     sigma_w=1e-4),
    # configs[3]: gather-only sweep (marker count is swept by the caller)
    "cfg4": Workload("cfg4", 64, 256, "uniform", (0, 5, 10), 1 << 22, 0.0, 0, seed=4,
                     sigma_w=0.0),
    # configs[4]: many-mode stress case, 10 % of markers start in the outer ring
    "cfg5": Workload("cfg5", 96, 384, "uniform", tuple(range(0, 31, 2)), 1 << 24, 0.01, 50,
                     seed=5, kappa_n=1.0, kappa_T=10.0, sigma_w=1e-4,
                     marker_recipe="edge10"),
}


# --------------------------------------------------------------------------
# mesh node positions (layout only; triangles and geometry factors are built
# independently by the oracle and by the CUDA library from these nodes)
# --------------------------------------------------------------------------
def radial_nodes(wl: Workload) -> np.ndarray:
    """r_0=0 < r_1 < ... < r_{n_r}=a.  'tanh' = reading G13 (denser near a/2)."""
    i = np.arange(wl.n_r + 1, dtype=np.float64)
    if wl.radial == "uniform":
        r = wl.a * i / wl.n_r
    elif wl.radial == "tanh":
        beta = wl.tanh_beta
        u = (2.0 * i / wl.n_r - 1.0) * math.tanh(beta)
        u = np.clip(u, -math.tanh(beta), math.tanh(beta))
        r = 0.5 * wl.a * (1.0 + np.arctanh(u) / beta)
    else:
        raise ValueError(wl.radial)
    r[0] = 0.0
    r[-1] = wl.a
    assert np.all(np.diff(r) > 0)
    return np.ascontiguousarray(r)


def vertex_coords(n_r: int, n_theta: int, r_nodes: np.ndarray, R0: float):
    """Vertex numbering of SURVEY.md §8(c) O1: vertex 0 = axis (R0, 0);
    v(i, j) = 1 + (i-1) n_theta + j at (R0 + r_i cos th_j, r_i sin th_j)."""
    th = TWO_PI * np.arange(n_theta, dtype=np.float64) / n_theta
    c, s = np.cos(th), np.sin(th)
    Rv = np.empty(1 + n_r * n_theta, dtype=np.float64)
    Zv = np.empty_like(Rv)
    Rv[0], Zv[0] = R0, 0.0
    for i in range(1, n_r + 1):
        lo = 1 + (i - 1) * n_theta
        Rv[lo:lo + n_theta] = R0 + r_nodes[i] * c
        Zv[lo:lo + n_theta] = r_nodes[i] * s
    return Rv, Zv


def mesh_nodes(wl: Workload):
    r = radial_nodes(wl)
    Rv, Zv = vertex_coords(wl.n_r, wl.n_theta, r, wl.R0)
    return r, Rv, Zv


# --------------------------------------------------------------------------
# nodal degrees of freedom of the seeded analytic function (reading G14)
# --------------------------------------------------------------------------
def _q(wl: Workload, r):
    return wl.q0 + wl.q2 * (r / wl.a) ** 2


def mode_amplitudes(wl: Workload, seed: Optional[int] = None, sigma: float = 1e-3):
    """A_{n,m} = sigma (N(0,1) + i N(0,1)) / sqrt(2), drawn n-ascending then
    m-ascending.  Returns {n: (m_lo, amplitudes[m_lo .. m_hi])}."""
    rng = np.random.default_rng([wl.seed if seed is None else seed, 1])
    out = {}
    for n in wl.modes:
        if wl.field_recipe == "m123":
            m_lo, m_hi = 1, 3
        else:
            m_lo = int(math.floor(n * wl.q0)) - 3
            m_hi = int(math.ceil(n * (wl.q0 + wl.q2))) + 3
        k = m_hi - m_lo + 1
        re = rng.standard_normal(k)
        im = rng.standard_normal(k)
        out[n] = (m_lo, sigma * (re + 1j * im) / math.sqrt(2.0))
    return out


def analytic_field(wl: Workload, amps, n: int, R, Z):
    """Value and R/Z derivatives up to second order of
        f_n(R, Z) = sum_m A_{n,m} g(r) e^{i m theta},  g = (r/a)(1 - r/a),
    with the poloidal window |m - n q(r)| <= 3 for the q_window recipe (held
    constant when differentiating).  Returns complex array [..., 6] in the
    nodal-DOF order (f, f_R, f_Z, f_RR, f_RZ, f_ZZ) of PAPER.md:350-353.
    Points with r == 0 get all-zero DOFs (reading G14)."""
    R = np.asarray(R, dtype=np.float64)
    Z = np.asarray(Z, dtype=np.float64)
    x = R - wl.R0
    r = np.hypot(x, Z)
    th = np.arctan2(Z, x)
    ok = r > 0.0
    rs = np.where(ok, r, 1.0)
    c, s = np.cos(th), np.sin(th)
    a = wl.a
    g = (rs / a) * (1.0 - rs / a)
    g1 = (1.0 - 2.0 * rs / a) / a
    g2 = -2.0 / (a * a) * np.ones_like(rs)
    m_lo, A = amps[n]
    out = np.zeros(R.shape + (6,), dtype=np.complex128)
    qv = _q(wl, rs)
    for k, Am in enumerate(A):
        m = m_lo + k
        if wl.field_recipe == "q_window":
            sel = ok & (np.abs(m - n * qv) <= 3.0)
        else:
            sel = ok
        if not np.any(sel):
            continue
        e = Am * np.exp(1j * m * th)
        f_r = g1 * e
        f_t = 1j * m * g * e
        f_rr = g2 * e
        f_rt = 1j * m * g1 * e
        f_tt = -(m * m) * g * e
        f = g * e
        f_R = c * f_r - (s / rs) * f_t
        f_Z = s * f_r + (c / rs) * f_t
        f_RR = (c * c * f_rr - (2 * c * s / rs) * f_rt + (s * s / rs ** 2) * f_tt
                + (s * s / rs) * f_r + (2 * c * s / rs ** 2) * f_t)
        f_ZZ = (s * s * f_rr + (2 * c * s / rs) * f_rt + (c * c / rs ** 2) * f_tt
                + (c * c / rs) * f_r - (2 * c * s / rs ** 2) * f_t)
        f_RZ = (c * s * f_rr + ((c * c - s * s) / rs) * f_rt - (c * s / rs ** 2) * f_tt
                - (c * s / rs) * f_r - ((c * c - s * s) / rs ** 2) * f_t)
        comp = np.stack([f, f_R, f_Z, f_RR, f_RZ, f_ZZ], axis=-1)
        out += np.where(sel[..., None], comp, 0.0)
    return out


def field_dofs(wl: Workload, seed: Optional[int] = None, sigma: float = 1e-3) -> np.ndarray:
    """Nodal DOFs [M][n_vert][6] complex128 at the mesh vertices."""
    _, Rv, Zv = mesh_nodes(wl)
    amps = mode_amplitudes(wl, seed, sigma)
    dofs = np.empty((len(wl.modes), wl.n_vert, 6), dtype=np.complex128)
    for k, n in enumerate(wl.modes):
        dofs[k] = analytic_field(wl, amps, n, Rv, Zv)
    dofs[:, 0, :] = 0.0  # axis vertex (reading G14)
    return np.ascontiguousarray(dofs)


def unstructured_mesh(wl: Workload, seed: Optional[int] = None, jitter: float = 0.25):
    """Row f4 (general geometry): an unstructured triangulation of the workload's cross-section -- the ring x sector vertices,
    interior ones displaced at random by up to `jitter` of the local spacing, Delaunay-triangulated (scipy), then vertex
    numbers, triangle order and the starting vertex of every triangle shuffled, so that nothing of the ring x sector
    structure is left in the numbering.  The outer ring stays on the circle r = a (the boundary polygon is the structured
    mesh's).  Returns (Rv, Zv, tri int32 [n_tri][3], counter-clockwise)."""
    from scipy.spatial import Delaunay
    rng = np.random.default_rng([wl.seed if seed is None else seed, 7])
    r_nodes, Rv, Zv = mesh_nodes(wl)
    Rv, Zv = Rv.copy(), Zv.copy()
    nth = wl.n_theta
    for i in range(1, wl.n_r):                                   # interior rings (the axis vertex and the last ring stay)
        dr = min(r_nodes[i] - r_nodes[i - 1], r_nodes[i + 1] - r_nodes[i])
        h = jitter * min(dr, 2.0 * np.pi * r_nodes[i] / nth)
        sl = slice(1 + (i - 1) * nth, 1 + i * nth)
        Rv[sl] += h * (2.0 * rng.random(nth) - 1.0)
        Zv[sl] += h * (2.0 * rng.random(nth) - 1.0)
    tri = Delaunay(np.stack([Rv, Zv], axis=1)).simplices.astype(np.int64)
    e1R, e1Z = Rv[tri[:, 1]] - Rv[tri[:, 0]], Zv[tri[:, 1]] - Zv[tri[:, 0]]
    e2R, e2Z = Rv[tri[:, 2]] - Rv[tri[:, 0]], Zv[tri[:, 2]] - Zv[tri[:, 0]]
    area2 = e1R * e2Z - e2R * e1Z
    tri = tri[np.abs(area2) > 1e-12 * np.abs(area2).max()]         # slivers between collinear hull points, if any
    cw = (Rv[tri[:, 1]] - Rv[tri[:, 0]]) * (Zv[tri[:, 2]] - Zv[tri[:, 0]]) - (Rv[tri[:, 2]] - Rv[tri[:, 0]]) * (Zv[tri[:, 1]] - Zv[tri[:, 0]]) < 0
    tri[cw] = tri[cw][:, [0, 2, 1]]
    perm_v = rng.permutation(Rv.size)                              # new number of old vertex v is inv[v]
    inv = np.empty_like(perm_v); inv[perm_v] = np.arange(Rv.size)
    Rv, Zv = Rv[perm_v], Zv[perm_v]
    tri = inv[tri]
    tri = tri[rng.permutation(tri.shape[0])]
    rot = rng.integers(0, 3, tri.shape[0])
    tri = np.stack([tri[np.arange(tri.shape[0]), (rot + k) % 3] for k in range(3)], axis=1)
    return np.ascontiguousarray(Rv), np.ascontiguousarray(Zv), np.ascontiguousarray(tri, dtype=np.int32)


def _bspline_prefilter(y: np.ndarray, axis: int) -> np.ndarray:
    """Coefficients c[-1..n] (returned with index shift +1, length n + 2) of the uniform cubic B-spline that interpolates the
    n samples y along `axis` with zero second derivative at both ends: (c[i-1] + 4 c[i] + c[i+1])/6 = y[i]."""
    y = np.moveaxis(np.asarray(y, dtype=np.float64), axis, 0)
    n = y.shape[0]
    A = np.zeros((n + 2, n + 2))
    rhs = np.zeros((n + 2,) + y.shape[1:])
    A[0, 0:3] = (1.0, -2.0, 1.0)
    A[n + 1, n - 1:n + 2] = (1.0, -2.0, 1.0)
    for i in range(n):
        A[i + 1, i:i + 3] = (1.0 / 6.0, 4.0 / 6.0, 1.0 / 6.0)
        rhs[i + 1] = y[i]
    c = np.linalg.solve(A, rhs.reshape(n + 2, -1)).reshape((n + 2,) + y.shape[1:])
    return np.moveaxis(c, 0, axis)


def equilibrium_table(wl: Workload, nR: int = 65, nZ: int = 65, nF: int = 17, kappa: float = 1.0, f1: float = 0.0) -> Dict:
    """Row f4 (tabulated equilibrium): stands in for an EQDSK file.  psi(R, Z) = psi_c(x^2 + (Z/kappa)^2), psi_c the poloidal
    flux of the configs' circular equilibrium (psi' = B0 r/q, q = q0 + q2 r^2/a^2; kappa = 1 is that equilibrium itself,
    kappa > 1 an elongated one), sampled on nR x nZ points over [R0 -+ 1.25 a] x [-+ 1.25 kappa a] and turned into uniform
    cubic-B-spline coefficients (interpolating, natural ends); F(psi) = B0 R0 (1 + f1 psi), exactly representable.  Returns
    dict(C [nR+2][nZ+2], Ra, Za, hR, hZ, D [nF], pa, hp): psi = sum C[i][j] beta((R-Ra)/hR - i) beta((Z-Za)/hZ - j)."""
    Rg = np.linspace(wl.R0 - 1.25 * wl.a, wl.R0 + 1.25 * wl.a, nR)
    Zg = np.linspace(-1.25 * kappa * wl.a, 1.25 * kappa * wl.a, nZ)
    s = (Rg[:, None] - wl.R0) ** 2 + (Zg[None, :] / kappa) ** 2
    a2 = wl.a * wl.a
    psi = wl.B0 * a2 / (2.0 * wl.q2) * np.log1p(wl.q2 * s / (wl.q0 * a2)) if wl.q2 != 0.0 else wl.B0 * s / (2.0 * wl.q0)
    C = _bspline_prefilter(_bspline_prefilter(psi, 0), 1)
    hR, hZ = Rg[1] - Rg[0], Zg[1] - Zg[0]
    pmax = float(psi.max())
    hp = pmax / (nF - 3)
    pk = -hp + hp * np.arange(nF)                                  # knot k of F sits at psi = pa + k hp, pa = -hp
    D = wl.B0 * wl.R0 * (1.0 + f1 * pk)
    return dict(C=np.ascontiguousarray(C), Ra=float(Rg[0] - hR), Za=float(Zg[0] - hZ), hR=float(hR), hZ=float(hZ),
                D=np.ascontiguousarray(D), pa=float(-hp), hp=float(hp), kappa=float(kappa), f1=float(f1))


def field_dofs_at(wl: Workload, Rv, Zv, seed: Optional[int] = None, sigma: float = 1e-3) -> np.ndarray:
    """Nodal DOFs [M][n_vert][6] complex128 of the workload's analytic perturbation at arbitrary vertices (row f4)."""
    amps = mode_amplitudes(wl, seed, sigma)
    dofs = np.empty((len(wl.modes), Rv.size, 6), dtype=np.complex128)
    for k, n in enumerate(wl.modes):
        dofs[k] = analytic_field(wl, amps, n, Rv, Zv)
    ax = np.hypot(Rv - wl.R0, Zv) < 1e-12
    dofs[:, ax, :] = 0.0                                           # axis vertex (reading G14)
    return np.ascontiguousarray(dofs)


def spline_dofs(wl: Workload, n_phi: int, seed: Optional[int] = None, sigma: float = 1e-3) -> np.ndarray:
    """Row f3: real nodal DOFs [n_phi][n_vert][6] for the cubic B-spline toroidal basis -- the workload's perturbation
    sum_n Re(Y_n e^{i n phi}) sampled on the n_phi planes phi_j = 2 pi j/n_phi (same radial envelopes, helicity and
    amplitudes as field_dofs; the samples are used as spline coefficients as they are)."""
    Y = field_dofs(wl, seed, sigma)
    phi_j = 2.0 * np.pi * np.arange(n_phi) / n_phi
    out = np.zeros((n_phi, wl.n_vert, 6))
    for k, n in enumerate(wl.modes):
        e = np.exp(1j * n * phi_j)
        out += (Y[k][None, :, :] * e[:, None, None]).real
    return np.ascontiguousarray(out)


# --------------------------------------------------------------------------
# markers
# --------------------------------------------------------------------------
def _B_loading(wl: Workload, R, Z):
    """|B| of the configs' circular equilibrium (B_phi = B0 R0/R, poloidal field
    from q(r)), used ONLY to turn the sampled v_perp into mu = v_perp^2 / 2B as
    the configs prescribe.  It is part of the loading recipe; neither the
    oracle nor the CUDA path calls it."""
    x = R - wl.R0
    s = x * x + Z * Z
    qb = wl.q0 + wl.q2 * s / (wl.a * wl.a)
    return wl.B0 * np.sqrt(wl.R0 ** 2 + s / (qb * qb)) / R


def markers(wl: Workload, n: Optional[int] = None, seed: Optional[int] = None) -> Dict[str, np.ndarray]:
    """SoA marker sample {R, Z, phi, vpar, mu, w} (float64, length n).
    Draw order: u_r, u_theta, u_phi ~ U(0,1); vpar ~ N(0,1);
    v_perp ~ Rayleigh(1); w ~ N(0,1) sigma_w."""
    n = wl.n_markers if n is None else int(n)
    rng = np.random.default_rng([wl.seed if seed is None else seed, 2])
    u_r = rng.random(n)
    u_t = rng.random(n)
    u_p = rng.random(n)
    vpar = rng.standard_normal(n)
    vperp = rng.rayleigh(1.0, n)
    w = rng.standard_normal(n) * wl.sigma_w
    a = wl.a
    if wl.marker_recipe == "linear_r":
        r = a * (0.1 + 0.8 * u_r)
    elif wl.marker_recipe == "volume":
        r = a * np.sqrt(0.01 + 0.80 * u_r)
    elif wl.marker_recipe == "edge10":
        r = a * np.sqrt(0.01 + 0.80 * u_r)
        n_core = (9 * n) // 10
        r[n_core:] = a * np.sqrt(0.95 ** 2 + (1.0 - 0.95 ** 2) * u_r[n_core:])
    else:
        raise ValueError(wl.marker_recipe)
    th = TWO_PI * u_t
    R = wl.R0 + r * np.cos(th)
    Z = r * np.sin(th)
    phi = TWO_PI * u_p
    mu = vperp * vperp / (2.0 * _B_loading(wl, R, Z))
    out = dict(R=R, Z=Z, phi=phi, vpar=vpar, mu=mu, w=w)
    if wl.marker_recipe == "edge10":
        perm = rng.permutation(n)
        out = {k: v[perm] for k, v in out.items()}
    return {k: np.ascontiguousarray(v, dtype=np.float64) for k, v in out.items()}


def positions(wl: Workload, n: Optional[int] = None, seed: Optional[int] = None) -> Dict[str, np.ndarray]:
    """{R, Z, phi} of markers(wl, n) alone (the first three draws of the same stream: bit-identical to the full
    sample for the recipes without a final permutation) -- for the gather-only sweep, whose largest sizes (2^28)
    would otherwise draw three more 2 GB arrays nobody reads."""
    n = wl.n_markers if n is None else int(n)
    if wl.marker_recipe == "edge10":
        m = markers(wl, n, seed)
        return {k: m[k] for k in ("R", "Z", "phi")}
    rng = np.random.default_rng([wl.seed if seed is None else seed, 2])
    u_r = rng.random(n)
    r = wl.a * (0.1 + 0.8 * u_r) if wl.marker_recipe == "linear_r" else wl.a * np.sqrt(0.01 + 0.80 * u_r)
    del u_r
    th = TWO_PI * rng.random(n)
    R = wl.R0 + r * np.cos(th)
    Z = r * np.sin(th)
    del r, th
    phi = TWO_PI * rng.random(n)
    return dict(R=R, Z=Z, phi=phi)


def subsample(m: Dict[str, np.ndarray], stride: int) -> Dict[str, np.ndarray]:
    """Every stride-th marker (markers are independent: PAPER.md:590)."""
    return {k: np.ascontiguousarray(v[::stride]) for k, v in m.items()}
