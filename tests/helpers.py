"""Test-side helpers: independent evaluation of the element polynomials with numpy's
polynomial routines, tolerance helpers, small meshes.  Nothing here is imported by the
oracle or by the CUDA package."""
from __future__ import annotations

import numpy as np
from numpy.polynomial import polynomial as npoly

# degree-major monomial order of the coefficient tables: k <-> (i, j) = xi^i eta^j
MONO_IJ = [(d - j, j) for d in range(6) for j in range(d + 1)]
assert len(MONO_IJ) == 21


def coef_matrix(c21):
    """21 coefficients (degree-major) -> 6x6 matrix C[i, j] for numpy.polynomial."""
    c21 = np.asarray(c21)
    C = np.zeros((6, 6), dtype=c21.dtype)
    for k, (i, j) in enumerate(MONO_IJ):
        C[i, j] = c21[k]
    return C


def poly_eval(c21, xi, eta, a=0, b=0):
    """d^a/dxi^a d^b/deta^b P(xi, eta) using numpy.polynomial (polyder + polyval2d)."""
    C = coef_matrix(c21)
    if a:
        C = npoly.polyder(C, a, axis=0)
    if b:
        C = npoly.polyder(C, b, axis=1)
    return npoly.polyval2d(np.asarray(xi, dtype=np.float64), np.asarray(eta, dtype=np.float64), C)


def phys_derivs(c21, g, xi, eta):
    """(P, P_R, P_Z, P_RR, P_RZ, P_ZZ) at (xi, eta) for a triangle with geometry row
    g = (R_v0, Z_v0, xi_R, xi_Z, eta_R, eta_Z); chain rule with the affine map."""
    xR, xZ, eR, eZ = g[2], g[3], g[4], g[5]
    P = poly_eval(c21, xi, eta)
    Px, Pe = poly_eval(c21, xi, eta, 1, 0), poly_eval(c21, xi, eta, 0, 1)
    Pxx, Pxe, Pee = poly_eval(c21, xi, eta, 2, 0), poly_eval(c21, xi, eta, 1, 1), poly_eval(c21, xi, eta, 0, 2)
    return np.stack([
        P,
        xR * Px + eR * Pe,
        xZ * Px + eZ * Pe,
        xR * xR * Pxx + 2 * xR * eR * Pxe + eR * eR * Pee,
        xR * xZ * Pxx + (xR * eZ + xZ * eR) * Pxe + eR * eZ * Pee,
        xZ * xZ * Pxx + 2 * xZ * eZ * Pxe + eZ * eZ * Pee,
    ], axis=-1)


def local_coords(g, R, Z):
    dx, dz = R - g[0], Z - g[1]
    return g[2] * dx + g[3] * dz, g[4] * dx + g[5] * dz


def poly_dofs(poly_RZ, Rv, Zv):
    """Nodal DOFs (f, f_R, f_Z, f_RR, f_RZ, f_ZZ) of a global polynomial given as a
    numpy.polynomial 2-D coefficient matrix in (R - 10, Z)."""
    x, z = Rv - 10.0, Zv
    C = np.asarray(poly_RZ)
    def der(a, b):
        D = C
        if a:
            D = npoly.polyder(D, a, axis=0)
        if b:
            D = npoly.polyder(D, b, axis=1)
        return npoly.polyval2d(x, z, D)
    return np.stack([der(0, 0), der(1, 0), der(0, 1), der(2, 0), der(1, 1), der(0, 2)], axis=-1)


def rel_err(a, b, scale):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), scale)


def wrap_diff(a, b):
    """|a - b| modulo 2 pi (phi is compared modulo 2 pi, reading G17)."""
    d = (np.asarray(a) - np.asarray(b) + np.pi) % (2 * np.pi) - np.pi
    return np.abs(d)


def interior_edges(tri):
    """{(va, vb) sorted: [triangle ids]} for edges shared by two triangles."""
    edges = {}
    for t, (a, b, c) in enumerate(tri):
        for e in ((a, b), (b, c), (c, a)):
            edges.setdefault(tuple(sorted((int(e[0]), int(e[1])))), []).append(t)
    return {e: ts for e, ts in edges.items() if len(ts) == 2}
