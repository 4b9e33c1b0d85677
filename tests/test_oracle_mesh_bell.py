"""Pins for the oracle's mesh (O1) and Bell reduced-quintic expansion (O2).

What fixes the expected values (SURVEY.md §8(c) "What pins each part"):
closed-form counts and areas; the defining properties of the element
(18 quintic basis functions, 6 DOFs per vertex, C1 continuity);
exact reproduction of P4; an exact-rational solve of the element's definition
written with sympy derivatives (no hand-derived rows)."""
import math

import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

import oracle
from helpers import (MONO_IJ, interior_edges, local_coords, phys_derivs, poly_dofs, poly_eval)


def test_counts_cfg1(oracle_cfg1):
    # BASELINE.json configs[0]: 8 rings x 32 sectors: 257 vertices, 480 triangles (G12)
    assert oracle_cfg1.n_vert == 257
    assert oracle_cfg1.n_tri == 480


@pytest.mark.parametrize("name,ntri", [("cfg2", 32512), ("cfg3", 130560), ("cfg5", 73344)])
def test_counts_formula(inputs, name, ntri):
    wl = inputs.WORKLOADS[name]
    assert wl.n_tri == ntri == (2 * wl.n_r - 1) * wl.n_theta
    assert wl.n_vert == 1 + wl.n_r * wl.n_theta


def test_triangles_ccw_and_area(inputs, cfg1, oracle_cfg1):
    g = oracle_cfg1.geom()
    # D = 1 / (xi_R eta_Z - xi_Z eta_R) = twice the signed area
    det = g[:, 2] * g[:, 5] - g[:, 3] * g[:, 4]
    assert np.all(det > 0)                     # counter-clockwise
    area = 0.5 / det
    poly_area = 0.5 * cfg1.n_theta * cfg1.a ** 2 * math.sin(2 * math.pi / cfg1.n_theta)
    assert abs(area.sum() - poly_area) < 1e-13


def test_vertices_map_to_reference(inputs, cfg1, oracle_cfg1):
    # vertices at (xi, eta) = (0,0), (1,0), (0,1)
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    g, tri = oracle_cfg1.geom(), oracle_cfg1.triangles()
    ref = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0]])
    for k in range(3):
        xi, eta = local_coords(g.T, Rv[tri[:, k]], Zv[tri[:, k]])
        assert np.abs(xi - ref[k, 0]).max() < 1e-12
        assert np.abs(eta - ref[k, 1]).max() < 1e-12


def test_each_interior_edge_shared_by_two(oracle_cfg1, cfg1):
    tri = oracle_cfg1.triangles()
    n_edges_total = (3 * oracle_cfg1.n_tri + cfg1.n_theta) // 2   # boundary edges = n_theta
    assert len(interior_edges(tri)) == n_edges_total - cfg1.n_theta


@pytest.fixture(scope="module")
def bell_cfg1(inputs, cfg1, oracle_cfg1):
    dofs = inputs.field_dofs(cfg1)
    coef = oracle_cfg1.bell_from_dofs(cfg1.modes, dofs)
    return dofs, coef


def test_dof_reproduction(inputs, cfg1, oracle_cfg1, bell_cfg1):
    """(i) coefficients reproduce value, first and second derivatives at the vertices."""
    dofs, coef = bell_cfg1
    g, tri = oracle_cfg1.geom(), oracle_cfg1.triangles()
    ref = [(0.0, 0.0), (1.0, 0.0), (0.0, 1.0)]
    worst = 0.0
    for t in range(oracle_cfg1.n_tri):
        for m in range(len(cfg1.modes)):
            for k, (xi, eta) in enumerate(ref):
                got = phys_derivs(coef[t, m], g[t], xi, eta)
                want = dofs[m, tri[t, k]]
                scale = np.maximum(np.abs(want), np.abs(dofs[m]).max(axis=0))
                worst = max(worst, float((np.abs(got - want) / scale).max()))
    assert worst < 1e-12, worst


def test_c1_continuity_across_edges(inputs, cfg1, oracle_cfg1, bell_cfg1):
    """(ii) value and normal derivative are continuous across every interior edge."""
    dofs, coef = bell_cfg1
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    g, tri = oracle_cfg1.geom(), oracle_cfg1.triangles()
    worst_v = worst_n = 0.0
    fscale = np.abs(dofs[..., 0]).max()
    gscale = np.abs(dofs[..., 1:3]).max()
    for (va, vb), (t1, t2) in interior_edges(tri).items():
        tR, tZ = Rv[vb] - Rv[va], Zv[vb] - Zv[va]
        L = math.hypot(tR, tZ)
        nR, nZ = tZ / L, -tR / L
        for s in (0.2, 0.5, 0.83):
            R, Z = Rv[va] + s * tR, Zv[va] + s * tZ
            vals = []
            for t in (t1, t2):
                xi, eta = local_coords(g[t], R, Z)
                d = phys_derivs(coef[t, 1], g[t], xi, eta)
                vals.append((d[0], nR * d[1] + nZ * d[2]))
            worst_v = max(worst_v, abs(vals[0][0] - vals[1][0]) / fscale)
            worst_n = max(worst_n, abs(vals[0][1] - vals[1][1]) / gscale)
    assert worst_v < 1e-12, worst_v
    assert worst_n < 1e-12, worst_n


def _random_poly(rng, deg):
    C = np.zeros((deg + 1, deg + 1))
    for i in range(deg + 1):
        for j in range(deg + 1 - i):
            C[i, j] = rng.standard_normal()
    return C


def test_p4_reproduced_quintic_not(inputs, cfg1, oracle_cfg1):
    """(iii) Bell's space contains P4: a global quartic in (R - R0, Z) is reproduced exactly
    everywhere; (iv) negative control: a global quintic is not."""
    rng = np.random.default_rng(11)
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    m = inputs.markers(cfg1, n=2000, seed=7)
    for deg, expect_exact in ((4, True), (5, False)):
        C = _random_poly(rng, deg)
        dofs = poly_dofs(C, Rv, Zv).astype(np.complex128)[None]
        oracle_cfg1.bell_from_dofs([0], dofs)
        out = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
        x, z = m["R"] - 10.0, m["Z"]
        f = npoly.polyval2d(x, z, C)
        fR = npoly.polyval2d(x, z, npoly.polyder(C, 1, axis=0))
        fZ = npoly.polyval2d(x, z, npoly.polyder(C, 1, axis=1))
        err = max(np.abs(out["dphi"] - f).max(), np.abs(out["dphi_dR"] - fR).max(),
                  np.abs(out["dphi_dZ"] - fZ).max())
        if expect_exact:
            assert err < 1e-12, err
        else:
            assert err > 1e-8, err


def test_convergence_order(inputs):
    """(v) smooth function: error falls ~2^5 per mesh halving (P4-complete element)."""
    f = lambda R, Z: np.sin(1.3 * (R - 10.0) + 0.4) * np.cos(0.9 * Z - 0.2)
    errs = []
    for n_r, n_t in ((4, 16), (8, 32), (16, 64)):
        import dataclasses
        wl = dataclasses.replace(inputs.WORKLOADS["cfg1"], n_r=n_r, n_theta=n_t)
        o = oracle.from_workload(wl, inputs)
        _, Rv, Zv = inputs.mesh_nodes(wl)
        x, z = Rv - 10.0, Zv
        s, c = np.sin(1.3 * x + 0.4), np.cos(1.3 * x + 0.4)
        cz, sz = np.cos(0.9 * z - 0.2), np.sin(0.9 * z - 0.2)
        dofs = np.stack([s * cz, 1.3 * c * cz, -0.9 * s * sz,
                         -1.69 * s * cz, -1.17 * c * sz, -0.81 * s * cz], axis=-1)
        o.bell_from_dofs([0], dofs.astype(np.complex128)[None])
        m = inputs.markers(wl, n=4000, seed=3)
        out = o.gather(m["R"], m["Z"], m["phi"])
        errs.append(np.abs(out["dphi"] - f(m["R"], m["Z"])).max())
    assert errs[0] / errs[1] > 16 and errs[1] / errs[2] > 16, errs


@pytest.mark.parametrize("t", [3, 40, 41, 479])
def test_bell_against_exact_rational_definition(inputs, cfg1, oracle_cfg1, t):
    """The element's definition solved exactly: unknown quintic in (xi, eta), xi/eta affine in
    (R, Z); sympy differentiates in R, Z (no hand-derived chain-rule rows); the normal
    derivative along each edge must be a cubic in the edge parameter."""
    import sympy as sp
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    tri = oracle_cfg1.triangles()[t]
    rng = np.random.default_rng(100 + t)
    dof = rng.integers(-5, 6, size=(3, 6))
    dofs = np.zeros((1, oracle_cfg1.n_vert, 6), dtype=np.complex128)
    for k in range(3):
        dofs[0, tri[k]] = dof[k]
    coef = oracle_cfg1.bell_from_dofs([0], dofs)[t, 0].real

    R, Z, s = sp.symbols("R Z s")
    V = [(sp.Rational(float(Rv[v])), sp.Rational(float(Zv[v]))) for v in tri]
    # affine map with vertices -> (0,0), (1,0), (0,1)
    M = sp.Matrix([[V[1][0] - V[0][0], V[2][0] - V[0][0]], [V[1][1] - V[0][1], V[2][1] - V[0][1]]])
    xe = M.inv() * sp.Matrix([R - V[0][0], Z - V[0][1]])
    xi, eta = xe[0], xe[1]
    c = sp.symbols("c0:21")
    P = sum(c[k] * xi ** i * eta ** j for k, (i, j) in enumerate(MONO_IJ))
    eqs = []
    ders = [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]
    for k in range(3):
        for d, (a, b) in enumerate(ders):
            e = P
            if a:
                e = sp.diff(e, R, a)
            if b:
                e = sp.diff(e, Z, b)
            eqs.append(sp.expand(e.subs({R: V[k][0], Z: V[k][1]})) - int(dof[k, d]))
    for a, b in ((0, 1), (0, 2), (1, 2)):
        tR, tZ = V[b][0] - V[a][0], V[b][1] - V[a][1]
        dn = tZ * sp.diff(P, R) - tR * sp.diff(P, Z)
        on_edge = sp.expand(dn.subs({R: V[a][0] + s * tR, Z: V[a][1] + s * tZ}))
        eqs.append(sp.Poly(on_edge, s).coeff_monomial(s ** 4))
    A, bvec = sp.linear_eq_to_matrix(eqs, list(c))
    sol = A.LUsolve(bvec)
    exact = np.array([float(v) for v in sol])
    assert np.abs(coef - exact).max() <= 1e-12 * max(1.0, np.abs(exact).max()), \
        (np.abs(coef - exact).max(), np.abs(exact).max())
