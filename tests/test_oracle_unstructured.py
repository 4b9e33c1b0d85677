"""Pins for the oracle on an unstructured triangulation with the thesis's box-grid locator (O13; an
intermediate grid of boxes, each holding the triangles that overlap it; the particle's box is found in O(1) and its triangles
are tested one by one).  What fixes it without the oracle's own locator code:
  * the located triangle contains the point by an orientation test with numpy cross products; far points are outside;
  * the box grid gives the result of the same rule over ALL triangles, for any grid resolution;
  * the ring x sector mesh handed in as an "unstructured" list gives the cells, the gather and the push of the structured
    oracle (pinned by test_oracle_locator.py / _gather.py / _physics.py) bit for bit;
  * on a genuinely unstructured (jittered Delaunay, shuffled) mesh the Bell field is C1 across every interior edge, reproduces
    P4 exactly and a quintic not, and the scatter is the adjoint of the gather -- the element code does not lean on the ring
    x sector numbering;
  * the generator's mesh is a valid triangulation of the same polygon (areas add up, interior edges shared by two)."""
import math

import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

import oracle
from helpers import interior_edges, local_coords, phys_derivs, poly_dofs


@pytest.fixture(scope="module")
def umesh(inputs, cfg1):
    Rv, Zv, tri = inputs.unstructured_mesh(cfg1)
    return Rv, Zv, tri


@pytest.fixture(scope="module")
def ou(inputs, cfg1, umesh):
    return oracle.Oracle.unstructured(*umesh, cfg1.params())


def cross2(u, v):
    return u[:, 0] * v[:, 1] - u[:, 1] * v[:, 0]


def _points(cfg1, umesh, n=6000, seed=3):
    """Random points in and around the disc, every vertex, edge midpoints and points a rounding away from edges."""
    Rv, Zv, tri = umesh
    rng = np.random.default_rng(seed)
    r = 1.15 * np.sqrt(rng.random(n)); th = 2 * np.pi * rng.random(n)
    R = [cfg1.R0 + r * np.cos(th), Rv, 0.5 * (Rv[tri[:, 0]] + Rv[tri[:, 1]]), (Rv[tri[:, 1]] + 2 * Rv[tri[:, 2]]) / 3]
    Z = [r * np.sin(th), Zv, 0.5 * (Zv[tri[:, 0]] + Zv[tri[:, 1]]), (Zv[tri[:, 1]] + 2 * Zv[tri[:, 2]]) / 3]
    R, Z = np.concatenate(R), np.concatenate(Z)
    R = np.concatenate([R, R[n:] * (1 + 1e-16), R[n:] * (1 - 1e-16), [np.nan, 1e9, -1e9]])
    Z = np.concatenate([Z, Z[n:] + 1e-17, Z[n:] - 1e-17, [0.0, 0.0, np.nan]])
    return R, Z


def test_generator_gives_a_valid_triangulation_of_the_same_polygon(inputs, cfg1, umesh):
    Rv, Zv, tri = umesh
    _, Rs, Zs = inputs.mesh_nodes(cfg1)
    assert tri.shape == (cfg1.n_tri, 3) and Rv.size == cfg1.n_vert
    a2 = (Rv[tri[:, 1]] - Rv[tri[:, 0]]) * (Zv[tri[:, 2]] - Zv[tri[:, 0]]) - (Rv[tri[:, 2]] - Rv[tri[:, 0]]) * (Zv[tri[:, 1]] - Zv[tri[:, 0]])
    assert np.all(a2 > 0)                                                  # counter-clockwise
    poly = 0.5 * cfg1.n_theta * cfg1.a ** 2 * math.sin(2 * math.pi / cfg1.n_theta)
    assert abs(0.5 * a2.sum() - poly) < 1e-12 * poly
    edges = {}
    for t, (a, b, c) in enumerate(tri):
        for e in ((a, b), (b, c), (c, a)):
            edges.setdefault(tuple(sorted((int(e[0]), int(e[1])))), []).append(t)
    counts = np.array([len(v) for v in edges.values()])
    assert set(counts) == {1, 2} and (counts == 1).sum() == cfg1.n_theta   # boundary = the outer ring's chords
    # the numbering is not the ring x sector one
    assert not np.array_equal(np.sort(Rv), np.sort(Rs)) and not np.array_equal(tri[:50], np.sort(tri[:50], axis=1))


def test_located_triangle_contains_the_point(cfg1, umesh, ou):
    Rv, Zv, tri = umesh
    R, Z = _points(cfg1, umesh)
    cell = ou.locate(R, Z)
    ok = cell >= 0
    t = tri[cell[ok]]
    P = np.stack([R[ok], Z[ok]], axis=1)
    V = [np.stack([Rv[t[:, k]], Zv[t[:, k]]], axis=1) for k in range(3)]
    scale = 0.0
    for k in range(3):
        a, b = V[k], V[(k + 1) % 3]
        cr = cross2(b - a, P - a)                                          # >= 0 for a point on the left of every ccw edge
        scale = max(scale, np.abs(cross2(b - a, V[(k + 2) % 3] - a)).max())
        assert cr.min() > -1e-12 * scale
    # outside: farther than the polygon's circumradius; inside the inscribed circle every point is found
    rr = np.hypot(R - cfg1.R0, Z)
    assert np.all(cell[rr > cfg1.a * (1 + 1e-9)] == -1)
    assert np.all(cell[rr < cfg1.a * math.cos(math.pi / cfg1.n_theta) * (1 - 1e-9)] >= 0)
    assert np.all(cell[-3:] == -1)                                         # NaN and far away


@pytest.mark.parametrize("grid", [(1, 1), (7, 5), (0, 0), (200, 160)])
def test_box_grid_equals_the_rule_over_all_triangles(cfg1, umesh, grid):
    o = oracle.Oracle.unstructured(*umesh, cfg1.params(), nbx=grid[0], nby=grid[1])
    R, Z = _points(cfg1, umesh, seed=5)
    a = o.locate(R, Z)
    b = o.locate_brute(R, Z)
    assert np.array_equal(a, b)
    assert (a >= 0).sum() > 4000 and (a < 0).sum() > 500
    # a vertex is given to one of the triangles that own it (which one is decided by the rounding of the test at the vertex:
    # exact only at a triangle's first vertex) -- and to the lowest-numbered one among those whose first vertex it is
    Rv, Zv, tri = umesh
    cv = o.locate(Rv, Zv)
    assert np.all(cv >= 0) and np.all((tri[cv] == np.arange(Rv.size)[:, None]).any(axis=1))
    first = np.full(Rv.size, 10 ** 9)
    for t in range(tri.shape[0] - 1, -1, -1):
        first[tri[t, 0]] = t
    has = first < 10 ** 9
    assert np.all(cv[has] <= first[has])


def test_structured_mesh_as_a_list_gives_the_structured_oracle(inputs, cfg1, oracle_cfg1):
    """Same vertices, same triangle order: cells, gather and push equal O3 / O4 / O7 bit for bit (random points do not land
    in rounding gaps, where the two gap rules -- inscribed circle, reading O3; margin, reading G31 -- could differ)."""
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    o = oracle.Oracle.unstructured(Rv, Zv, oracle_cfg1.triangles(), cfg1.params())
    assert np.array_equal(o.geom(), oracle_cfg1.geom())
    m = inputs.markers(cfg1, n=3000, seed=9)
    assert np.array_equal(o.locate(m["R"], m["Z"]), oracle_cfg1.locate(m["R"], m["Z"]))
    dofs = inputs.field_dofs(cfg1)
    c1 = oracle_cfg1.bell_from_dofs(cfg1.modes, dofs)
    c2 = o.bell_from_dofs(cfg1.modes, dofs)
    assert np.array_equal(c1, c2)
    g1, g2 = oracle_cfg1.gather(m["R"], m["Z"], m["phi"]), o.gather(m["R"], m["Z"], m["phi"])
    for k in g1:
        assert np.array_equal(g1[k], g2[k]), k
    m["w"] = np.zeros_like(m["R"])
    p1, p2 = oracle_cfg1.push(m, cfg1.dt, 5), o.push(m, cfg1.dt, 5)
    for k in p1:
        assert np.array_equal(p1[k], p2[k]), k


def test_bell_field_on_the_unstructured_mesh_is_c1_and_contains_p4(inputs, cfg1, umesh, ou):
    Rv, Zv, tri = umesh
    rng = np.random.default_rng(11)
    m = inputs.markers(cfg1, n=2000, seed=7)
    for deg, exact in ((4, True), (5, False)):
        C = np.zeros((deg + 1, deg + 1))
        for i in range(deg + 1):
            for j in range(deg + 1 - i):
                C[i, j] = rng.standard_normal()
        ou.bell_from_dofs([0], poly_dofs(C, Rv, Zv).astype(np.complex128)[None])
        out = ou.gather(m["R"], m["Z"], m["phi"])
        x, z = m["R"] - 10.0, m["Z"]
        err = max(np.abs(out["dphi"] - npoly.polyval2d(x, z, C)).max(),
                  np.abs(out["dphi_dR"] - npoly.polyval2d(x, z, npoly.polyder(C, 1, axis=0))).max(),
                  np.abs(out["dphi_dZ"] - npoly.polyval2d(x, z, npoly.polyder(C, 1, axis=1))).max())
        assert (err < 1e-11) if exact else (err > 1e-8), (deg, err)
    # the workload's analytic perturbation: value and normal derivative continuous across every interior edge
    dofs = inputs.field_dofs_at(cfg1, Rv, Zv)
    coef = ou.bell_from_dofs(cfg1.modes, dofs)
    g = ou.geom()
    fscale, gscale = np.abs(dofs[..., 0]).max(), np.abs(dofs[..., 1:3]).max()
    worst_v = worst_n = 0.0
    for (va, vb), (t1, t2) in interior_edges(tri).items():
        tR, tZ = Rv[vb] - Rv[va], Zv[vb] - Zv[va]
        L = math.hypot(tR, tZ)
        nR, nZ = tZ / L, -tR / L
        for s in (0.2, 0.83):
            R, Z = Rv[va] + s * tR, Zv[va] + s * tZ
            vals = []
            for t in (t1, t2):
                xi, eta = local_coords(g[t], R, Z)
                d = phys_derivs(coef[t, 1], g[t], xi, eta)
                vals.append((d[0], nR * d[1] + nZ * d[2]))
            worst_v = max(worst_v, abs(vals[0][0] - vals[1][0]) / fscale)
            worst_n = max(worst_n, abs(vals[0][1] - vals[1][1]) / gscale)
    assert worst_v < 1e-12 and worst_n < 1e-11, (worst_v, worst_n)


def test_scatter_is_the_adjoint_of_gather_and_push_runs(inputs, cfg1, umesh, ou):
    Rv, Zv, tri = umesh
    rng = np.random.default_rng(13)
    modes = [0, 1, 4]
    Y = rng.standard_normal((3, ou.n_vert, 6)) + 1j * rng.standard_normal((3, ou.n_vert, 6))
    m = inputs.markers(cfg1, n=4000, seed=31)
    w = rng.standard_normal(4000)
    ou.bell_from_dofs(modes, Y)
    f = ou.gather(m["R"], m["Z"], m["phi"])["dphi"]
    rhs = ou.scatter(m["R"], m["Z"], m["phi"], w)
    lhs = (w * f).sum()
    tot = (Y[0].real * rhs[0].real).sum() + (Y[1:] * np.conj(rhs[1:])).real.sum()
    assert abs(lhs - tot) < 1e-12 * np.abs(w * f).sum()
    # a push under the workload's field: same physics as on the ring x sector mesh up to the field's discretisation error
    ou.bell_from_dofs(cfg1.modes, inputs.field_dofs_at(cfg1, Rv, Zv))
    os_ = oracle.from_workload(cfg1, inputs)
    os_.bell_from_dofs(cfg1.modes, inputs.field_dofs(cfg1))
    m["w"] = np.zeros(4000)
    a, b = ou.push(m, cfg1.dt, 20), os_.push(m, cfg1.dt, 20)
    assert np.array_equal(a["cell"] < 0, b["cell"] < 0)
    assert np.abs(a["R"] - b["R"]).max() < 1e-4 and np.abs(a["w"] - b["w"]).max() < 0.1 * np.abs(b["w"]).max()
    assert np.abs(a["w"]).max() > 1e-7
