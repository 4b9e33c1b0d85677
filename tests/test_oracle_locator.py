"""Pins for the oracle's locator (O3): the plain definition is brute force over all
triangles; the O(1) candidate search must agree with it bit for bit."""
import dataclasses
import math

import numpy as np
import pytest

import oracle


def _numpy_point_in_triangle(Rv, Zv, tri, R, Z):
    """Independent formulation: signs of the three edge cross products (no local
    coordinates, no division).  Returns, per point, the list of containing triangles."""
    a, b, c = tri[:, 0], tri[:, 1], tri[:, 2]
    def cross(p, q):
        return (Rv[q] - Rv[p])[None, :] * (Z[:, None] - Zv[p][None, :]) - \
               (Zv[q] - Zv[p])[None, :] * (R[:, None] - Rv[p][None, :])
    d1, d2, d3 = cross(a, b), cross(b, c), cross(c, a)
    return (d1 > 0) & (d2 > 0) & (d3 > 0), np.minimum(np.minimum(d1, d2), d3)


def test_brute_force_matches_cross_product_test(inputs, cfg1, oracle_cfg1):
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    tri = oracle_cfg1.triangles()
    rng = np.random.default_rng(5)
    n = 20000
    r = np.sqrt(rng.random(n)) * 1.05
    th = 2 * np.pi * rng.random(n)
    R, Z = 10.0 + r * np.cos(th), r * np.sin(th)
    strict, margin = _numpy_point_in_triangle(Rv, Zv, tri, R, Z)
    cnt = strict.sum(axis=1)
    cell = oracle_cfg1.locate_brute(R, Z)
    # away from edges (cross products are twice areas, ~1e-3..1e-2 here) the answer is unique
    clear = np.abs(margin).min(axis=1) > 1e-9
    assert clear.mean() > 0.99
    assert np.all(cnt[clear] <= 1)                                   # at most one triangle
    inside = clear & (cnt == 1)
    assert np.array_equal(cell[inside], strict[inside].argmax(axis=1))
    outside = clear & (cnt == 0)
    assert np.all(cell[outside] == -1)
    assert outside.sum() > 100 and inside.sum() > 10000


def _probe_points(wl, n, seed):
    rng = np.random.default_rng(seed)
    r = np.concatenate([np.sqrt(rng.random(n)) * 1.02 * wl.a,          # whole disc + a bit outside
                        rng.random(n // 8) * 1e-3 * wl.a,              # near the axis
                        wl.a * (1 - 5e-3 * rng.random(n // 8))])       # near the outer boundary
    th = 2 * np.pi * rng.random(r.size)
    return wl.R0 + r * np.cos(th), r * np.sin(th)


def test_o1_locator_equals_brute_force_cfg1(cfg1, oracle_cfg1):
    R, Z = _probe_points(cfg1, 60000, 1)
    assert np.array_equal(oracle_cfg1.locate(R, Z), oracle_cfg1.locate_brute(R, Z))


@pytest.mark.parametrize("name,n", [("cfg2", 3000), ("cfg3", 800), ("cfg5", 1500)])
def test_o1_locator_equals_brute_force_large_meshes(inputs, name, n):
    wl = inputs.WORKLOADS[name]
    o = oracle.from_workload(wl, inputs)
    R, Z = _probe_points(wl, n, 2)
    a, b = o.locate(R, Z), o.locate_brute(R, Z)
    assert np.array_equal(a, b)
    assert (a >= 0).sum() > n // 2 and (a < 0).sum() > 0


def test_barycentric_sum_and_signs(cfg1, oracle_cfg1):
    R, Z = _probe_points(cfg1, 5000, 3)
    cell = oracle_cfg1.locate(R, Z)
    ok = cell >= 0
    b = oracle_cfg1.bary(cell[ok], R[ok], Z[ok])
    assert np.abs(b.sum(axis=1) - 1.0).max() < 1e-12      # xi + eta + lambda0 = 1
    assert b.min() >= 0.0                                    # inside() passed


def test_points_on_vertices_and_edges_resolve_to_lowest_index(inputs, cfg1, oracle_cfg1):
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    tri = oracle_cfg1.triangles()
    # every vertex: the point is a vertex of several triangles; brute force and O(1) must agree,
    # and the result must be one of the triangles that own the vertex
    cb, cl = oracle_cfg1.locate_brute(Rv, Zv), oracle_cfg1.locate(Rv, Zv)
    assert np.array_equal(cb, cl)
    outer = np.arange(Rv.size) >= 1 + (cfg1.n_r - 1) * cfg1.n_theta
    for v in range(Rv.size):
        owners = np.where((tri == v).any(axis=1))[0]
        if cb[v] >= 0:
            # lowest t with inside(t): all owners lower than the hit must have failed inside()
            assert cb[v] in owners
        else:
            assert outer[v]          # only outer-boundary vertices may round to "outside"
    # axis vertex is shared by all fan triangles: lowest index is 0
    assert cb[0] == 0
    # midpoints of the radial edges theta = 0 (exactly representable: Z = 0)
    i = np.arange(1, cfg1.n_r)
    Rm = 0.5 * (Rv[1 + (i - 1) * cfg1.n_theta] + Rv[1 + i * cfg1.n_theta])
    cm = oracle_cfg1.locate_brute(Rm, np.zeros_like(Rm))
    b = oracle_cfg1.bary(cm, Rm, np.zeros_like(Rm))
    assert np.all(cm >= 0) and np.all(b.min(axis=1) == 0.0)   # on an edge exactly
    assert np.array_equal(cm, oracle_cfg1.locate(Rm, np.zeros_like(Rm)))
    # the two triangles sharing that edge: k=0 of sector 0 (lower index) vs k=1 of sector n_theta-1
    lower = cfg1.n_theta + 2 * ((i - 1) * cfg1.n_theta + 0)
    assert np.array_equal(cm, lower)


def test_outside_and_nan(cfg1, oracle_cfg1):
    R = np.array([10.0 + 1.0001, 10.0, 12.0, np.nan, 10.0 + math.cos(math.pi / 32) * 1.0 + 1e-9])
    Z = np.array([0.0, 1.01, 0.0, 0.0, 0.0])
    # last point: beyond the midpoint... of no chord (theta = 0 is a vertex direction) -> inside
    c = oracle_cfg1.locate(R, Z)
    assert list(c[:4]) == [-1, -1, -1, -1]
    assert c[4] >= 0
    assert np.array_equal(c, oracle_cfg1.locate_brute(R, Z))
    # chord midpoint direction: the domain is the outer POLYGON, not the circle r <= a (rule L4)
    th = math.pi / 32
    rin = math.cos(th)
    for r, want_inside in ((rin - 1e-9, True), (rin + 1e-9, False)):
        cc = oracle_cfg1.locate([10.0 + r * math.cos(th)], [r * math.sin(th)])[0]
        assert (cc >= 0) == want_inside
    assert abs(oracle_cfg1.rin2() - rin * rin) < 1e-14


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5"])
def test_sagitta_rule_l4_holds_for_all_workloads(inputs, name):
    """The 3x3 neighbourhood suffices iff the chord sagitta is smaller than the next ring."""
    wl = inputs.WORKLOADS[name]
    r = inputs.radial_nodes(wl)
    sag = r[1:-1] * (1 - math.cos(math.pi / wl.n_theta))
    assert np.all(sag < np.diff(r)[1:])
