"""Pins for the oracle's cubic B-spline toroidal basis (O11; C1 triangles in (R, Z), cubic splines in
Phi on a uniform periodic grid).  What the mathematics fixes: the uniform cubic B-spline itself (checked against
scipy.interpolate.BSpline and its textbook values), partition of unity, Marsden's identities (linear and quadratic
reproduction), C2 continuity across the knots, d/dphi against finite differences; and the (R, Z) part against the pinned
harmonic gather (O4) of the same element polynomial."""
import numpy as np
import pytest
from scipy.interpolate import BSpline


@pytest.fixture(scope="module")
def setup(inputs, cfg1, oracle_cfg1):
    m = inputs.markers(cfg1, n=600, seed=61)
    return m


def _const_planes(o, n_phi, values):
    """every plane j carries the constant polynomial values[j] on every triangle"""
    c = np.zeros((o.n_tri, n_phi, 21))
    c[:, :, 0] = np.asarray(values)[None, :]
    o.set_spline_coeffs(n_phi, c)


def test_basis_function_is_the_uniform_cubic_b_spline(oracle_cfg1, setup):
    o, m = oracle_cfg1, setup
    n_phi = 16
    h = 2 * np.pi / n_phi
    vals = np.zeros(n_phi); vals[5] = 1.0
    _const_planes(o, n_phi, vals)
    x = np.linspace(-2.5, 2.5, 401)
    R = np.full_like(x, m["R"][0]); Z = np.full_like(x, m["Z"][0])
    g = o.gather(R, Z, 5 * h + x * h)
    beta = BSpline.basis_element([-2, -1, 0, 1, 2], extrapolate=False)
    want = np.nan_to_num(beta(x))
    assert np.abs(g["dphi"] - want).max() < 1e-14
    dwant = np.nan_to_num(beta.derivative()(x)) / h
    assert np.abs(g["dphi_dphi"] - dwant).max() < 1e-13 / h
    for xx, v in ((0.0, 2 / 3), (1.0, 1 / 6), (-1.0, 1 / 6), (2.0, 0.0), (0.5, 23 / 48)):
        assert abs(o.gather([R[0]], [Z[0]], [5 * h + xx * h])["dphi"][0] - v) < 1e-15
    assert np.all(g["dphi_dR"] == 0.0) and np.all(g["dphi_dZ"] == 0.0)
    # periodic images: plane 0 is felt just below 2 pi
    vals = np.zeros(n_phi); vals[0] = 1.0
    _const_planes(o, n_phi, vals)
    assert abs(o.gather([R[0]], [Z[0]], [2 * np.pi - 0.5 * h])["dphi"][0] - 23 / 48) < 1e-15
    o.set_spline_coeffs(0, None)


def test_partition_of_unity_and_marsden_identities(oracle_cfg1, setup):
    o, m = oracle_cfg1, setup
    n_phi = 12
    h = 2 * np.pi / n_phi
    _const_planes(o, n_phi, np.ones(n_phi))
    g = o.gather(m["R"], m["Z"], m["phi"])
    assert np.abs(g["dphi"] - 1.0).max() < 1e-15 and np.abs(g["dphi_dphi"]).max() < 1e-14
    # sum_j phi_j N_j(phi) = phi and sum_j (phi_j^2 - h^2/3) N_j(phi) = phi^2 (away from the periodic seam)
    phi = 2 * h + (2 * np.pi - 5 * h) * np.random.default_rng(1).random(m["R"].size)
    pj = h * np.arange(n_phi)
    _const_planes(o, n_phi, pj)
    g = o.gather(m["R"], m["Z"], phi)
    assert np.abs(g["dphi"] - phi).max() < 1e-14 and np.abs(g["dphi_dphi"] - 1.0).max() < 1e-13
    _const_planes(o, n_phi, pj * pj - h * h / 3)
    g = o.gather(m["R"], m["Z"], phi)
    assert np.abs(g["dphi"] - phi * phi).max() < 1e-13 and np.abs(g["dphi_dphi"] - 2 * phi).max() < 1e-12
    o.set_spline_coeffs(0, None)


def test_c2_across_knots_and_dphi_against_finite_differences(oracle_cfg1, setup):
    o, m = oracle_cfg1, setup
    n_phi = 8
    h = 2 * np.pi / n_phi
    rng = np.random.default_rng(2)
    _const_planes(o, n_phi, rng.standard_normal(n_phi))
    R, Z = m["R"][:1], m["Z"][:1]
    f = lambda p: o.gather(np.full(len(p), R[0]), np.full(len(p), Z[0]), np.asarray(p))
    d = 1e-3
    for k in range(n_phi):
        knot = k * h
        left = f([knot - 2 * d, knot - d, knot])["dphi"]
        right = f([knot, knot + d, knot + 2 * d])["dphi"]
        s_left = (left[0] - 2 * left[1] + left[2]) / d ** 2
        s_right = (right[0] - 2 * right[1] + right[2]) / d ** 2
        assert abs(s_left - s_right) < 20 * d          # second derivative continuous (third jumps: O(d) difference)
    phi = 2 * np.pi * rng.random(50)
    g = f(phi)
    e = 1e-5
    fd = (f(phi + e)["dphi"] - f(phi - e)["dphi"]) / (2 * e)
    assert np.abs(g["dphi_dphi"] - fd).max() < 1e-8
    o.set_spline_coeffs(0, None)


def test_poloidal_part_is_the_pinned_element_polynomial(inputs, cfg1, oracle_cfg1, setup):
    """One plane carries the Bell expansion of real nodal values; at phi = phi_j the field is 2/3 of that polynomial (value
    and R, Z derivatives) = 2/3 of the harmonic gather's n = 0 mode (O4, pinned); a separable field factorises; locality:
    planes more than two away do not matter."""
    o, m = oracle_cfg1, setup
    rng = np.random.default_rng(3)
    n_phi = 10
    h = 2 * np.pi / n_phi
    d0 = rng.standard_normal((o.n_vert, 6))
    coef_c = o.bell_from_dofs([0], (d0 + 0j)[None])                      # harmonic field with the single mode n = 0
    ref = o.gather(m["R"], m["Z"], m["phi"])
    a = rng.standard_normal(n_phi)
    dofs = a[:, None, None] * d0[None]
    cs = o.bell_spline_from_dofs(dofs)
    assert np.abs(cs[:, 3, :] - a[3] * coef_c[:, 0, :].real).max() < 1e-12 * np.abs(coef_c).max()
    beta = BSpline.basis_element([-2, -1, 0, 1, 2], extrapolate=False)
    phi = m["phi"]
    x = (phi[:, None] - h * np.arange(n_phi)[None, :]) / h
    x = x - n_phi * np.floor(x / n_phi + 0.5)
    Nw = np.nan_to_num(beta(x))
    s = (Nw * a[None, :]).sum(axis=1)
    g = o.gather(m["R"], m["Z"], phi)
    for k in ("dphi", "dphi_dR", "dphi_dZ"):
        assert np.abs(g[k] - s * ref[k]).max() < 1e-12 * np.abs(ref[k]).max(), k
    ds = (np.nan_to_num(beta.derivative()(x)) * a[None, :]).sum(axis=1) / h
    assert np.abs(g["dphi_dphi"] - ds * ref["dphi"]).max() < 1e-11 * np.abs(ref["dphi"]).max() / h
    # locality
    j0 = np.floor(phi / h).astype(int)
    far = (np.arange(n_phi)[None, :] - j0[:, None]) % n_phi
    sel = phi[far[:, 5] == 5]                                            # plane j0 + 5 is out of reach
    c2 = cs.copy()
    pick = 0
    o.set_spline_coeffs(n_phi, cs)
    g1 = o.gather(m["R"][:1], m["Z"][:1], phi[:1])
    c2[:, (j0[0] + 5) % n_phi, :] += 7.0
    o.set_spline_coeffs(n_phi, c2)
    g2 = o.gather(m["R"][:1], m["Z"][:1], phi[:1])
    assert g1["dphi"][0] == g2["dphi"][0]
    # the right-hand side and the push run on the spline field (O6, O7 unchanged: they see the gather's four numbers)
    o.set_spline_coeffs(n_phi, 1e-3 * cs)
    mm = inputs.markers(cfg1, n=200, seed=62)
    out = o.push(mm, 0.05, 3)
    assert np.all(np.isfinite(out["R"])) and np.abs(out["w"]).max() > 0
    o.set_spline_coeffs(0, None)
