"""Pins for the oracle's particle-to-grid projection (O8; "the charge of each particle is projected onto the
basis functions", PAPER.md:249 P2G is the counterpart of G2P):
    rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p}.
What the paper and the mathematics fix without reference to the oracle's own element code: the nodal basis is a Kronecker
delta at the vertices; the element space contains every polynomial of degree <= 4 (so the moments of the marker weights
against any such polynomial are reproduced exactly from the nodal values of the polynomial); local support; linearity.
And, against the oracle's gather (O4, pinned by tests/test_oracle_gather.py): scatter is its adjoint."""
import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

from helpers import poly_dofs


@pytest.fixture(scope="module")
def sample(inputs, cfg1):
    m = inputs.markers(cfg1, n=5000, seed=31)
    rng = np.random.default_rng(32)
    m["w"] = rng.standard_normal(5000)
    return m


def test_single_marker_at_a_vertex_hits_the_value_dof_only(inputs, cfg1, oracle_cfg1):
    """Lambda_{v',d}(x_v) = delta_{vv'} delta_{d0}: a marker of weight w0 sitting exactly on vertex v at phi0 gives
    rhs[n][v][0] = w0 e^{-i n phi0} and nothing anywhere else."""
    o = oracle_cfg1
    o.set_modes([0, 1, 3])
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    for v in (1, 37, 100, 200, 256 - 32):                 # vertices of the first ring, interior rings, last interior ring
        w0, phi0 = 1.7, 0.9
        rhs = o.scatter([Rv[v]], [Zv[v]], [phi0], [w0])
        want = np.zeros_like(rhs)
        want[:, v, 0] = w0 * np.exp(-1j * np.array([0, 1, 3]) * phi0)
        assert np.abs(rhs - want).max() < 1e-12, v
    # the axis vertex
    rhs = o.scatter([Rv[0]], [Zv[0]], [0.0], [1.0])
    want = np.zeros_like(rhs); want[:, 0, 0] = 1.0
    assert np.abs(rhs - want).max() < 1e-12


def test_moments_against_polynomials_of_degree_four_are_exact(inputs, cfg1, oracle_cfg1, sample):
    """The element space contains P4 (Bell's element; pinned for O2 by test_oracle_mesh_bell.py): for a polynomial q of degree
    <= 4 with nodal values D_d q(x_v),  sum_{v,d} D_d q(x_v) rhs[n][v][d] = sum_p w_p q(x_p) e^{-i n phi_p}.  The right-hand
    side is computed here with numpy alone."""
    o = oracle_cfg1
    modes = [0, 2, 5]
    o.set_modes(modes)
    m = sample
    rhs = o.scatter(m["R"], m["Z"], m["phi"], m["w"])
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    rng = np.random.default_rng(7)
    for trial in range(4):
        C = np.zeros((5, 5))
        for i in range(5):
            for j in range(5 - i):
                C[i, j] = rng.standard_normal()
        if trial == 0:
            C[:] = 0.0; C[0, 0] = 1.0                      # partition of unity: sum_v rhs[n][v][0] = sum_p w_p e^{-i n phi_p}
        dofs = poly_dofs(C, Rv, Zv)                        # [n_vert][6] nodal values of q and its derivatives
        q = npoly.polyval2d(m["R"] - 10.0, m["Z"], C)
        for k, n in enumerate(modes):
            got = (dofs * rhs[k]).sum()
            want = (m["w"] * q * np.exp(-1j * n * m["phi"])).sum()
            scale = np.abs(m["w"] * q).sum()
            assert abs(got - want) < 1e-12 * scale, (trial, n, abs(got - want) / scale)
    # a quintic is NOT in the element space: the identity must fail (the test has teeth)
    C = np.zeros((6, 6)); C[5, 0] = 1.0; C[2, 3] = 1.0
    dofs = poly_dofs(C, Rv, Zv)
    q = npoly.polyval2d(m["R"] - 10.0, m["Z"], C)
    got = (dofs * rhs[0]).sum(); want = (m["w"] * q).sum()
    assert abs(got - want) > 1e-9 * np.abs(m["w"] * q).sum()


def test_scatter_is_the_adjoint_of_gather(inputs, cfg1, oracle_cfg1, sample):
    """sum_p w_p dphi(x_p) = Re sum_{n,v,d} Y_{n,v,d} conj(rhs[n][v][d]) for arbitrary nodal values Y (complex), with dphi
    from the oracle's own Bell expansion + gather; likewise for one mode at a time (sign of the toroidal factor)."""
    o = oracle_cfg1
    modes = [0, 1, 4]
    rng = np.random.default_rng(11)
    Y = rng.standard_normal((3, o.n_vert, 6)) + 1j * rng.standard_normal((3, o.n_vert, 6))
    m = sample
    o.bell_from_dofs(modes, Y)
    f = o.gather(m["R"], m["Z"], m["phi"])["dphi"]
    rhs = o.scatter(m["R"], m["Z"], m["phi"], m["w"])
    lhs = (m["w"] * f).sum()
    r = (Y * np.conj(rhs)).real
    # the n = 0 mode takes the real part of Y only (reading G15): Im(Y_0) must not contribute
    r0 = (Y[0].real * rhs[0].real).sum()
    total = r0 + r[1:].sum()
    assert abs(lhs - total) < 1e-12 * np.abs(m["w"] * f).sum()
    assert np.abs(rhs[0].imag).max() == 0.0
    for k in range(3):
        Yk = np.zeros_like(Y); Yk[k] = Y[k]
        o.bell_from_dofs(modes, Yk)
        fk = o.gather(m["R"], m["Z"], m["phi"])["dphi"]
        want = (m["w"] * fk).sum()
        got = (Y[k].real * rhs[k].real).sum() if k == 0 else (Y[k] * np.conj(rhs[k])).real.sum()
        assert abs(want - got) < 1e-12 * np.abs(m["w"] * fk).sum(), k


def test_linearity_local_support_and_lost_markers(inputs, cfg1, oracle_cfg1, sample):
    o = oracle_cfg1
    o.set_modes([0, 2])
    m = sample
    n = m["R"].size
    a = o.scatter(m["R"], m["Z"], m["phi"], m["w"])
    w2 = np.random.default_rng(3).standard_normal(n)
    b = o.scatter(m["R"], m["Z"], m["phi"], w2)
    c = o.scatter(m["R"], m["Z"], m["phi"], 2.0 * m["w"] - 3.0 * w2)
    assert np.abs(c - (2.0 * a - 3.0 * b)).max() < 1e-12 * np.abs(a).max()
    # halves add up
    h1 = o.scatter(m["R"][: n // 2], m["Z"][: n // 2], m["phi"][: n // 2], m["w"][: n // 2])
    h2 = o.scatter(m["R"][n // 2:], m["Z"][n // 2:], m["phi"][n // 2:], m["w"][n // 2:])
    assert np.abs(a - (h1 + h2)).max() < 1e-12 * np.abs(a).max()
    # local support: one marker touches the 18 degrees of freedom of its triangle's vertices only
    p = 17
    one = o.scatter(m["R"][p:p + 1], m["Z"][p:p + 1], m["phi"][p:p + 1], [1.0])
    t = o.locate(m["R"][p:p + 1], m["Z"][p:p + 1])[0]
    verts = set(int(v) for v in o.triangles()[t])
    touched = set(np.nonzero(np.abs(one).max(axis=(0, 2)) > 0)[0].tolist())
    assert touched and touched <= verts
    # markers outside the mesh, and markers flagged cell < 0, contribute nothing
    R = np.concatenate([m["R"][:100], [12.5, 7.0]]); Z = np.concatenate([m["Z"][:100], [0.0, 0.3]])
    phi = np.concatenate([m["phi"][:100], [0.0, 1.0]]); w = np.concatenate([m["w"][:100], [1e6, 1e6]])
    x = o.scatter(R, Z, phi, w)
    y = o.scatter(R[:100], Z[:100], phi[:100], w[:100])
    assert np.array_equal(x, y) and o.last_scatter_count == 100
    flag = np.zeros(100, dtype=np.int32); flag[::3] = -1
    z = o.scatter(R[:100], Z[:100], phi[:100], w[:100], cell=flag)
    keep = flag >= 0
    z2 = o.scatter(R[:100][keep], Z[:100][keep], phi[:100][keep], w[:100][keep])
    assert np.array_equal(z, z2)
    assert o.scatter([], [], [], []).shape == (2, o.n_vert, 6)


def test_scatter_on_the_itg_mesh_against_polynomial_moments(inputs):
    """The same P4 identity on the cfg3 mesh (non-uniform rings, 130 560 triangles) with cfg3's modes."""
    import oracle
    wl = inputs.WORKLOADS["cfg3"]
    o = oracle.from_workload(wl, inputs)
    o.set_modes(wl.modes)
    m = inputs.markers(wl, n=20000)
    w = np.random.default_rng(5).standard_normal(20000)
    rhs = o.scatter(m["R"], m["Z"], m["phi"], w)
    _, Rv, Zv = inputs.mesh_nodes(wl)
    rng = np.random.default_rng(9)
    C = np.zeros((5, 5))
    for i in range(5):
        for j in range(5 - i):
            C[i, j] = rng.standard_normal()
    dofs = poly_dofs(C, Rv, Zv)
    q = npoly.polyval2d(m["R"] - 10.0, m["Z"], C)
    for k, n in enumerate(wl.modes):
        got = (dofs * rhs[k]).sum()
        want = (w * q * np.exp(-1j * n * m["phi"])).sum()
        assert abs(got - want) < 1e-11 * np.abs(w * q).sum()
