"""Pins for the oracle's grid-to-particle gather (O4): what the
toroidal-harmonic representation fixes by itself (periodicities, linearity, d/dphi) and
an independent numpy evaluation of the element polynomial."""
import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

from helpers import local_coords, poly_dofs, poly_eval


@pytest.fixture(scope="module")
def setup(inputs, cfg1, oracle_cfg1):
    dofs = inputs.field_dofs(cfg1)
    coef = oracle_cfg1.bell_from_dofs(cfg1.modes, dofs)
    m = inputs.markers(cfg1, n=3000, seed=21)
    return dofs, coef.copy(), m


def test_gather_equals_independent_polynomial_evaluation(cfg1, oracle_cfg1, setup):
    dofs, coef, m = setup
    oracle_cfg1.set_coeffs(cfg1.modes, coef)
    out = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    g = oracle_cfg1.geom()
    f = np.zeros(m["R"].size); fR = np.zeros_like(f); fZ = np.zeros_like(f); fp = np.zeros_like(f)
    for p in range(0, m["R"].size, 7):
        t = out["cell"][p]
        xi, eta = local_coords(g[t], m["R"][p], m["Z"][p])
        for k, n in enumerate(cfg1.modes):
            E = np.exp(1j * n * m["phi"][p])
            P = poly_eval(coef[t, k], xi, eta)
            Px, Pe = poly_eval(coef[t, k], xi, eta, 1, 0), poly_eval(coef[t, k], xi, eta, 0, 1)
            f[p] += (P * E).real
            fR[p] += ((g[t, 2] * Px + g[t, 4] * Pe) * E).real
            fZ[p] += ((g[t, 3] * Px + g[t, 5] * Pe) * E).real
            fp[p] += (1j * n * P * E).real
    sel = slice(0, None, 7)
    for a, b in ((out["dphi"], f), (out["dphi_dR"], fR), (out["dphi_dZ"], fZ), (out["dphi_dphi"], fp)):
        assert np.abs(a[sel] - b[sel]).max() < 1e-13 * max(1.0, np.abs(b[sel]).max())


def test_toroidal_symmetries(inputs, cfg1, oracle_cfg1, setup):
    dofs, coef, m = setup
    # single mode n = 3: invariant under phi -> phi + 2 pi / 3; n = 0 mode: phi-independent
    amps3 = coef[:, 1:2, :]
    oracle_cfg1.set_coeffs([3], amps3)
    a = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    b = oracle_cfg1.gather(m["R"], m["Z"], m["phi"] + 2 * np.pi / 3)
    c = oracle_cfg1.gather(m["R"], m["Z"], m["phi"] + 2 * np.pi / 6)      # half period: sign flip
    for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
        s = np.abs(a[k]).max()
        assert np.abs(a[k] - b[k]).max() < 1e-12 * s
        assert np.abs(a[k] + c[k]).max() < 1e-12 * s
    oracle_cfg1.set_coeffs([0], coef[:, 0:1, :])
    a = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    b = oracle_cfg1.gather(m["R"], m["Z"], m["phi"] * 0.37 + 1.0)
    assert np.array_equal(a["dphi"], b["dphi"]) and np.all(a["dphi_dphi"] == 0.0)
    # Im of the n = 0 mode is ignored (reading G15)
    oracle_cfg1.set_coeffs([0], coef[:, 0:1, :].real.astype(np.complex128))
    c = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    assert np.array_equal(a["dphi"], c["dphi"])


def test_dphi_dphi_against_finite_difference_and_linearity(cfg1, oracle_cfg1, setup):
    dofs, coef, m = setup
    oracle_cfg1.set_coeffs([0, 7], coef)
    h = 1e-5
    a = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    p = oracle_cfg1.gather(m["R"], m["Z"], m["phi"] + h)
    q = oracle_cfg1.gather(m["R"], m["Z"], m["phi"] - h)
    fd = (p["dphi"] - q["dphi"]) / (2 * h)
    assert np.abs(fd - a["dphi_dphi"]).max() < 1e-7 * np.abs(a["dphi_dphi"]).max()
    # spatial derivatives against centred differences at points away from element edges
    g = oracle_cfg1.geom()
    b = oracle_cfg1.bary(a["cell"], m["R"], m["Z"])
    deep = b.min(axis=1) > 0.05
    hR = 1e-6
    pr = oracle_cfg1.gather(m["R"] + hR, m["Z"], m["phi"])
    qr = oracle_cfg1.gather(m["R"] - hR, m["Z"], m["phi"])
    same = deep & (pr["cell"] == a["cell"]) & (qr["cell"] == a["cell"])
    fdR = (pr["dphi"] - qr["dphi"]) / (2 * hR)
    assert same.sum() > 1000
    assert np.abs(fdR - a["dphi_dR"])[same].max() < 1e-6 * np.abs(a["dphi_dR"]).max()
    pz = oracle_cfg1.gather(m["R"], m["Z"] + hR, m["phi"])
    qz = oracle_cfg1.gather(m["R"], m["Z"] - hR, m["phi"])
    same = deep & (pz["cell"] == a["cell"]) & (qz["cell"] == a["cell"])
    fdZ = (pz["dphi"] - qz["dphi"]) / (2 * hR)
    assert np.abs(fdZ - a["dphi_dZ"])[same].max() < 1e-6 * np.abs(a["dphi_dZ"]).max()
    # linearity in the coefficients
    oracle_cfg1.set_coeffs([0, 7], 2.5 * coef)
    a2 = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    assert np.abs(a2["dphi"] - 2.5 * a["dphi"]).max() < 1e-15


def test_no_factor_two_and_real_part_convention(inputs, cfg1, oracle_cfg1):
    """A single mode with DOFs of the constant function c = 2 - 3i: dphi = Re(c e^{i n phi})."""
    _, Rv, Zv = inputs.mesh_nodes(cfg1)
    dofs = np.zeros((1, oracle_cfg1.n_vert, 6), dtype=np.complex128)
    dofs[0, :, 0] = 2.0 - 3.0j
    oracle_cfg1.bell_from_dofs([4], dofs)
    m = inputs.markers(cfg1, n=500, seed=4)
    out = oracle_cfg1.gather(m["R"], m["Z"], m["phi"])
    want = 2.0 * np.cos(4 * m["phi"]) + 3.0 * np.sin(4 * m["phi"])
    assert np.abs(out["dphi"] - want).max() < 1e-13
    assert np.abs(out["dphi_dphi"] - (-8.0 * np.sin(4 * m["phi"]) + 12.0 * np.cos(4 * m["phi"]))).max() < 1e-12
    assert np.abs(out["dphi_dR"]).max() < 1e-11 and np.abs(out["dphi_dZ"]).max() < 1e-11


def test_generator_dofs_match_finite_differences(inputs, cfg1):
    """The polar-form derivative formulas of the input generator (reading G14)."""
    amps = inputs.mode_amplitudes(cfg1)
    rng = np.random.default_rng(9)
    r = 0.2 + 0.6 * rng.random(200); th = 2 * np.pi * rng.random(200)
    R, Z = 10.0 + r * np.cos(th), r * np.sin(th)
    h = 1e-4
    F = lambda R_, Z_: inputs.analytic_field(cfg1, amps, 1, R_, Z_)
    d = F(R, Z)
    fR = (F(R + h, Z)[:, 0] - F(R - h, Z)[:, 0]) / (2 * h)
    fZ = (F(R, Z + h)[:, 0] - F(R, Z - h)[:, 0]) / (2 * h)
    fRR = (F(R + h, Z)[:, 1] - F(R - h, Z)[:, 1]) / (2 * h)
    fRZ = (F(R, Z + h)[:, 1] - F(R, Z - h)[:, 1]) / (2 * h)
    fZZ = (F(R, Z + h)[:, 2] - F(R, Z - h)[:, 2]) / (2 * h)
    for got, want in ((d[:, 1], fR), (d[:, 2], fZ), (d[:, 3], fRR), (d[:, 4], fRZ), (d[:, 5], fZZ)):
        assert np.abs(got - want).max() < 1e-6 * max(np.abs(want).max(), 1e-3)
