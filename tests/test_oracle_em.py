"""Pins for the oracle's electromagnetic right-hand side (O9) and pullback (O10;
PAPER.md:616, 1109-1128).  The component formulas A.7-A.9, A.14-A.17 are checked against the VECTOR form the paper prints
above them evaluated with numpy's cross and dot products in the right-handed (R, phi, Z) basis
 on the pinned equilibrium: a wrong sign, index or 1/R in any component fails.  Limits: dA = 0 gives the
electrostatic equations of O6 minus the parallel electric field (ideal Ohm's law); the weight rate is the directional
derivative of ln f_M at v_par = u_par - (q/m) dA^h."""
import dataclasses

import numpy as np
import pytest

import oracle


@pytest.fixture(scope="module")
def pts(cfg1):
    rng = np.random.default_rng(41)
    n = 400
    r = 0.1 + 0.8 * rng.random(n)
    th = 2 * np.pi * rng.random(n)
    return dict(R=cfg1.R0 + r * np.cos(th), Z=r * np.sin(th), u=rng.standard_normal(n), mu=rng.random(n) * 2,
                w=0.1 * rng.standard_normal(n), fld=1e-2 * rng.standard_normal((n, 3, 4)))


def _vec(e, names):
    return np.stack([e[k] for k in names], axis=-1)


def _vector_form(o, wl, p, eom_variant=0):
    """PAPER.md:1218-1227 with numpy vector algebra; components ordered (R, phi, Z)."""
    e = o.equilibrium(p["R"], p["Z"])
    R, u, mu, fld = p["R"], p["u"], p["mu"], p["fld"]
    eps, qom, rB = wl.rho0 * wl.B0 / wl.qs_over_ms, wl.qs_over_ms, wl.rho0 * wl.B0
    b = _vec(e, ("bR", "bphi", "bZ"))
    curlb = np.stack([-e["dbphi_dZ"], e["dbR_dZ"] - e["dbZ_dR"], e["dbphi_dR"] + e["bphi"] / R], axis=-1)
    gradB = np.stack([e["dBdR"], 0 * R, e["dBdZ"]], axis=-1)

    def grad(f):                                      # (d/dR, (1/R) d/dphi, d/dZ)
        return np.stack([f[:, 1], f[:, 3] / R, f[:, 2]], axis=-1)

    gPhi, gAs, gAh = grad(fld[:, 0]), grad(fld[:, 1]), grad(fld[:, 2])
    Ah = fld[:, 2, 0]
    Bsp = e["B"] + eps * u * np.einsum("ij,ij->i", b, curlb)
    lead = (e["B"] / Bsp) if eom_variant == 1 else np.ones_like(Bsp)
    b0s = lead[:, None] * b + (eps * u / Bsp)[:, None] * curlb
    bs = b0s + (rB / Bsp)[:, None] * np.cross(gAs, b)
    bxgB = np.cross(b, gradB)
    R0 = u[:, None] * b0s + (eps * mu / Bsp)[:, None] * bxgB
    u0 = -mu * np.einsum("ij,ij->i", b0s, gradB)
    gG = gPhi - u[:, None] * (gAs + gAh)
    dR = (rB / Bsp)[:, None] * np.cross(b, gG) - (qom * Ah)[:, None] * bs
    du = -qom * (np.einsum("ij,ij->i", bs - b, gPhi) - u * np.einsum("ij,ij->i", bs, gAh)) \
        - (eps * mu / Bsp) * np.einsum("ij,ij->i", bxgB, gAs)
    tot = R0 + dR
    return np.stack([tot[:, 0], tot[:, 2], tot[:, 1] / R, u0 + du], axis=-1), dR, du, e


@pytest.mark.parametrize("variant", [0, 1])
def test_components_equal_the_vector_form(inputs, cfg1, pts, variant):
    o = oracle.from_workload(cfg1, inputs, eom_variant=variant)
    got = o.rhs_point_em(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], pts["fld"])
    want, _, _, _ = _vector_form(o, cfg1, pts, variant)
    for k in range(4):
        assert np.abs(got[:, k] - want[:, k]).max() < 1e-13 * max(1.0, np.abs(want[:, k]).max()), k
    # one field at a time (a term that mixes two fields wrongly would cancel in the sum only by accident)
    for a in range(3):
        p1 = dict(pts, fld=np.zeros_like(pts["fld"]))
        p1["fld"][:, a] = pts["fld"][:, a]
        g1 = o.rhs_point_em(p1["R"], p1["Z"], p1["u"], p1["mu"], p1["w"], p1["fld"])
        w1, _, _, _ = _vector_form(o, cfg1, p1, variant)
        assert np.abs(g1[:, :4] - w1).max() < 1e-13 * max(1.0, np.abs(w1).max()), a


def test_without_vector_potential_it_is_the_electrostatic_model_under_ohms_law(inputs, cfg1, oracle_cfg1, pts):
    """dA^s = dA^h = 0: positions as in O6 (pinned by test_oracle_physics.py); the parallel acceleration is O6's plus
    (q/m) b.grad(dPhi) (the parallel electric field cancels against d_t dA^s)."""
    o = oracle_cfg1
    fld = np.zeros_like(pts["fld"]); fld[:, 0] = pts["fld"][:, 0]
    em = o.rhs_point_em(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], fld)
    es = o.rhs_point(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], fld[:, 0])
    for k in range(3):
        assert np.array_equal(em[:, k], es[:, k]) or np.abs(em[:, k] - es[:, k]).max() < 1e-15 * np.abs(es[:, k]).max()
    e = o.equilibrium(pts["R"], pts["Z"])
    bgrad = e["bR"] * fld[:, 0, 1] + e["bZ"] * fld[:, 0, 2] + e["bphi"] / pts["R"] * fld[:, 0, 3]
    assert np.abs(em[:, 3] - (es[:, 3] + cfg1.qs_over_ms * bgrad)).max() < 1e-14 * np.abs(es[:, 3]).max()
    # no field at all: the unperturbed orbit, weight at rest
    z = o.rhs_point_em(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], np.zeros_like(fld))
    z0 = o.rhs_point(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], np.zeros((pts["R"].size, 4)))
    assert np.array_equal(z[:, :4], z0[:, :4]) and np.all(z[:, 4] == 0.0)


def test_weight_rate_is_directional_derivative_of_ln_fM_at_the_physical_velocity(inputs, cfg1, oracle_cfg1, pts):
    """L = d ln f_M/dt along the perturbed velocity with v_par = u_par - (q/m) dA^h in the Maxwellian."""
    o = oracle_cfg1
    k = o.rhs_point_em(pts["R"], pts["Z"], pts["u"], pts["mu"], pts["w"], pts["fld"])
    _, dR, du, _ = _vector_form(o, cfg1, pts)
    kn, kT, Tb = cfg1.kappa_n, cfg1.kappa_T, cfg1.T
    r0 = np.hypot(pts["R"] - 10.0, pts["Z"])
    v = pts["u"] - cfg1.qs_over_ms * pts["fld"][:, 2, 0]

    def lnf(R, Z, vv):
        r = np.hypot(R - 10.0, Z)
        B = o.equilibrium(R, Z)["B"]
        T = Tb * np.exp(-kT * (r - r0))
        return -kn * (r - r0) - 1.5 * np.log(T) - (vv * vv + 2 * pts["mu"] * B) / T

    h = 1e-4
    L = (lnf(pts["R"] + h * dR[:, 0], pts["Z"] + h * dR[:, 2], v + h * du)
         - lnf(pts["R"] - h * dR[:, 0], pts["Z"] - h * dR[:, 2], v - h * du)) / (2 * h)
    want = -(1.0 - pts["w"]) * L
    assert np.abs(k[:, 4] - want).max() < 1e-7 * np.abs(want).max()


def test_full_em_rhs_gathers_three_fields(inputs, cfg1, oracle_cfg1):
    """orc_rhs_em = locate + three gathers (each the pinned O4 on its own table) + the pointwise equations."""
    o = oracle_cfg1
    rng = np.random.default_rng(43)
    modes = (0, 1, 3)
    tabs = [rng.standard_normal((3, o.n_vert, 6)) * s + 1j * rng.standard_normal((3, o.n_vert, 6)) * s for s in (1e-3, 2e-3, 5e-4)]
    cPhi = o.bell_from_dofs(modes, tabs[0])
    cAs = o.bell_from_dofs(modes, tabs[1]); cAh = o.bell_from_dofs(modes, tabs[2])
    m = inputs.markers(cfg1, n=2000, seed=44)
    m["R"][::97] = 12.0                                # outside
    u = m["vpar"]
    flds = []
    for c in (cPhi, cAs, cAh):
        o.set_coeffs(modes, c)
        g = o.gather(m["R"], m["Z"], m["phi"])
        flds.append(np.stack([g["dphi"], g["dphi_dR"], g["dphi_dZ"], g["dphi_dphi"]], axis=-1))
    cell = g["cell"]
    o.set_coeffs(modes, cPhi); o.set_aux_coeffs(0, cAs); o.set_aux_coeffs(1, cAh)
    got = o.rhs_em(m["R"], m["Z"], m["phi"], u, m["mu"], m["w"])
    want = o.rhs_point_em(m["R"], m["Z"], u, m["mu"], m["w"], np.stack(flds, axis=1))
    assert np.array_equal(got["cell"], cell)
    ins = cell >= 0
    for k, name in enumerate(("dRdt", "dZdt", "dphidt", "dudt", "dwdt")):
        assert np.array_equal(got[name][ins], want[ins, k]), name
        assert np.all(got[name][~ins] == 0.0)
    # aux tables absent = zero fields
    o.set_aux_coeffs(0, None); o.set_aux_coeffs(1, None)
    g0 = o.rhs_em(m["R"], m["Z"], m["phi"], u, m["mu"], m["w"])
    f0 = np.stack([flds[0], 0 * flds[0], 0 * flds[0]], axis=1)
    w0 = o.rhs_point_em(m["R"], m["Z"], u, m["mu"], m["w"], f0)
    assert np.array_equal(g0["dudt"][ins], w0[ins, 3])


def test_pullback(inputs, cfg1):
    """u_new = u_old - (q/m) dA^h; the weight changes by the first-order change of f_M under v -> v + (q/m) dA^h
    (PAPER.md:1112-1128): checked against the Maxwellian itself; dA^h = 0 is a no-op; markers outside stay untouched."""
    wl = dataclasses.replace(cfg1, qs_over_ms=-1.0 * 1.5)          # a species with q/m != 1, and negative
    o = oracle.from_workload(wl, inputs)
    rng = np.random.default_rng(45)
    modes = (0, 2)
    amp = 1e-5
    dofs = amp * (rng.standard_normal((2, o.n_vert, 6)) + 1j * rng.standard_normal((2, o.n_vert, 6)))
    cAh = o.bell_from_dofs(modes, dofs)
    m = inputs.markers(wl, n=3000, seed=46)
    m["R"][::101] = 7.5
    w0 = 0.2 * rng.standard_normal(3000)
    o.set_coeffs(modes, cAh)
    Ah = o.gather(m["R"], m["Z"], m["phi"])
    cell, Ah = Ah["cell"], Ah["dphi"]
    o.set_coeffs(modes, 0 * cAh); o.set_aux_coeffs(1, cAh)
    un, wn = o.pullback(m["R"], m["Z"], m["phi"], m["vpar"], w0)
    ins = cell >= 0
    qom = wl.qs_over_ms
    assert np.array_equal(un[ins], (m["vpar"] - qom * Ah)[ins])
    assert np.array_equal(un[~ins], m["vpar"][~ins]) and np.array_equal(wn[~ins], w0[~ins]) and (~ins).sum() > 10
    # delta f_new - delta f_old = f_M(v + (q/m) A) - f_M(v) to first order, per unit f = f_0 / (1 - w)
    fM = lambda v: np.exp(-v * v / wl.T)
    v = un
    rel = (fM(v + qom * Ah) - fM(v)) / fM(v)
    want = w0 + rel * (1.0 - w0)
    assert np.abs(wn - want)[ins].max() < 50 * (amp * 10) ** 2          # second order in the amplitude
    assert np.abs(wn - w0)[ins].max() > 1e-6                            # and it did something
    # linear weights
    ol = oracle.from_workload(wl, inputs, weight_mode=1)
    ol.set_coeffs(modes, 0 * cAh); ol.set_aux_coeffs(1, cAh)
    _, wl_ = ol.pullback(m["R"], m["Z"], m["phi"], m["vpar"], w0)
    assert np.abs(wl_ - (w0 + rel))[ins].max() < 50 * (amp * 10) ** 2
    # no dA^h: nothing happens
    o.set_aux_coeffs(1, None)
    u2, w2 = o.pullback(m["R"], m["Z"], m["phi"], m["vpar"], w0)
    assert np.array_equal(u2, m["vpar"]) and np.array_equal(w2, w0)
    # flagged markers are skipped
    o.set_aux_coeffs(1, cAh)
    flag = np.zeros(3000, dtype=np.int32); flag[::5] = -1
    u3, w3 = o.pullback(m["R"], m["Z"], m["phi"], m["vpar"], w0, cell=flag)
    assert np.array_equal(u3[::5], m["vpar"][::5]) and np.array_equal(u3[1::5], un[1::5])
