"""Pins for the oracle's equilibrium (O5), right-hand side (O6) and RK4 (O7).

Expected values come from what the paper and the mathematics fix:
* B = grad psi x grad phi + F grad phi, B_R = -psi_Z/R, B_Z = psi_R/R, B_phi = F/R
   -> finite differences of psi, div B = 0, R B_phi = const;
* the vector form of the equations of motion conserves the energy
  v_par^2/2 + mu B (+ (q/m) dphi for a static potential) pointwise -> pins every sign of
  A.10-A.17 and the reading G1 (A.11's sign);
* canonical toroidal momentum P_phi = psi + eps v_par R b_phi (axisymmetry) for the
  Hamiltonian-consistent variant (reading G2);
* d ln f_M/dt is the directional derivative of ln f_M of PAPER.md:1204;
* classic RK4 has global order 4; field-line following has the textbook safety factor."""
import dataclasses
import math

import numpy as np
import pytest

import oracle

EPS = 1.0 / 60.0       # (m/q) rho0 B0 in all workloads (G9)


@pytest.fixture(scope="module")
def pts(inputs, cfg1):
    m = inputs.markers(cfg1, n=4000, seed=31)
    rng = np.random.default_rng(32)
    m["w"] = 0.3 * rng.standard_normal(m["R"].size)
    return m


def test_equilibrium_against_definition(oracle_cfg1, pts):
    R, Z = pts["R"], pts["Z"]
    e = oracle_cfg1.equilibrium(R, Z)
    h = 1e-5
    psiR = (oracle_cfg1.equilibrium(R + h, Z)["psi"] - oracle_cfg1.equilibrium(R - h, Z)["psi"]) / (2 * h)
    psiZ = (oracle_cfg1.equilibrium(R, Z + h)["psi"] - oracle_cfg1.equilibrium(R, Z - h)["psi"]) / (2 * h)
    assert np.abs(e["BR"] + psiZ / R).max() < 1e-9           # B_R = -psi_Z / R
    assert np.abs(e["BZ"] - psiR / R).max() < 1e-9           # B_Z = +psi_R / R
    assert np.abs(e["Bphi"] * R - 10.0).max() < 1e-13        # B_phi = F / R, F = B0 R0
    B = np.sqrt(e["BR"] ** 2 + e["BZ"] ** 2 + e["Bphi"] ** 2)
    assert np.abs(e["B"] - B).max() < 1e-14
    for k, K in (("bR", "BR"), ("bZ", "BZ"), ("bphi", "Bphi")):
        assert np.abs(e[k] - e[K] / B).max() < 1e-14
    # cylindrical safety factor of the configs: q = r B_phi / (R0 B_pol)
    r = np.hypot(R - 10.0, Z)
    q = r * e["Bphi"] / (10.0 * np.hypot(e["BR"], e["BZ"]))
    assert np.abs(q - (1.4 + 2.0 * r ** 2)).max() < 1e-12
    # poloidal field direction: counter-clockwise for B0 > 0 (psi increasing outward)
    assert np.all(e["BR"] * (-Z) + e["BZ"] * (R - 10.0) > 0)


def test_equilibrium_derivatives_and_divergence(oracle_cfg1, pts):
    R, Z = pts["R"], pts["Z"]
    e = oracle_cfg1.equilibrium(R, Z)
    h = 1e-5
    eRp, eRm = oracle_cfg1.equilibrium(R + h, Z), oracle_cfg1.equilibrium(R - h, Z)
    eZp, eZm = oracle_cfg1.equilibrium(R, Z + h), oracle_cfg1.equilibrium(R, Z - h)
    dR = lambda k: (eRp[k] - eRm[k]) / (2 * h)
    dZ = lambda k: (eZp[k] - eZm[k]) / (2 * h)
    assert np.abs(e["dBdR"] - dR("B")).max() < 1e-9
    assert np.abs(e["dBdZ"] - dZ("B")).max() < 1e-9
    assert np.abs(e["dbR_dZ"] - dZ("bR")).max() < 1e-9
    assert np.abs(e["dbZ_dR"] - dR("bZ")).max() < 1e-9
    assert np.abs(e["dbphi_dR"] - dR("bphi")).max() < 1e-9
    assert np.abs(e["dbphi_dZ"] - dZ("bphi")).max() < 1e-9
    divB = ((R + h) * eRp["BR"] - (R - h) * eRm["BR"]) / (2 * h) / R + dZ("BZ")
    assert np.abs(divB).max() < 1e-9


def _rhs(o, m, fld):
    return o.rhs_point(m["R"], m["Z"], m["vpar"], m["mu"], m["w"], fld)


def test_unperturbed_energy_identity_pins_a11_sign(oracle_cfg1, pts):
    """v_par dv_par/dt + mu (Rdot dB/dR + Zdot dB/dZ) = 0 pointwise (G1: A.11 needs '-')."""
    e = oracle_cfg1.equilibrium(pts["R"], pts["Z"])
    k = _rhs(oracle_cfg1, pts, np.zeros((pts["R"].size, 4)))
    res = pts["vpar"] * k[:, 3] + pts["mu"] * (k[:, 0] * e["dBdR"] + k[:, 1] * e["dBdZ"])
    scale = np.abs(pts["vpar"] * k[:, 3]) + np.abs(pts["mu"] * k[:, 0] * e["dBdR"]) + 1e-30
    assert (np.abs(res) / scale).max() < 1e-12
    # the drift terms matter in this identity: with A.11's printed '+' it is O(1e-7..1e-6)
    Cd_term = EPS * pts["mu"] / (e["B"] ** 2) * e["Bphi"] * e["dBdR"]      # ~ magnitude of the flipped term
    wrong = res + pts["mu"] * (2 * Cd_term) * e["dBdZ"]
    assert np.abs(wrong).max() > 1e-9
    assert np.all(k[:, 4] == 0.0)                                          # no field -> wdot = 0 exactly


def test_canonical_momentum(inputs, cfg1, oracle_cfg1, pts):
    """P_phi = psi + eps v_par R b_phi.  Variant 1 (Hamiltonian-consistent b0*) conserves it
    pointwise; variant 0 (as printed, A.4-A.6) has the residual of reading G2."""
    e = oracle_cfg1.equilibrium(pts["R"], pts["Z"])
    R, v, mu = pts["R"], pts["vpar"], pts["mu"]
    dP_dR = R * e["BZ"] + EPS * v * (e["bphi"] + R * e["dbphi_dR"])
    dP_dZ = -R * e["BR"] + EPS * v * R * e["dbphi_dZ"]
    dP_dv = EPS * R * e["bphi"]
    zero = np.zeros((R.size, 4))
    o1 = oracle.from_workload(cfg1, inputs, eom_variant=1)
    k = _rhs(o1, pts, zero)
    res = k[:, 0] * dP_dR + k[:, 1] * dP_dZ + k[:, 3] * dP_dv
    scale = np.abs(k[:, 0] * dP_dR) + np.abs(k[:, 1] * dP_dZ) + np.abs(k[:, 3] * dP_dv)
    assert (np.abs(res) / scale).max() < 1e-11
    # variant 0: dP_phi/dt = -lambda eps (F/B) (b.grad B) (mu + v^2/B), lambda = eps v b.curl b / B*par
    k0 = _rhs(oracle_cfg1, pts, zero)
    res0 = k0[:, 0] * dP_dR + k0[:, 1] * dP_dZ + k0[:, 3] * dP_dv
    curl_R, curl_Z = -e["dbphi_dZ"], e["dbphi_dR"] + e["bphi"] / R
    curl_P = e["dbR_dZ"] - e["dbZ_dR"]
    bcb = e["bR"] * curl_R + e["bZ"] * curl_Z + e["bphi"] * curl_P
    Bsp = e["B"] + EPS * v * bcb
    lam = EPS * v * bcb / Bsp
    pred = -lam * EPS * (10.0 / e["B"]) * (e["bR"] * e["dBdR"] + e["bZ"] * e["dBdZ"]) * (mu + v * v / e["B"])
    assert np.abs(res0 - pred).max() < 1e-10 * np.abs(pred).max()
    assert np.abs(pred).max() > 1e-9


def test_perturbed_energy_identity_pins_a14_to_a17(oracle_cfg1, pts):
    """E_tot = v^2/2 + mu B + (q/m) dphi with a static dphi: dE_tot/dt = 0 pointwise, for ANY
    gradient values (dphi_R, dphi_Z, dphi_phi) -> signs of A.14-A.17 and C_E (G3)."""
    rng = np.random.default_rng(33)
    n = pts["R"].size
    fld = 1e-2 * rng.standard_normal((n, 4))
    e = oracle_cfg1.equilibrium(pts["R"], pts["Z"])
    k = _rhs(oracle_cfg1, pts, fld)
    terms = [pts["vpar"] * k[:, 3], pts["mu"] * k[:, 0] * e["dBdR"], pts["mu"] * k[:, 1] * e["dBdZ"],
             k[:, 0] * fld[:, 1], k[:, 1] * fld[:, 2], k[:, 2] * fld[:, 3]]
    res = sum(terms)
    scale = sum(np.abs(t) for t in terms)
    assert (np.abs(res) / scale).max() < 1e-12
    # E x B drift is perpendicular to grad(dphi) and to b: (dR, dZ, R dphi) . grad = 0
    k0 = _rhs(oracle_cfg1, pts, np.zeros((n, 4)))
    d = k - k0
    perp = d[:, 0] * fld[:, 1] + d[:, 1] * fld[:, 2] + d[:, 2] * fld[:, 3]
    sc = np.abs(d[:, 0] * fld[:, 1]) + np.abs(d[:, 1] * fld[:, 2]) + np.abs(d[:, 2] * fld[:, 3])
    assert (np.abs(perp) / sc).max() < 1e-8      # d = k - k0 loses digits
    along_b = d[:, 0] * e["bR"] + d[:, 1] * e["bZ"] + pts["R"] * d[:, 2] * e["bphi"]
    sc = np.abs(d[:, 0] * e["bR"]) + np.abs(d[:, 1] * e["bZ"]) + np.abs(pts["R"] * d[:, 2] * e["bphi"])
    assert (np.abs(along_b) / sc).max() < 1e-8
    # magnitude: |v_E| = |b x grad dphi| rho0 B0 / B*par
    g = np.stack([fld[:, 1], fld[:, 3] / pts["R"], fld[:, 2]], axis=1)          # (R, phi, Z)
    b = np.stack([e["bR"], e["bphi"], e["bZ"]], axis=1)
    vE = np.stack([d[:, 0], pts["R"] * d[:, 2], d[:, 1]], axis=1)
    cr = np.cross(b, g)                                                          # right-handed (R, phi, Z)
    curl_R, curl_Z = -e["dbphi_dZ"], e["dbphi_dR"] + e["bphi"] / pts["R"]
    bcb = e["bR"] * curl_R + e["bZ"] * curl_Z + e["bphi"] * (e["dbR_dZ"] - e["dbZ_dR"])
    Bsp = e["B"] + EPS * pts["vpar"] * bcb
    assert np.abs(vE - cr * (EPS / Bsp)[:, None]).max() < 1e-14


def test_weight_rate_is_directional_derivative_of_ln_fM(inputs, cfg1, oracle_cfg1, pts):
    """L = d ln f_M/dt along the PERTURBED velocity for
    f_M = n0(r) / T(r)^{3/2} exp(-(v^2 + 2 mu B)/T(r)),  n0 = exp(-kappa_n (r - r_p)),
    T = Tbar exp(-kappa_T (r - r_p)) (readings G6, G10); wdot = -(1 - w) L (G7)."""
    rng = np.random.default_rng(34)
    n = pts["R"].size
    fld = 1e-2 * rng.standard_normal((n, 4))
    k = _rhs(oracle_cfg1, pts, fld)
    k0 = _rhs(oracle_cfg1, pts, np.zeros((n, 4)))
    d = k - k0                                      # (dRdot, dZdot, dphidot, dvdot, .)
    kn, kT, Tb = cfg1.kappa_n, cfg1.kappa_T, cfg1.T
    r0 = np.hypot(pts["R"] - 10.0, pts["Z"])

    def lnf(R, Z, v):
        r = np.hypot(R - 10.0, Z)
        B = oracle_cfg1.equilibrium(R, Z)["B"]
        T = Tb * np.exp(-kT * (r - r0))
        return -kn * (r - r0) - 1.5 * np.log(T) - (v * v + 2 * pts["mu"] * B) / T

    h = 1e-4
    L = (lnf(pts["R"] + h * d[:, 0], pts["Z"] + h * d[:, 1], pts["vpar"] + h * d[:, 3])
         - lnf(pts["R"] - h * d[:, 0], pts["Z"] - h * d[:, 1], pts["vpar"] - h * d[:, 3])) / (2 * h)
    want = -(1.0 - pts["w"]) * L
    assert np.abs(k[:, 4] - want).max() < 1e-7 * np.abs(want).max()
    # linear option
    o_lin = oracle.from_workload(cfg1, inputs, weight_mode=1)
    kl = _rhs(o_lin, pts, fld)
    assert np.abs(kl[:, 4] + L).max() < 1e-7 * np.abs(L).max()


def test_weight_rate_without_gradients_is_kinetic_energy_rate(inputs, cfg1, pts):
    """kappa_n = kappa_T = 0: L = -(2/Tbar) d(v^2/2 + mu B)/dt exactly."""
    wl = dataclasses.replace(cfg1, kappa_n=0.0, kappa_T=0.0)
    o = oracle.from_workload(wl, inputs)
    rng = np.random.default_rng(35)
    n = pts["R"].size
    fld = 1e-2 * rng.standard_normal((n, 4))
    e = o.equilibrium(pts["R"], pts["Z"])
    k = _rhs(o, pts, fld)
    dK = pts["vpar"] * k[:, 3] + pts["mu"] * (k[:, 0] * e["dBdR"] + k[:, 1] * e["dBdZ"])
    want = (1.0 - pts["w"]) * (2.0 / wl.T) * dK
    assert np.abs(k[:, 4] - want).max() < 1e-12 * np.abs(want).max()


# ------------------------------------------------------------------- RK4 -----
def _markers(inputs, cfg1, n, seed):
    m = inputs.markers(cfg1, n=n, seed=seed)
    # keep orbits well inside the mesh for the long integrations
    r = np.hypot(m["R"] - 10.0, m["Z"])
    th = np.arctan2(m["Z"], m["R"] - 10.0)
    r = 0.25 + 0.5 * (r - 0.1) / 0.8
    m["R"], m["Z"] = 10.0 + r * np.cos(th), r * np.sin(th)
    return m


def test_rk4_order_four(inputs, cfg1, oracle_cfg1):
    """dphi = 0 (smooth RHS): error ratio ~16 per halving of dt (SURVEY.md §8(c) RK4 pin)."""
    oracle_cfg1.set_modes([])
    m = _markers(inputs, cfg1, 64, 41)
    T = 8.0
    ref = oracle_cfg1.push(m, T / 4096, 4096)
    assert np.all(ref["cell"] >= 0)
    errs = []
    for ns in (20, 40, 80):
        out = oracle_cfg1.push(m, T / ns, ns)
        errs.append(max(np.abs(out[k] - ref[k]).max() for k in ("R", "Z", "vpar")))
    assert 12.0 < errs[0] / errs[1] < 20.0, errs
    assert 12.0 < errs[1] / errs[2] < 20.0, errs


def test_push_conserves_energy_mu_and_weights_without_field(inputs, cfg1, oracle_cfg1):
    oracle_cfg1.set_modes([])
    m = _markers(inputs, cfg1, 500, 42)
    m["w"] = np.random.default_rng(1).standard_normal(500) * 1e-2
    out = oracle_cfg1.push(m, 0.05, 160)
    assert np.all(out["cell"] >= 0)
    E0 = 0.5 * m["vpar"] ** 2 + m["mu"] * oracle_cfg1.equilibrium(m["R"], m["Z"])["B"]
    E1 = 0.5 * out["vpar"] ** 2 + out["mu"] * oracle_cfg1.equilibrium(out["R"], out["Z"])["B"]
    assert (np.abs(E1 - E0) / E0).max() < 1e-11
    assert np.array_equal(out["mu"], m["mu"])          # magnetic moment: bit-identical
    assert np.array_equal(out["w"], m["w"])            # dphi = 0 -> wdot = 0 exactly
    assert np.array_equal(out["cell"], oracle_cfg1.locate(out["R"], out["Z"]))
    assert out["phi"].min() >= 0.0 and out["phi"].max() < 2 * np.pi


def test_push_conserves_canonical_momentum_variant1(inputs, cfg1):
    o = oracle.from_workload(cfg1, inputs, eom_variant=1)
    o.set_modes([])
    m = _markers(inputs, cfg1, 300, 43)
    def Pphi(mm):
        e = o.equilibrium(mm["R"], mm["Z"])
        return e["psi"] + EPS * mm["vpar"] * mm["R"] * e["bphi"]
    out = o.push(m, 0.05, 160)
    assert np.abs(Pphi(out) - Pphi(m)).max() < 1e-11
    # variant 0 (as printed): secular drift ~1e-5 over t = 8 (reading G2), far above truncation
    o0 = oracle.from_workload(cfg1, inputs, eom_variant=0)
    o0.set_modes([])
    out0 = o0.push(m, 0.05, 160)
    assert 1e-7 < np.abs(Pphi(out0) - Pphi(m)).max() < 1e-3


def test_total_energy_with_static_field(inputs, cfg1, oracle_cfg1):
    """E_tot = v^2/2 + mu B + dphi is conserved to truncation order with the C1 field."""
    dofs = inputs.field_dofs(cfg1)
    oracle_cfg1.bell_from_dofs(cfg1.modes, dofs)
    m = _markers(inputs, cfg1, 400, 44)
    def Etot(mm):
        return 0.5 * mm["vpar"] ** 2 + mm["mu"] * oracle_cfg1.equilibrium(mm["R"], mm["Z"])["B"] + \
            oracle_cfg1.gather(mm["R"], mm["Z"], mm["phi"])["dphi"]
    e0 = Etot(m)
    d1 = np.abs(Etot(oracle_cfg1.push(m, 0.1, 20)) - e0).max()
    d2 = np.abs(Etot(oracle_cfg1.push(m, 0.05, 40)) - e0).max()
    assert d2 < 2e-9 and d2 < d1
    # and the kinetic part alone is NOT conserved (the field does work)
    out = oracle_cfg1.push(m, 0.05, 40)
    K = lambda mm: 0.5 * mm["vpar"] ** 2 + mm["mu"] * oracle_cfg1.equilibrium(mm["R"], mm["Z"])["B"]
    assert np.abs(K(out) - K(m)).max() > 1e-6


def test_weight_invariant_without_profile_gradients(inputs, cfg1):
    """kappa = 0, mode 0: (1 - w) exp((v^2 + 2 mu B)/Tbar) is constant along perturbed orbits;
    mode 1: w - (v^2 + 2 mu B)/Tbar is."""
    wl = dataclasses.replace(cfg1, kappa_n=0.0, kappa_T=0.0)
    dofs = 30.0 * inputs.field_dofs(wl)
    m = _markers(inputs, wl, 300, 45)
    m["w"] = np.random.default_rng(2).standard_normal(300) * 1e-2
    for mode in (0, 1):
        o = oracle.from_workload(wl, inputs, weight_mode=mode)
        o.bell_from_dofs(wl.modes, dofs)
        def inv(mm):
            en = (mm["vpar"] ** 2 + 2 * mm["mu"] * o.equilibrium(mm["R"], mm["Z"])["B"]) / wl.T
            return (1 - mm["w"]) * np.exp(en) if mode == 0 else mm["w"] - en
        i0 = inv(m)
        errs = [np.abs(inv(o.push(m, dt, ns)) / i0 - 1).max() if mode == 0 else
                np.abs(inv(o.push(m, dt, ns)) - i0).max() for dt, ns in ((0.1, 20), (0.05, 40))]
        assert errs[1] < 1e-8 and errs[1] < errs[0], (mode, errs)
        out = o.push(m, 0.05, 40)
        assert np.abs(out["w"] - m["w"]).max() > 1e-5          # weights really moved


def test_field_line_following_gives_the_safety_factor(inputs, cfg1):
    """rho0 -> 0, mu = 0: guiding centres follow field lines; r stays constant and one
    poloidal turn advances phi by 2 pi q / sqrt(1 - r^2/R0^2) (textbook, circular flux surfaces)."""
    wl = dataclasses.replace(cfg1, rho0=0.0)
    o = oracle.from_workload(wl, inputs)
    o.set_modes([])
    r = np.array([0.3, 0.5, 0.7])
    m = dict(R=10.0 + r, Z=np.zeros(3), phi=np.zeros(3), vpar=np.ones(3), mu=np.zeros(3), w=np.zeros(3))
    qb = 1.4 + 2.0 * r * r
    h = 1.0 / (qb * np.sqrt(100.0 + r * r / qb ** 2))        # theta_dot = v_par h
    for k in range(3):
        Tpol = 2 * np.pi / h[k]
        ns = 4000
        mk = {key: v[k:k + 1] for key, v in m.items()}
        out = o.push(mk, Tpol / ns, ns)
        assert abs(np.hypot(out["R"][0] - 10.0, out["Z"][0]) - r[k]) < 1e-11
        assert abs(out["Z"][0]) < 1e-9 and out["R"][0] > 10.0                   # back at theta = 0
        want = (2 * np.pi * qb[k] / math.sqrt(1 - (r[k] / 10.0) ** 2)) % (2 * np.pi)
        assert abs(out["phi"][0] - want) < 1e-9


def test_lost_markers_are_flagged_restored_and_skipped(inputs, cfg1, oracle_cfg1):
    oracle_cfg1.set_modes([])
    # start just inside the boundary with outward grad-B drift (drift is vertical): use large mu
    th = np.linspace(0, 2 * np.pi, 64, endpoint=False)
    r = 0.995 * math.cos(math.pi / 32)
    m = dict(R=10.0 + r * np.cos(th), Z=r * np.sin(th), phi=np.zeros(64), vpar=0.3 * np.ones(64),
             mu=400.0 * np.ones(64), w=np.zeros(64))
    c0 = oracle_cfg1.locate(m["R"], m["Z"])
    assert np.all(c0 >= 0)
    out = oracle_cfg1.push(m, 0.05, 40)
    lost = out["cell"] < 0
    assert 5 < lost.sum() < 60
    # a lost marker keeps a state from which one more step leaves the mesh, and is inside itself
    assert np.all(oracle_cfg1.locate(out["R"][lost], out["Z"][lost]) >= 0)
    again = oracle_cfg1.push({k: out[k] for k in m}, 0.05, 1)
    assert np.all(again["cell"][lost] < 0)
    # pushing the flagged set again does not move it (skipped from then on)
    out2 = oracle_cfg1.push({k: out[k] for k in m}, 0.05, 5, cell=out["cell"])
    for k in ("R", "Z", "phi", "vpar", "w"):
        assert np.array_equal(out2[k][lost], out[k][lost])
