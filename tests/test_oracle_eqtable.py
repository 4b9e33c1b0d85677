"""Pins for the oracle's tabulated equilibrium (O14; "the magnetic equilibrium constructed from the EQDSK output
file ... b-spline interpolation of the poloidal current function F"; PAPER.md:1156-1164 B = grad psi x grad phi + F grad phi;
reading G32: uniform cubic B-spline tables of psi(R, Z) and F(psi), coefficients handed in).  What fixes it:
  * psi, its first and second derivatives, F and F' against scipy.interpolate.BSpline on the same knots and coefficients, and
    every derived field (B, b, grad B, the derivatives of b) against the quotient rule written with numpy on those;
  * the table of the circular equilibrium converges to the analytic one (O5, pinned by test_oracle_physics.py): psi as h^4,
    B_R, B_Z as h^3, second-derivative quantities as h^2;
  * canonical toroidal momentum P_phi = psi + eps v R b_phi is conserved pointwise by the Hamiltonian-consistent variant in an
    ELONGATED table with F' != 0 (signs of B_R, B_Z, of the derivatives of b and of the F' terms), energy by every variant;
  * the profile gradients act along grad psi: the weight rate is the directional derivative of ln f_M(psi);
  * pushes in the tabulated circular equilibrium approach the analytic-equilibrium pushes as the table is refined."""
import numpy as np
import pytest
from scipy.interpolate import BSpline

import oracle

EPS = 1.0 / 60.0


@pytest.fixture(scope="module")
def pts(cfg1):
    rng = np.random.default_rng(61)
    n = 300
    r = 0.05 + 0.9 * rng.random(n)
    th = 2 * np.pi * rng.random(n)
    return dict(R=cfg1.R0 + r * np.cos(th), Z=r * np.sin(th), vpar=rng.standard_normal(n), mu=rng.random(n) * 2,
                w=0.1 * rng.standard_normal(n))


def _scipy_fields(tab, R, Z):
    """psi and derivatives, F, F' from scipy's B-splines; then B, b, grad B, db by the quotient rule."""
    C, D = tab["C"], tab["D"]
    nR, nZ = C.shape
    tR = tab["Ra"] + tab["hR"] * (np.arange(nR + 4) - 2.0)
    tZ = tab["Za"] + tab["hZ"] * (np.arange(nZ + 4) - 2.0)
    tF = tab["pa"] + tab["hp"] * (np.arange(D.size + 4) - 2.0)
    bR = BSpline(tR, np.eye(nR), 3)
    bZ = BSpline(tZ, np.eye(nZ), 3)

    def ev(a, b):
        MR = (bR.derivative(a) if a else bR)(R)                   # [n][nR]
        MZ = (bZ.derivative(b) if b else bZ)(Z)
        return np.einsum("pi,ij,pj->p", MR, C, MZ)

    psi, pR, pZ, pRR, pRZ, pZZ = ev(0, 0), ev(1, 0), ev(0, 1), ev(2, 0), ev(1, 1), ev(0, 2)
    sF = BSpline(tF, D, 3)
    F, Fp = sF(psi), sF.derivative(1)(psi)
    BR, BZ, BP = -pZ / R, pR / R, F / R
    BR_R, BR_Z = -pRZ / R + pZ / R ** 2, -pZZ / R
    BZ_R, BZ_Z = pRR / R - pR / R ** 2, pRZ / R
    BP_R, BP_Z = Fp * pR / R - F / R ** 2, Fp * pZ / R
    B = np.sqrt(BR ** 2 + BZ ** 2 + BP ** 2)
    B_R = (BR * BR_R + BZ * BZ_R + BP * BP_R) / B
    B_Z = (BR * BR_Z + BZ * BZ_Z + BP * BP_Z) / B
    return dict(psi=psi, B=B, BR=BR, BZ=BZ, Bphi=BP, bR=BR / B, bZ=BZ / B, bphi=BP / B, dBdR=B_R, dBdZ=B_Z,
                dbR_dZ=(BR_Z - BR / B * B_Z) / B, dbZ_dR=(BZ_R - BZ / B * B_R) / B,
                dbphi_dR=(BP_R - BP / B * B_R) / B, dbphi_dZ=(BP_Z - BP / B * B_Z) / B, psiR=pR, psiZ=pZ)


@pytest.mark.parametrize("kappa,f1", [(1.0, 0.0), (1.4, 0.3)])
def test_fields_against_scipy_bsplines(inputs, cfg1, pts, kappa, f1):
    tab = inputs.equilibrium_table(cfg1, 41, 49, 13, kappa=kappa, f1=f1)
    o = oracle.from_workload(cfg1, inputs)
    o.set_equilibrium_table(tab)
    got = o.equilibrium(pts["R"], pts["Z"])
    want = _scipy_fields(tab, pts["R"], pts["Z"])
    for k in oracle.EQ_FIELDS:
        # absolute: the fields are O(1) combinations of O(1) terms (grad B on the midplane is a cancellation)
        assert np.abs(got[k] - want[k]).max() < 1e-13, (k, np.abs(got[k] - want[k]).max())
    if f1:
        assert np.abs(want["Bphi"] * pts["R"] - cfg1.B0 * cfg1.R0).max() > 1e-4      # F really varies
    # back to the analytic equilibrium
    o.set_equilibrium_table(None)
    assert np.array_equal(o.equilibrium(pts["R"], pts["Z"])["B"], oracle.from_workload(cfg1, inputs).equilibrium(pts["R"], pts["Z"])["B"])


def test_circular_table_converges_to_the_analytic_equilibrium(inputs, cfg1, pts):
    o = oracle.from_workload(cfg1, inputs)
    ea = o.equilibrium(pts["R"], pts["Z"])
    err = {}
    for N in (33, 65, 129):
        o.set_equilibrium_table(inputs.equilibrium_table(cfg1, N, N))
        et = o.equilibrium(pts["R"], pts["Z"])
        err[N] = {k: np.abs(et[k] - ea[k]).max() for k in oracle.EQ_FIELDS}
    for k, lo in (("psi", 12.0), ("BR", 6.0), ("BZ", 6.0), ("dBdR", 3.0), ("dbR_dZ", 3.0), ("dbphi_dZ", 3.0)):
        assert err[33][k] / err[65][k] > lo and err[65][k] / err[129][k] > lo, (k, err[33][k], err[65][k], err[129][k])
    assert err[129]["B"] < 1e-9 and err[129]["BR"] < 1e-7 and err[129]["dbR_dZ"] < 1e-4


def test_momentum_and_energy_identities_in_an_elongated_table(inputs, cfg1, pts):
    tab = inputs.equilibrium_table(cfg1, 65, 65, 17, kappa=1.4, f1=0.3)
    zero = np.zeros((pts["R"].size, 4))
    R, v, mu = pts["R"], pts["vpar"], pts["mu"]
    for variant in (0, 1, 2):
        o = oracle.from_workload(cfg1, inputs, eom_variant=variant)
        o.set_equilibrium_table(tab)
        e = o.equilibrium(R, pts["Z"])
        k = o.rhs_point(R, pts["Z"], v, mu, pts["w"], zero)
        dE = v * k[:, 3] + mu * (k[:, 0] * e["dBdR"] + k[:, 1] * e["dBdZ"])
        assert np.abs(dE).max() < 1e-14 * max(1.0, np.abs(v * k[:, 3]).max())          # every variant, any table
        if variant == 0:
            acc0 = k[:, 3]
        if variant == 2:
            # reading G29 matters here: with F' != 0 the mirror force along b0* (A.13, and A.22 as printed) is not the one along b
            assert np.abs(k[:, 3] - acc0).max() > 1e-7
        if variant == 1:
            s = _scipy_fields(tab, R, pts["Z"])                    # grad psi from scipy, not from the oracle
            dP_dR = s["psiR"] + EPS * v * (e["bphi"] + R * e["dbphi_dR"])
            dP_dZ = s["psiZ"] + EPS * v * R * e["dbphi_dZ"]
            dP_dv = EPS * R * e["bphi"]
            res = k[:, 0] * dP_dR + k[:, 1] * dP_dZ + k[:, 3] * dP_dv
            scale = np.abs(k[:, 0] * dP_dR) + np.abs(k[:, 1] * dP_dZ) + np.abs(k[:, 3] * dP_dv)
            assert (np.abs(res) / scale).max() < 1e-11


def test_weight_rate_follows_grad_psi(inputs, cfg1, pts):
    """ln f_M = -kappa_n rho - (3/2) ln T - (v^2 + 2 mu B)/T with the radial label rho advancing along grad psi/|grad psi|:
    the weight rate is its directional derivative along the perturbed velocity (reading G32)."""
    tab = inputs.equilibrium_table(cfg1, 65, 65, 17, kappa=1.4)
    o = oracle.from_workload(cfg1, inputs)
    o.set_equilibrium_table(tab)
    rng = np.random.default_rng(5)
    fld = 1e-2 * rng.standard_normal((pts["R"].size, 4))
    zero = np.zeros_like(fld)
    k = o.rhs_point(pts["R"], pts["Z"], pts["vpar"], pts["mu"], pts["w"], fld)
    k0 = o.rhs_point(pts["R"], pts["Z"], pts["vpar"], pts["mu"], pts["w"], zero)
    dR, dZ, dv = k[:, 0] - k0[:, 0], k[:, 1] - k0[:, 1], k[:, 3] - k0[:, 3]        # perturbed velocity
    s = _scipy_fields(tab, pts["R"], pts["Z"])
    g = np.hypot(s["psiR"], s["psiZ"])
    drho = (dR * s["psiR"] + dZ * s["psiZ"]) / g
    kn, kT, T = cfg1.kappa_n, cfg1.kappa_T, cfg1.T
    en = pts["vpar"] ** 2 / T + 2 * pts["mu"] * s["B"] / T - 1.5
    L = drho * (-kn - en * kT) - (2 * pts["mu"] / T) * (dR * s["dBdR"] + dZ * s["dBdZ"]) - (2 * pts["vpar"] / T) * dv
    want = -(1.0 - pts["w"]) * L
    assert np.abs(k[:, 4] - want).max() < 1e-12 * np.abs(want).max()
    # and it is not the circular rhat any more
    x, z = pts["R"] - cfg1.R0, pts["Z"]
    drho_c = (dR * x + dZ * z) / np.hypot(x, z)
    assert np.abs(drho - drho_c).max() > 1e-3 * np.abs(drho).max()


def test_pushes_approach_the_analytic_equilibrium_pushes(inputs, cfg1):
    m = inputs.markers(cfg1, n=256, seed=23)
    m["w"] = np.zeros(256)
    oa = oracle.from_workload(cfg1, inputs, eom_variant=1)
    oa.bell_from_dofs(cfg1.modes, inputs.field_dofs(cfg1))
    ref = oa.push(m, cfg1.dt, 40)
    errs = []
    for N in (33, 65, 129):
        o = oracle.from_workload(cfg1, inputs, eom_variant=1)
        o.bell_from_dofs(cfg1.modes, inputs.field_dofs(cfg1))
        o.set_equilibrium_table(inputs.equilibrium_table(cfg1, N, N))
        out = o.push(m, cfg1.dt, 40)
        ok = (out["cell"] >= 0) & (ref["cell"] >= 0)
        errs.append(max(np.abs(out["R"] - ref["R"])[ok].max(), np.abs(out["Z"] - ref["Z"])[ok].max()))
        # canonical momentum in the table's own psi: conserved to the RK4 error
        def P(mm):
            e = o.equilibrium(mm["R"], mm["Z"])
            return e["psi"] + EPS * mm["vpar"] * mm["R"] * e["bphi"]
        oo = oracle.from_workload(cfg1, inputs, eom_variant=1)
        oo.set_modes([])
        oo.set_equilibrium_table(inputs.equilibrium_table(cfg1, N, N))
        free = oo.push(m, cfg1.dt, 40)
        okf = free["cell"] >= 0
        e0, e1 = oo.equilibrium(m["R"], m["Z"]), oo.equilibrium(free["R"], free["Z"])
        P0 = e0["psi"] + EPS * m["vpar"] * m["R"] * e0["bphi"]
        P1 = e1["psi"] + EPS * free["vpar"] * free["R"] * e1["bphi"]
        assert np.abs(P1 - P0)[okf].max() < 1e-9
    assert errs[0] > 3 * errs[1] > 9 * errs[2] and errs[2] < 1e-5
