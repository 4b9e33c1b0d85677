"""GPU parity of row f4's tabulated equilibrium (trimeg_equilibrium_upload; reading G32) against
oracle O14 through the C ABI: one right-hand side in every equation variant, the electromagnetic right-hand side, the RK4 push
in every schedule, on the ring x sector and on the unstructured mesh, with an elongated table and F' != 0.  Bars as for the
analytic equilibrium (tests/test_gpu_parity.py)."""
import numpy as np
import pytest

import oracle
from helpers import rel_err, wrap_diff

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2601_14301_b200 import binding
    binding.load()
    return binding


def _setup(B, inputs, name, variant=0, wmode=0, kappa=1.3, f1=0.2, N=65):
    wl = inputs.WORKLOADS[name]
    o = oracle.from_workload(wl, inputs, eom_variant=variant, weight_mode=wmode)
    ctx = B.context_for(wl, inputs, eom_variant=variant, weight_mode=wmode)
    tab = inputs.equilibrium_table(wl, N, N, 17, kappa=kappa, f1=f1)
    o.set_equilibrium_table(tab)
    ctx.equilibrium_upload(tab)
    coef = o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    return wl, o, ctx, coef, tab


SCALES = dict(R=10.0, Z=1.0, vpar=1.0)


def _assert_state_close(got, want, tol, wscale=1e-4):
    for k in ("R", "Z", "vpar"):
        e = rel_err(got[k], want[k], SCALES[k]).max()
        assert e < tol, (k, e)
    e = (wrap_diff(got["phi"], want["phi"]) / (2 * np.pi)).max()
    assert e < tol, ("phi", e)
    e = rel_err(got["w"], want["w"], wscale).max()
    assert e < tol, ("w", e)


@pytest.mark.parametrize("name,n,variant,wmode", [("cfg1", 4096, 0, 0), ("cfg1", 2000, 1, 1), ("cfg1", 2000, 2, 0),
                                                  ("cfg2", 50021, 0, 0), ("cfg5", 20011, 2, 0)])
def test_rhs_parity_with_a_table(B, inputs, name, n, variant, wmode):
    wl, o, ctx, _, _ = _setup(B, inputs, name, variant, wmode)
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    want = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    d["cell"] = ctx.locate(d["R"], d["Z"])
    got = ctx.rhs(d)
    for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt"):
        e = rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max()
        assert e < 1e-12, (k, e)
    # the table is in use: the analytic equilibrium gives something else; and it comes back when the table is dropped
    ctx.equilibrium_upload(None)
    o.set_equilibrium_table(None)
    back = ctx.rhs(d)["dZdt"].cpu().numpy()
    assert np.abs(back - want["dZdt"]).max() > 1e-4 * np.abs(want["dZdt"]).max()
    wa = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])["dZdt"]
    assert rel_err(back, wa, np.abs(wa).max()).max() < 1e-12


@pytest.mark.parametrize("variant", [0, 2])
def test_rhs_em_parity_with_a_table(B, inputs, variant):
    wl, o, ctx, coef, _ = _setup(B, inputs, "cfg2", variant)
    rng = np.random.default_rng(9)
    cs = coef * (0.5 + 0.1 * rng.standard_normal(coef.shape))
    ch = coef * (-0.25 + 0.1 * rng.standard_normal(coef.shape))
    o.set_aux_coeffs(0, cs); o.set_aux_coeffs(1, ch)
    ctx.field_upload_aux(B.FIELD_AS, torch.from_numpy(cs).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AH, torch.from_numpy(ch).cuda(), kind=1)
    n = 40009
    m = inputs.markers(wl, n=n)
    m["w"] = rng.standard_normal(n) * 1e-2
    want = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    got = ctx.rhs_em(d)
    for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt"):
        e = rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max()
        assert e < 1e-12, (k, e)


@pytest.mark.parametrize("schedule", [0, 1, 2])
@pytest.mark.parametrize("name,n,nsteps,tol,variant", [("cfg1", 4096, 1, 1e-12, 0), ("cfg1", 4096, 20, 1e-9, 1),
                                                       ("cfg2", 30011, 3, 1e-10, 0), ("cfg5", 40009, 5, 1e-10, 2)])
def test_push_parity_with_a_table(B, inputs, schedule, name, n, nsteps, tol, variant):
    wl, o, ctx, _, _ = _setup(B, inputs, name, variant)
    ctx.set_push_kernel(schedule)
    m = inputs.markers(wl, n=n)
    if wl.sigma_w == 0.0:
        m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    want = o.push(m, wl.dt, nsteps)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, nsteps)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, tol)


def test_table_on_the_unstructured_mesh_and_the_host_path(B, inputs):
    wl = inputs.WORKLOADS["cfg2"]
    Rv, Zv, tri = inputs.unstructured_mesh(wl)
    tri = np.ascontiguousarray(tri[B.mesh_locality_order(Rv, Zv, tri)])
    tab = inputs.equilibrium_table(wl, 97, 97, 17, kappa=1.2, f1=0.1)
    o = oracle.Oracle.unstructured(Rv, Zv, tri, wl.params(1, 0))
    ctx = B.Context.unstructured(Rv, Zv, tri, wl.params(1, 0))
    o.set_equilibrium_table(tab); ctx.equilibrium_upload(tab)
    coef = o.bell_from_dofs(wl.modes, inputs.field_dofs_at(wl, Rv, Zv))
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    n = 50021
    m = inputs.markers(wl, n=n)
    want = o.push(m, wl.dt, 12)
    h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
    ctx.push_host(h, wl.dt, 12, locate_first=True)
    got = {k: v.numpy() for k, v in h.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-9)


def test_table_errors(B, inputs):
    wl = inputs.WORKLOADS["cfg1"]
    ctx = B.context_for(wl, inputs)
    tab = inputs.equilibrium_table(wl, 33, 33, 9)
    small = dict(tab, Ra=tab["Ra"] + 10 * tab["hR"])                 # the mesh sticks out of the table
    with pytest.raises(B.TrimegError) as e:
        ctx.equilibrium_upload(small)
    assert e.value.code == B.ERR_INVALID_ARG
    with pytest.raises(B.TrimegError) as e:
        ctx.equilibrium_upload(dict(tab, hZ=0.0))
    assert e.value.code == B.ERR_INVALID_ARG
    with pytest.raises(B.TrimegError) as e:
        ctx.equilibrium_upload(dict(tab, D=tab["D"][:3]))
    assert e.value.code == B.ERR_INVALID_ARG
    ctx.equilibrium_upload(tab)
    ctx.equilibrium_upload(None)
