"""GPU parity of row f4's reduced equations of motion (eom_variant 2, A.19-A.29) against oracle O12
through the C ABI: one right-hand side (trimeg_rhs: A.28 with dA = 0; trimeg_rhs_em: A.24-A.26, A.29), the RK4 push in every
schedule, on the harmonic and on the B-spline field.  Bars as for the rigorous model (tests/test_gpu_parity.py)."""
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


def _setup(B, inputs, name, wmode=0):
    wl = inputs.WORKLOADS[name]
    o = oracle.from_workload(wl, inputs, eom_variant=2, weight_mode=wmode)
    ctx = B.context_for(wl, inputs, eom_variant=2, weight_mode=wmode)
    coef = o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    return wl, o, ctx, coef


SCALES = dict(R=10.0, Z=1.0, vpar=1.0)


def _assert_state_close(got, want, tol, wscale=1e-4):
    for k in ("R", "Z", "vpar"):
        e = rel_err(got[k], want[k], SCALES[k]).max()
        assert e < tol, (k, e)
    e = (wrap_diff(got["phi"], want["phi"]) / (2 * np.pi)).max()
    assert e < tol, ("phi", e)
    e = rel_err(got["w"], want["w"], wscale).max()
    assert e < tol, ("w", e)


@pytest.mark.parametrize("name,n,wmode", [("cfg1", 4096, 0), ("cfg1", 1000, 1), ("cfg2", 50021, 0), ("cfg5", 20011, 0)])
def test_reduced_rhs_parity(B, inputs, name, n, wmode):
    wl, o, ctx, _ = _setup(B, inputs, name, wmode)
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    want = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    d["cell"] = ctx.locate(d["R"], d["Z"])
    got = ctx.rhs(d)
    for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt"):
        scale = np.abs(want[k]).max()
        e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
        assert e < 1e-12, (k, e)
    # and it is not the rigorous model's answer
    ctx.set_params(wl.params(0, wmode))
    full = ctx.rhs(d)["dZdt"].cpu().numpy()
    assert np.abs(full - want["dZdt"]).max() > 1e-7 * np.abs(want["dZdt"]).max()


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("name,n,nsteps,tol", [("cfg1", 4096, 1, 1e-12), ("cfg1", 4096, 20, 1e-9), ("cfg2", 30011, 3, 1e-10),
                                               ("cfg5", 40009, 5, 1e-10)])
def test_reduced_push_parity_every_schedule(B, inputs, variant, name, n, nsteps, tol):
    wl, o, ctx, _ = _setup(B, inputs, name)
    ctx.set_push_kernel(variant)
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
    if name == "cfg5":
        assert (want["cell"] < 0).sum() > 0


def test_reduced_push_on_the_spline_field(B, inputs):
    wl = inputs.WORKLOADS["cfg2"]
    o = oracle.from_workload(wl, inputs, eom_variant=2)
    ctx = B.context_for(wl, inputs, eom_variant=2)
    sd = inputs.spline_dofs(wl, 16)
    coef = o.bell_spline_from_dofs(sd)
    ctx.field_upload_spline(torch.from_numpy(coef).cuda(), kind=1)
    n = 30011
    m = inputs.markers(wl, n=n)
    want = o.push(m, wl.dt, 3)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 3)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10)


@pytest.mark.parametrize("name,n,wmode,qom", [("cfg1", 4096, 0, 1.0), ("cfg1", 2000, 1, -1.5), ("cfg5", 20011, 0, 1.0)])
def test_reduced_rhs_em_parity(B, inputs, name, n, wmode, qom):
    import dataclasses
    wl = dataclasses.replace(inputs.WORKLOADS[name], qs_over_ms=qom)
    o = oracle.from_workload(wl, inputs, eom_variant=2, weight_mode=wmode)
    ctx = B.context_for(wl, inputs, eom_variant=2, weight_mode=wmode)
    coef = o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    rng = np.random.default_rng(9)
    cs = coef * (0.5 + 0.1 * rng.standard_normal(coef.shape))
    ch = coef * (-0.25 + 0.1 * rng.standard_normal(coef.shape))
    o.set_aux_coeffs(0, cs); o.set_aux_coeffs(1, ch)
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AS, torch.from_numpy(cs).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AH, torch.from_numpy(ch).cuda(), kind=1)
    m = inputs.markers(wl, n=n)
    m["w"] = rng.standard_normal(n) * 1e-2
    want = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    got = ctx.rhs_em(d)
    for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt"):
        scale = np.abs(want[k]).max()
        e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
        assert e < 1e-12, (k, e)


def test_params_reject_unknown_variant(B, inputs):
    wl = inputs.WORKLOADS["cfg1"]
    ctx = B.context_for(wl, inputs)
    with pytest.raises(B.TrimegError) as e:
        ctx.set_params(wl.params(3, 0))
    assert e.value.code == B.ERR_INVALID_ARG
