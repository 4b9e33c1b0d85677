"""GPU parity of row f2 -- trimeg_rhs_em (the thesis's K1 with the electromagnetic model on) and trimeg_pullback (K2) --
against the oracle's O9 / O10 through the C ABI.  Bars as for trimeg_rhs: 1e-12 relative to the largest entry of each output
array; cells implied (markers outside the mesh get 0 / are left untouched)."""
import dataclasses

import numpy as np
import pytest

import oracle
from helpers import rel_err

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2601_14301_b200 import binding
    binding.load()
    return binding


def _setup(B, inputs, name, seed, amps=(1e-3, 2e-3, 5e-4), **replace):
    wl = inputs.WORKLOADS[name]
    if replace:
        wl = dataclasses.replace(wl, **replace)
    o = oracle.from_workload(wl, inputs)
    ctx = B.context_for(wl, inputs)
    rng = np.random.default_rng(seed)
    M = len(wl.modes)
    dofs = [a * (rng.standard_normal((M, wl.n_vert, 6)) + 1j * rng.standard_normal((M, wl.n_vert, 6))) for a in amps]
    coefs = [o.bell_from_dofs(wl.modes, d) for d in dofs]
    o.set_coeffs(wl.modes, coefs[0]); o.set_aux_coeffs(0, coefs[1]); o.set_aux_coeffs(1, coefs[2])
    ctx.field_upload(wl.modes, torch.from_numpy(coefs[0]).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AS, torch.from_numpy(coefs[1]).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AH, torch.from_numpy(coefs[2]).cuda(), kind=1)
    return wl, o, ctx, dofs, coefs


@pytest.mark.parametrize("name,n,variant,wmode,qom", [("cfg1", 4096, 0, 0, 1.0), ("cfg1", 2000, 1, 1, -2.5), ("cfg2", 50021, 0, 0, 1.0),
                                                      ("cfg5", 30011, 0, 0, 1.0)])
def test_rhs_em_parity(B, inputs, name, n, variant, wmode, qom):
    wl, o, ctx, _, _ = _setup(B, inputs, name, 51, qs_over_ms=qom)
    o.set_params(wl.params(variant, wmode)); ctx.set_params(wl.params(variant, wmode))
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    m["R"][::499] = wl.R0 + 1.3 * wl.a                     # a few markers outside the mesh
    want = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    for hint in ("located", "none"):
        if hint == "located":
            ctx.locate(d["R"], d["Z"], cell=d["cell"])
            assert np.array_equal(d["cell"].cpu().numpy(), want["cell"])
        else:
            d["cell"].fill_(0)
        got = ctx.rhs_em(d)
        for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt"):
            e = rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max()
            assert e < 1e-12, (k, e)
    lost = want["cell"] < 0
    assert lost.sum() > 0 and np.all(got["dudt"].cpu().numpy()[lost] == 0.0) and np.all(got["dwdt"].cpu().numpy()[lost] == 0.0)


def test_rhs_em_tables_absent_and_from_dofs(B, inputs):
    """A field whose table was not uploaded is zero; kind 0 (nodal DOFs through the library's Bell expansion) agrees with the
    oracle's own chain; errors."""
    wl, o, ctx, dofs, coefs = _setup(B, inputs, "cfg1", 52)
    m = inputs.markers(wl, n=3000)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    keys = ("dRdt", "dZdt", "dphidt", "dudt", "dwdt")
    for drop in ((0,), (1,), (0, 1)):
        for a in (0, 1):
            ctx.field_upload_aux(B.FIELD_AS + a, None if a in drop else torch.from_numpy(coefs[1 + a]).cuda(), kind=1)
            o.set_aux_coeffs(a, None if a in drop else coefs[1 + a])
        want = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
        got = ctx.rhs_em(d)
        for k in keys:
            assert rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max() < 1e-12, (drop, k)
    for a in (0, 1):
        ctx.field_upload_aux(B.FIELD_AS + a, torch.from_numpy(dofs[1 + a]).cuda(), kind=0)
        o.set_aux_coeffs(a, coefs[1 + a])
    want = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    got = ctx.rhs_em(d)
    for k in keys:
        assert rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max() < 1e-10, k
    with pytest.raises(B.TrimegError):
        ctx.field_upload_aux(3, None, kind=1)
    ctx2 = B.context_for(wl, inputs)
    with pytest.raises(B.TrimegError) as e:
        ctx2.field_upload_aux(B.FIELD_AH, torch.from_numpy(coefs[2]).cuda(), kind=1)
    assert e.value.code == B.ERR_NO_FIELD
    with pytest.raises(B.TrimegError):
        ctx2.rhs_em(d)


@pytest.mark.parametrize("name,n,wmode", [("cfg1", 4096, 0), ("cfg5", 60013, 0), ("cfg2", 20011, 1)])
def test_pullback_parity(B, inputs, name, n, wmode):
    wl, o, ctx, _, _ = _setup(B, inputs, name, 53, qs_over_ms=-1.5)
    o.set_params(wl.params(0, wmode)); ctx.set_params(wl.params(0, wmode))
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(5).standard_normal(n) * 0.1
    un, wn = o.pullback(m["R"], m["Z"], m["phi"], m["vpar"], m["w"])
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    d["cell"][::11] = -1                                  # flagged markers stay as they are
    ctx.pullback(d)
    gu, gw = d["vpar"].cpu().numpy(), d["w"].cpu().numpy()
    flagged = np.arange(n) % 11 == 0
    assert np.array_equal(gu[flagged], m["vpar"][flagged]) and np.array_equal(gw[flagged], m["w"][flagged])
    assert np.abs(gu - un)[~flagged].max() < 1e-12 * np.abs(un).max()
    assert np.abs(gw - wn)[~flagged].max() < 1e-12 * max(np.abs(wn).max(), 1e-4)
    assert np.abs(gu - m["vpar"])[~flagged].max() > 1e-6
    for k in ("R", "Z", "phi", "mu"):
        assert np.array_equal(d[k].cpu().numpy(), m[k])
    # without a dA^h table nothing happens
    ctx.field_upload_aux(B.FIELD_AH, None, kind=1)
    before = {k: v.clone() for k, v in d.items()}
    ctx.pullback(d)
    assert all(torch.equal(d[k], before[k]) for k in d)
