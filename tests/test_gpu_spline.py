"""GPU parity of row f3, the field on the cubic B-spline toroidal basis (reading G28), against
oracle O11 through the C ABI: coefficient constructor, gather, one right-hand side, the RK4 push (device and host paths).
Bars as for the harmonic field (tests/test_gpu_parity.py): cells bit-exact, gather / rhs 1e-12 of the field's own scale,
push 1e-12 after one step, 1e-10 after a few, 1e-9 after twenty."""
import dataclasses

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


def _setup(B, inputs, name, n_phi, field="oracle", **replace):
    wl = inputs.WORKLOADS[name]
    if replace:
        wl = dataclasses.replace(wl, **replace)
    o = oracle.from_workload(wl, inputs)
    ctx = B.context_for(wl, inputs)
    dofs = inputs.spline_dofs(wl, n_phi)
    coef = o.bell_spline_from_dofs(dofs)
    if field == "oracle":
        ctx.field_upload_spline(torch.from_numpy(coef).cuda(), kind=1)
    else:
        ctx.field_upload_spline(torch.from_numpy(dofs).cuda(), kind=0)
    return wl, o, ctx, dofs, coef


SCALES = dict(R=10.0, Z=1.0, vpar=1.0)


def _assert_state_close(got, want, tol, wscale=1e-4):
    for k in ("R", "Z", "vpar"):
        e = rel_err(got[k], want[k], SCALES[k]).max()
        assert e < tol, (k, e)
    e = (wrap_diff(got["phi"], want["phi"]) / (2 * np.pi)).max()
    assert e < tol, ("phi", e)
    e = rel_err(got["w"], want["w"], wscale).max()
    assert e < tol, ("w", e)


@pytest.mark.parametrize("name,n_phi", [("cfg1", 8), ("cfg2", 16), ("cfg5", 32), ("cfg1", 5)])
def test_spline_constructor_matches_oracle(B, inputs, name, n_phi):
    wl, o, ctx, dofs, coef = _setup(B, inputs, name, n_phi, field="dofs")
    got = ctx.field_download_coeffs().cpu().numpy()
    assert got.shape == coef.shape == (wl.n_tri, n_phi, 21)
    scale = np.abs(coef).max(axis=2, keepdims=True)
    assert (np.abs(got - coef) / np.maximum(scale, 1e-300)).max() < 1e-11


@pytest.mark.parametrize("name,n,n_phi", [("cfg1", 4096 + 37, 8), ("cfg1", 2003, 4), ("cfg1", 2003, 7), ("cfg2", 70001, 16),
                                          ("cfg3", 30011, 64), ("cfg5", 30011, 32)])
def test_spline_gather_parity(B, inputs, name, n, n_phi):
    wl, o, ctx, _, coef = _setup(B, inputs, name, n_phi)
    m = inputs.markers(wl, n=n)
    # every branch of the periodic wrap: phi < 0, phi > 2 pi, several turns away, exactly on planes
    rng = np.random.default_rng(8)
    m["phi"][: n // 4] -= 2 * np.pi
    m["phi"][n // 4: n // 2] += 2 * np.pi * rng.integers(1, 6, n // 2 - n // 4)
    m["phi"][-64:] = 2 * np.pi * rng.integers(-n_phi, 2 * n_phi, 64) / n_phi
    m["phi"][-1] = 0.0
    want = o.gather(m["R"], m["Z"], m["phi"])
    d = B.markers_to_device(m)
    for hint in (None, torch.from_numpy(want["cell"]).cuda()):
        got = ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=hint)
        for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
            scale = np.abs(want[k]).max()
            assert scale > 0
            e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
            assert e < 1e-12, (k, e)


def test_spline_gather_large_sorted_batch_takes_the_general_kernel(B, inputs):
    """2^18+ hinted, cell-sorted markers: the sorted-batch kernel of the harmonic field must not be chosen."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg2", 16)
    n = 300007
    m = inputs.markers(wl, n=n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    perm = ctx.sort(d, want_perm=True).cpu().numpy()
    got = ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=d["cell"])
    idx = np.arange(0, n, 37)
    src = perm[idx]
    want = o.gather(m["R"][src], m["Z"][src], m["phi"][src])
    for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
        scale = np.abs(want[k]).max()
        e = rel_err(got[k].cpu().numpy()[idx], want[k], scale).max()
        assert e < 1e-12, (k, e)


@pytest.mark.parametrize("name,n,n_phi,variant,wmode", [("cfg1", 4096, 8, 0, 0), ("cfg1", 1000, 8, 1, 1),
                                                        ("cfg2", 50021, 16, 0, 0), ("cfg5", 20011, 32, 0, 0)])
def test_spline_rhs_parity(B, inputs, name, n, n_phi, variant, wmode):
    wl, o, ctx, _, _ = _setup(B, inputs, name, n_phi)
    o.set_params(wl.params(variant, wmode))
    ctx.set_params(wl.params(variant, wmode))
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    want = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = B.markers_to_device(m)
    d["cell"] = ctx.locate(d["R"], d["Z"])
    assert np.array_equal(d["cell"].cpu().numpy(), want["cell"])
    got = ctx.rhs(d)
    for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt"):
        scale = np.abs(want[k]).max()
        e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
        assert e < 1e-12, (k, e)


@pytest.mark.parametrize("name,n,n_phi,nsteps,tol", [("cfg1", 4096, 8, 1, 1e-12), ("cfg1", 4096, 8, 20, 1e-9),
                                                     ("cfg2", (1 << 16) + 13, 16, 3, 1e-10), ("cfg5", 40009, 32, 5, 1e-10)])
@pytest.mark.parametrize("requested", [-1, 0])
def test_spline_push_parity(B, inputs, name, n, n_phi, nsteps, tol, requested):
    """Automatic choice (the lane kernel with plane records in shared memory for an even n_phi <= 48) and the
    thread-per-marker kernel."""
    wl, o, ctx, _, _ = _setup(B, inputs, name, n_phi)
    ctx.set_push_kernel(requested)
    assert ctx.get_push_kernel() == (0 if requested == 0 else 1)
    m = inputs.markers(wl, n=n)
    if wl.sigma_w == 0.0:
        m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    want = o.push(m, wl.dt, nsteps)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, nsteps)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    assert np.array_equal(got["cell"], want["cell"])
    assert np.array_equal(got["mu"], m["mu"])
    _assert_state_close(got, want, tol)
    if nsteps == 20:
        assert np.abs(got["w"] - m["w"]).max() > 1e-6        # the weights evolved under the spline field


@pytest.mark.parametrize("n_phi,expect", [(7, 0), (64, 0), (48, 1), (4, 1)])
def test_spline_push_odd_and_many_planes(B, inputs, n_phi, expect):
    """Odd n_phi (records are not whole 16-byte units) and n_phi > 48 (too few records fit) take the thread kernel; 48
    planes leave the lane kernel a handful of record slots: markers of triangles without one go down its one-marker path."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", n_phi)
    assert ctx.get_push_kernel() == expect
    n = 3001
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    want = o.push(m, wl.dt, 3)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 3)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10)


def test_spline_lane_and_thread_kernels_agree(B, inputs):
    """Same arithmetic per marker in both kernels (the compiler contracts a few products of the RK4 bookkeeping differently:
    an ulp in phi for a handful of markers, as with the harmonic field): cells equal, states within 1e-14."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5", 32)
    n = 100003
    m = inputs.markers(wl, n=n)
    out = []
    for k in (0, 1):
        ctx.set_push_kernel(k)
        d = B.markers_to_device(m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        perm = ctx.sort(d, want_perm=True).cpu().numpy()     # the order inside a cell is not fixed: undo the sort
        ctx.push(d, wl.dt, 10)
        back = {}
        for k2, v in d.items():
            a = v.cpu().numpy()
            back[k2] = np.empty_like(a)
            back[k2][perm] = a
        out.append(back)
    assert np.array_equal(out[0]["cell"], out[1]["cell"]) and np.array_equal(out[0]["mu"], out[1]["mu"])
    _assert_state_close(out[0], out[1], 1e-14)


def test_spline_push_host_equals_device_push(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg2", 16)
    n = 50021
    m = inputs.markers(wl, n=n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 3)
    h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
    ctx.push_host(h, wl.dt, 3, locate_first=True)
    for k in ("R", "Z", "phi", "vpar", "w", "cell", "mu"):
        assert np.array_equal(h[k].numpy(), d[k].cpu().numpy()), k


def test_spline_field_switches_and_unsupported_calls(B, inputs):
    wl, o, ctx, dofs, coef = _setup(B, inputs, "cfg1", 8)
    n = 1000
    m = inputs.markers(wl, n=n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    for call in (lambda: ctx.scatter(d), lambda: ctx.rhs_em(d), lambda: ctx.pullback(d),
                 lambda: ctx.field_upload_aux(B.FIELD_AS, None, kind=1)):
        with pytest.raises(B.TrimegError) as e:
            call()
        assert e.value.code == B.ERR_UNSUPPORTED
    with pytest.raises(B.TrimegError) as e:
        ctx.field_upload_spline(torch.zeros((3, wl.n_vert, 6), dtype=torch.float64, device="cuda"), kind=0)
    assert e.value.code == B.ERR_INVALID_ARG
    a = ctx.gather(d["R"], d["Z"], d["phi"])["dphi"].cpu().numpy()
    # to harmonics and back: each upload replaces the field as a whole
    hd = inputs.field_dofs(wl)
    o.set_spline_coeffs(0, None)
    hc = o.bell_from_dofs(wl.modes, hd)
    ctx.field_upload(wl.modes, torch.from_numpy(hc).cuda(), kind=1)
    want_h = o.gather(m["R"], m["Z"], m["phi"])["dphi"]
    b = ctx.gather(d["R"], d["Z"], d["phi"])["dphi"].cpu().numpy()
    assert rel_err(b, want_h, np.abs(want_h).max()).max() < 1e-12
    assert ctx.scatter(d).shape[0] == len(wl.modes)
    ctx.field_upload_spline(torch.from_numpy(coef).cuda(), kind=1)
    c = ctx.gather(d["R"], d["Z"], d["phi"])["dphi"].cpu().numpy()
    assert np.array_equal(a, c)
    # another n_phi re-allocates
    o.bell_spline_from_dofs(inputs.spline_dofs(wl, 12))
    ctx.field_upload_spline(torch.from_numpy(inputs.spline_dofs(wl, 12)).cuda(), kind=0)
    want = o.gather(m["R"], m["Z"], m["phi"])["dphi"]
    g = ctx.gather(d["R"], d["Z"], d["phi"])["dphi"].cpu().numpy()
    assert rel_err(g, want, np.abs(want).max()).max() < 1e-11


def test_spline_full_size_sampled_parity_in_bench_configuration(B, inputs):
    """cfg5's mesh and markers at full size (2^24) with the field on 32 planes, in the configuration bench.py --basis
    spline times (locate -> sort -> push), every 1024-th marker against the oracle."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5", 32)
    n, nsteps = wl.n_markers, 4
    m = inputs.markers(wl, n=n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    perm = ctx.sort(d, want_perm=True)
    ctx.push(d, wl.dt, nsteps)
    idx = np.arange(0, n, 1024)
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(n, device="cuda", dtype=perm.dtype)
    pos = inv[torch.from_numpy(idx).cuda()]
    got = {k: v[pos].cpu().numpy() for k, v in d.items()}
    want = o.push({k: m[k][idx] for k in m}, wl.dt, nsteps)
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10)
