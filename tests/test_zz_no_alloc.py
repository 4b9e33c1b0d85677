"""trimeg_scatter_static, the projection for callers that cannot allocate device memory (all scratch in the library's static
16 MiB device array, no cudaMalloc / cudaFree anywhere in the call), against the existing trimeg_scatter on the same inputs:
|a - b| <= 1e-12 max|b| per toroidal mode (the bar of tests/test_gpu_scatter.py; the two paths run the same kernels, the
summation order inside a triangle follows an atomic cursor in both).  Two calls in a row on different batches: the array
keeps the last call's contents, the second result must not see them.  Collected last on purpose (file name)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2601_14301_b200 import binding
    binding.load()
    return binding


def _close(got, want, tol=1e-12):
    for k in range(want.shape[0]):
        scale = np.abs(want[k]).max()
        assert scale > 0
        err = np.abs(got[k] - want[k]).max()
        assert err <= tol * scale, (k, err / scale)


def test_scatter_static_equals_scatter_on_two_calls_in_a_row(B, inputs):
    wl = inputs.WORKLOADS["cfg1"]
    ctx = B.context_for(wl, inputs)
    ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).cuda(), kind=0)
    rng = np.random.default_rng(17)
    batches = []
    for n, seed in ((100003, 71), (30011, 72)):          # the second batch is smaller: stale indices of the first stay behind it
        m = inputs.markers(wl, n=n, seed=seed)
        m["w"] = rng.standard_normal(n)
        d = B.markers_to_device(m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        d["cell"][::7] = -1                               # flagged markers are skipped by both paths
        batches.append(d)
    want = [ctx.scatter(d).cpu().numpy() for d in batches]
    assert np.abs(want[0] - want[1][:, :, :]).max() > 0
    torch.cuda.synchronize()
    out = torch.full((len(wl.modes), wl.n_vert, 6), float("nan"), dtype=torch.complex128, device="cuda")
    before = torch.cuda.memory_allocated()
    free_before = torch.cuda.mem_get_info()[0]            # device-wide: a cudaMalloc inside the library would show here
    got = []
    for d in batches:                                     # two calls in a row, same stream, same output buffer
        ctx.scatter_static(d, out)
        got.append(out.cpu().numpy().copy())
    assert torch.cuda.memory_allocated() == before
    assert free_before - torch.cuda.mem_get_info()[0] < (1 << 20)
    for g, w in zip(got, want):
        assert np.isfinite(g.view(np.float64)).all()
        _close(g, w)
    # again in the other order, and an empty batch after a full one: all zeros
    ctx.scatter_static(batches[1], out)
    ctx.scatter_static(batches[0], out)
    _close(out.cpu().numpy(), want[0])
    empty = {k: v[:0].contiguous() for k, v in batches[0].items()}
    ctx.scatter_static(empty, out)
    assert np.all(out.cpu().numpy() == 0)
    # the existing path is untouched by the static one
    _close(ctx.scatter(batches[1]).cpu().numpy(), want[1])


def test_scatter_static_rejects_what_does_not_fit(B, inputs):
    wl = inputs.WORKLOADS["cfg2"]                         # 32 512 triangles x 3 modes: 28 MB of per-triangle results
    ctx = B.context_for(wl, inputs)
    ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).cuda(), kind=0)
    m = inputs.markers(wl, n=1000)
    d = B.markers_to_device(m)
    out = torch.zeros((len(wl.modes), wl.n_vert, 6), dtype=torch.complex128, device="cuda")
    with pytest.raises(B.TrimegError) as e:
        ctx.scatter_static(d, out)
    assert e.value.code == B.ERR_CAPACITY
    assert "static scratch" in str(e.value)
    # too many markers on a mesh that fits
    w1 = inputs.WORKLOADS["cfg1"]
    c1 = B.context_for(w1, inputs)
    c1.field_upload(w1.modes, torch.from_numpy(inputs.field_dofs(w1)).cuda(), kind=0)
    n = B.SCATTER_STATIC_BYTES // 8 + 1
    big = {k: torch.zeros(n, dtype=torch.float64, device="cuda") for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    big["cell"] = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    o1 = torch.zeros((len(w1.modes), w1.n_vert, 6), dtype=torch.complex128, device="cuda")
    with pytest.raises(B.TrimegError) as e:
        c1.scatter_static(big, o1)
    assert e.value.code == B.ERR_CAPACITY
    # no field / B-spline field: the codes of trimeg_scatter
    c2 = B.context_for(w1, inputs)
    with pytest.raises(B.TrimegError) as e:
        c2.scatter_static(d, o1)
    assert e.value.code == B.ERR_NO_FIELD
