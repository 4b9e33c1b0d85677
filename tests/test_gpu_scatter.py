"""GPU parity of row f1, the particle-to-grid projection trimeg_scatter, against the oracle's
plain definition (O8), through the C ABI.  Bar: |got - want| <= 1e-12 max|want| per toroidal mode (sums of up to 10^5
terms of mixed sign per degree of freedom: the scale is the largest entry of the mode's right-hand side)."""
import dataclasses

import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2601_14301_b200 import binding
    binding.load()
    return binding


def _setup(B, inputs, name, **replace):
    wl = inputs.WORKLOADS[name]
    if replace:
        wl = dataclasses.replace(wl, **replace)
    o = oracle.from_workload(wl, inputs)
    o.set_modes(wl.modes)
    ctx = B.context_for(wl, inputs)
    dofs = inputs.field_dofs(wl) if wl.modes else None
    ctx.field_upload(wl.modes, torch.from_numpy(dofs).cuda() if dofs is not None else None, kind=0)
    return wl, o, ctx


def _close(got, want, tol=1e-12):
    for k in range(want.shape[0]):
        scale = np.abs(want[k]).max()
        err = np.abs(got[k] - want[k]).max()
        assert err <= tol * scale, (k, err / scale)


@pytest.mark.parametrize("name,n,modes", [("cfg1", 4096 + 37, None), ("cfg2", 70001, None), ("cfg5", 150001, None),
                                          ("cfg1", 3001, (0, 1, 5)), ("cfg1", 5003, tuple(range(0, 40, 2))),
                                          ("cfg3", 40009, None)])
@pytest.mark.parametrize("order", ["as drawn", "sorted"])
def test_scatter_parity(B, inputs, name, n, modes, order):
    """Markers as drawn (any order is correct) and cell-sorted; lost markers (cfg5: some start outside the outer polygon);
    arithmetic and non-arithmetic mode lists; more modes than one pass of the kernel takes (20 > 16)."""
    wl, o, ctx = _setup(B, inputs, name, **({"modes": modes} if modes is not None else {}))
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(4).standard_normal(n)
    want = o.scatter(m["R"], m["Z"], m["phi"], m["w"])
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    if order == "sorted":
        ctx.sort(d)
    got = ctx.scatter(d).cpu().numpy()
    _close(got, want)
    if name == "cfg5":
        assert (d["cell"] < 0).sum() > 0


def test_scatter_is_the_adjoint_of_the_library_gather(B, inputs):
    """sum_p w_p dphi(x_p) = Re sum Y conj(rhs) with the library's own Bell expansion (kind 0 upload) and gather: the
    transposed expansion of trimeg_scatter is the transpose of bell_kernel."""
    wl = inputs.WORKLOADS["cfg2"]
    ctx = B.context_for(wl, inputs)
    rng = np.random.default_rng(12)
    modes = (0, 3, 7)
    Y = rng.standard_normal((3, wl.n_vert, 6)) + 1j * rng.standard_normal((3, wl.n_vert, 6))
    ctx.field_upload(modes, torch.from_numpy(Y).cuda(), kind=0)
    n = 50021
    m = inputs.markers(wl, n=n)
    m["w"] = rng.standard_normal(n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    f = ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=d["cell"])["dphi"].cpu().numpy()
    rhs = ctx.scatter(d).cpu().numpy()
    lhs = (m["w"] * f).sum()
    rs = (Y[0].real * rhs[0].real).sum() + (Y[1:] * np.conj(rhs[1:])).real.sum()
    assert abs(lhs - rs) < 1e-11 * np.abs(m["w"] * f).sum()
    assert np.abs(rhs[0].imag).max() == 0.0


def test_scatter_edge_cases(B, inputs):
    wl, o, ctx = _setup(B, inputs, "cfg1")
    m = inputs.markers(wl, n=1000)
    m["w"] = np.ones(1000)
    d = B.markers_to_device(m)
    # stale hints (cell = 0 everywhere): same result as with the right cells
    d["cell"].zero_()
    a = ctx.scatter(d).cpu().numpy()
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    b = ctx.scatter(d).cpu().numpy()
    _close(a, b, 1e-13)
    # partition of unity: the value degrees of freedom of the n = 0 mode sum to the number of markers
    assert abs(b[0, :, 0].sum().real - 1000.0) < 1e-9
    # flagged markers are skipped
    d["cell"][::2] = -1
    c = ctx.scatter(d).cpu().numpy()
    keep = np.arange(1000) % 2 == 1
    want = o.scatter(m["R"][keep], m["Z"][keep], m["phi"][keep], m["w"][keep])
    _close(c, want)
    # n = 0: all zeros
    empty = {k: v[:0].contiguous() for k, v in d.items()}
    z = ctx.scatter(empty).cpu().numpy()
    assert z.shape == (2, wl.n_vert, 6) and np.all(z == 0)
    # no mode list uploaded
    ctx2 = B.context_for(wl, inputs)
    with pytest.raises(B.TrimegError) as e:
        ctx2.scatter(d)
    assert e.value.code == B.ERR_NO_FIELD
    ctx2.field_upload([], None, kind=1)
    assert ctx2.scatter(d).numel() == 0


def test_scatter_full_size_sampled_against_polynomial_moments(B, inputs):
    """cfg5 at full size (2^24 markers, 16 modes, markers as drawn): what holds at any size -- the moments against a
    polynomial of degree <= 4 computed from the marker arrays with numpy (the element space contains P4) -- and, per mode,
    the sum of the value degrees of freedom."""
    from numpy.polynomial import polynomial as npoly
    from helpers import poly_dofs
    wl, o, ctx = _setup(B, inputs, "cfg5")
    n = wl.n_markers
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(6).standard_normal(n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    rhs = ctx.scatter(d).cpu().numpy()
    inside = d["cell"].cpu().numpy() >= 0
    _, Rv, Zv = inputs.mesh_nodes(wl)
    rng = np.random.default_rng(10)
    C = np.zeros((5, 5))
    for i in range(5):
        for j in range(5 - i):
            C[i, j] = rng.standard_normal()
    dofs = poly_dofs(C, Rv, Zv)
    q = npoly.polyval2d(m["R"] - 10.0, m["Z"], C)
    for k, nmode in enumerate(wl.modes):
        got = (dofs * rhs[k]).sum()
        want = (m["w"] * q * np.exp(-1j * nmode * m["phi"]))[inside].sum()
        assert abs(got - want) < 1e-10 * np.abs(m["w"] * q)[inside].sum(), (nmode, got, want)
