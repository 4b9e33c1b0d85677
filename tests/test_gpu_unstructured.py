"""GPU parity of row f4's general geometry -- an unstructured triangulation with the thesis's box-grid locator
(trimeg_mesh_create_unstructured; reading G31) -- against oracle O13 through the C ABI: geometry table
and cells bit-exact, Bell constructor, gather, right-hand side, RK4 push in every schedule, sort, scatter, the electromagnetic
right-hand side and the B-spline field on the same mesh.  Bars as on the ring x sector mesh (tests/test_gpu_parity.py)."""
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


_cache = {}


def _setup(B, inputs, name, grid=(0, 0), eom_variant=0):
    wl = inputs.WORKLOADS[name]
    if name not in _cache:
        _cache[name] = inputs.unstructured_mesh(wl)
    Rv, Zv, tri = _cache[name]
    o = oracle.Oracle.unstructured(Rv, Zv, tri, wl.params(eom_variant, 0))
    ctx = B.Context.unstructured(Rv, Zv, tri, wl.params(eom_variant, 0), nbx=grid[0], nby=grid[1])
    dofs = inputs.field_dofs_at(wl, Rv, Zv)
    coef = o.bell_from_dofs(wl.modes, dofs)
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    return wl, o, ctx, dofs, coef, (Rv, Zv, tri)


SCALES = dict(R=10.0, Z=1.0, vpar=1.0)


def _assert_state_close(got, want, tol, wscale=1e-4):
    for k in ("R", "Z", "vpar"):
        e = rel_err(got[k], want[k], SCALES[k]).max()
        assert e < tol, (k, e)
    e = (wrap_diff(got["phi"], want["phi"]) / (2 * np.pi)).max()
    assert e < tol, ("phi", e)
    e = rel_err(got["w"], want["w"], wscale).max()
    assert e < tol, ("w", e)


def _probe_points(wl, mesh, n, seed):
    Rv, Zv, tri = mesh
    rng = np.random.default_rng(seed)
    r = 1.1 * np.sqrt(rng.random(n)); th = 2 * np.pi * rng.random(n)
    R = np.concatenate([wl.R0 + r * np.cos(th), Rv, 0.5 * (Rv[tri[:, 0]] + Rv[tri[:, 1]]), (Rv[tri[:, 1]] + 2 * Rv[tri[:, 2]]) / 3,
                        [np.nan, 1e9, -1e9]])
    Z = np.concatenate([r * np.sin(th), Zv, 0.5 * (Zv[tri[:, 0]] + Zv[tri[:, 1]]), (Zv[tri[:, 1]] + 2 * Zv[tri[:, 2]]) / 3,
                        [0.0, 0.0, np.nan]])
    return R, Z


@pytest.mark.parametrize("name,grid", [("cfg1", (0, 0)), ("cfg1", (1, 1)), ("cfg1", (37, 5)), ("cfg2", (0, 0)), ("cfg5", (0, 0)),
                                       ("cfg5", (500, 400))])
def test_geometry_and_locate_bit_exact(B, inputs, name, grid):
    """Own box grid (any resolution) and the oracle's: both must give the rule over all triangles -- points in and around
    the mesh, every vertex, edge midpoints, NaN and far points; hints none, right, zero and random."""
    wl, o, ctx, _, _, mesh = _setup(B, inputs, name, grid)
    assert np.array_equal(ctx.mesh_download_geom().cpu().numpy(), o.geom())
    R, Z = _probe_points(wl, mesh, 100000, 3)
    want = o.locate(R, Z)
    if name == "cfg1":
        assert np.array_equal(want, o.locate_brute(R, Z))
    dR, dZ = torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda()
    rng = np.random.default_rng(1)
    for hint in (None, want, np.zeros_like(want), rng.integers(-5, wl.n_tri + 5, want.size).astype(np.int32)):
        cell = torch.full((R.size,), -1, dtype=torch.int32, device="cuda") if hint is None else torch.from_numpy(hint.astype(np.int32)).cuda()
        got = ctx.locate(dR, dZ, cell=cell).cpu().numpy()
        assert np.array_equal(got, want)
    assert (want >= 0).sum() > 80000 and (want < 0).sum() > 10000


@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_bell_constructor_on_the_unstructured_mesh(B, inputs, name):
    wl, o, ctx, dofs, coef, _ = _setup(B, inputs, name)
    ctx.field_upload(wl.modes, torch.from_numpy(dofs).cuda(), kind=0)
    got = ctx.field_download_coeffs().cpu().numpy()
    scale = np.abs(coef).max(axis=2, keepdims=True)
    assert (np.abs(got - coef) / np.maximum(scale, 1e-300)).max() < 1e-10


@pytest.mark.parametrize("name,n", [("cfg1", 4096 + 37), ("cfg2", 70001), ("cfg5", 30011)])
def test_gather_and_rhs_parity(B, inputs, name, n):
    wl, o, ctx, _, _, _ = _setup(B, inputs, name)
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    want = o.gather(m["R"], m["Z"], m["phi"])
    d = B.markers_to_device(m)
    for hint in (None, torch.from_numpy(want["cell"]).cuda()):
        got = ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=hint)
        for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
            e = rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max()
            assert e < 1e-12, (k, e)
    wr = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d["cell"] = ctx.locate(d["R"], d["Z"])
    assert np.array_equal(d["cell"].cpu().numpy(), wr["cell"])
    gr = ctx.rhs(d)
    for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt"):
        e = rel_err(gr[k].cpu().numpy(), wr[k], np.abs(wr[k]).max()).max()
        assert e < 1e-12, (k, e)


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("name,n,nsteps,tol,sort", [("cfg1", 4096, 1, 1e-12, False), ("cfg1", 4096, 20, 1e-9, False),
                                                    ("cfg2", 30011, 3, 1e-10, True), ("cfg5", 40009, 5, 1e-10, True)])
def test_push_parity_every_schedule(B, inputs, variant, name, n, nsteps, tol, sort):
    wl, o, ctx, _, _, _ = _setup(B, inputs, name)
    ctx.set_push_kernel(variant)
    m = inputs.markers(wl, n=n)
    if wl.sigma_w == 0.0:
        m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    want = o.push(m, wl.dt, nsteps)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    perm = ctx.sort(d, want_perm=True).cpu().numpy() if sort else np.arange(n)
    if sort:
        c = d["cell"].cpu().numpy()
        act = c[c >= 0]
        assert np.all(np.diff(act) >= 0)
    ctx.push(d, wl.dt, nsteps)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    wantp = {k: v[perm] for k, v in want.items()}
    assert np.array_equal(got["cell"], wantp["cell"])
    _assert_state_close(got, wantp, tol)
    if name == "cfg5":
        assert (want["cell"] < 0).sum() > 0


def test_push_host_and_reduced_equations(B, inputs):
    wl, o, ctx, _, _, _ = _setup(B, inputs, "cfg2", eom_variant=2)
    n = 50021
    m = inputs.markers(wl, n=n)
    want = o.push(m, wl.dt, 12)
    h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
    ctx.push_host(h, wl.dt, 12, locate_first=True)
    got = {k: v.numpy() for k, v in h.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-9)


def test_scatter_em_and_spline_field_on_the_unstructured_mesh(B, inputs):
    wl, o, ctx, _, coef, mesh = _setup(B, inputs, "cfg2")
    n = 60013
    m = inputs.markers(wl, n=n)
    rng = np.random.default_rng(4)
    m["w"] = rng.standard_normal(n)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    want = o.scatter(m["R"], m["Z"], m["phi"], m["w"])
    for order in ("as drawn", "sorted"):
        if order == "sorted":
            ctx.sort(d)
        got = ctx.scatter(d).cpu().numpy()
        for k in range(want.shape[0]):
            assert np.abs(got[k] - want[k]).max() <= 1e-12 * np.abs(want[k]).max(), (order, k)
    # electromagnetic right-hand side
    cs, ch = 0.5 * coef, -0.25 * coef
    o.set_aux_coeffs(0, cs); o.set_aux_coeffs(1, ch)
    ctx.field_upload_aux(B.FIELD_AS, torch.from_numpy(cs).cuda(), kind=1)
    ctx.field_upload_aux(B.FIELD_AH, torch.from_numpy(ch).cuda(), kind=1)
    m["w"] *= 1e-2
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    we = o.rhs_em(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    ge = ctx.rhs_em(d)
    for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt"):
        e = rel_err(ge[k].cpu().numpy(), we[k], np.abs(we[k]).max()).max()
        assert e < 1e-12, (k, e)
    # B-spline planes on the same mesh
    Rv, Zv, tri = mesh
    Y = inputs.field_dofs_at(wl, Rv, Zv)
    phi_j = 2 * np.pi * np.arange(16) / 16
    sd = sum((Y[k][None] * np.exp(1j * nn * phi_j)[:, None, None]).real for k, nn in enumerate(wl.modes))
    sc = o.bell_spline_from_dofs(np.ascontiguousarray(sd))
    ctx.field_upload_spline(torch.from_numpy(sc).cuda(), kind=1)
    m["w"] = np.zeros(n)
    wp = o.push(m, wl.dt, 3)
    d = B.markers_to_device(m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 3)
    got = {k: v.cpu().numpy() for k, v in d.items()}
    assert np.array_equal(got["cell"], wp["cell"])
    _assert_state_close(got, wp, 1e-10)


def test_locality_order_is_a_renumbering_with_the_same_physics(B, inputs):
    """tri[order] is the same mesh: cells map through the order, states agree to rounding (the same triangles, the same
    arithmetic: bit for bit unless a marker sits within the locator's margin of an edge)."""
    wl = inputs.WORKLOADS["cfg2"]
    Rv, Zv, tri = inputs.unstructured_mesh(wl)
    order = B.mesh_locality_order(Rv, Zv, tri)
    assert np.array_equal(np.sort(order), np.arange(tri.shape[0]))
    cen = np.stack([Rv[tri[order]].mean(axis=1), Zv[tri[order]].mean(axis=1)], axis=1)
    assert np.hypot(*(cen[1:] - cen[:-1]).T).mean() < 0.05                # neighbours in number are neighbours in space
    inv = np.empty_like(order); inv[order] = np.arange(order.size, dtype=order.dtype)
    n = 40009
    m = inputs.markers(wl, n=n)
    out = []
    for t in (tri, np.ascontiguousarray(tri[order])):
        ctx = B.Context.unstructured(Rv, Zv, t, wl.params())
        ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs_at(wl, Rv, Zv)).cuda(), kind=0)
        d = B.markers_to_device(m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        ctx.push(d, wl.dt, 5)
        out.append({k: v.cpu().numpy() for k, v in d.items()})
    a, b = out
    lost = a["cell"] < 0
    assert np.array_equal(lost, b["cell"] < 0)
    assert np.array_equal(inv[a["cell"][~lost]], b["cell"][~lost])
    _assert_state_close(a, b, 1e-13)


def test_mesh_errors(B, inputs):
    wl = inputs.WORKLOADS["cfg1"]
    Rv, Zv, tri = inputs.unstructured_mesh(wl)
    bad = tri.copy(); bad[3, 1] = Rv.size
    with pytest.raises(B.TrimegError) as e:
        B.Context.unstructured(Rv, Zv, bad, wl.params())
    assert e.value.code == B.ERR_MESH
    bad = tri.copy(); bad[5] = (7, 7, 9)
    with pytest.raises(B.TrimegError) as e:
        B.Context.unstructured(Rv, Zv, bad, wl.params())
    assert e.value.code == B.ERR_MESH
    dup = np.concatenate([tri, tri[:1]])
    with pytest.raises(B.TrimegError) as e:
        B.Context.unstructured(Rv, Zv, dup, wl.params())
    assert e.value.code == B.ERR_MESH
    # a clockwise triple is turned, as in the oracle
    cw = tri.copy(); cw[10] = cw[10][[0, 2, 1]]
    ctx = B.Context.unstructured(Rv, Zv, cw, wl.params())
    o = oracle.Oracle.unstructured(Rv, Zv, cw, wl.params())
    assert np.array_equal(ctx.mesh_download_geom().cpu().numpy(), o.geom())
