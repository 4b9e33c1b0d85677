"""GPU parity: the CUDA path (through the C ABI / ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.

Bars (BASELINE.json north_star): triangle indices bit-exact; positions, v_par, weights within
relative 1e-12 after one step and 1e-9 after 20 steps; "relative" = |a-b| / max(|a|,|b|,scale)
with scale R0 for R, a for Z, 2 pi for phi (compared modulo 2 pi), 1 for v_par, max|w| (>= 1e-4)
for w ("GPU vs oracle").  gather / rhs: 1e-12 with the field's own scale.
The coefficient constructor is compared separately (1e-11 max|c| per triangle and mode); every
other test uploads the ORACLE's coefficient table (kind 1) so both sides start from the same bits.
"""
import dataclasses
import math

import numpy as np
import pytest

import oracle
from helpers import interior_edges, local_coords, phys_derivs, rel_err, wrap_diff

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2601_14301_b200 import binding
    binding.load()          # raises if the extension is missing: no fallback
    return binding


def _setup(B, inputs, name, field="oracle", **replace):
    wl = inputs.WORKLOADS[name]
    if replace:
        wl = dataclasses.replace(wl, **replace)
    o = oracle.from_workload(wl, inputs)
    ctx = B.context_for(wl, inputs)
    dofs = inputs.field_dofs(wl)
    coef = o.bell_from_dofs(wl.modes, dofs)
    if field == "oracle":
        ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    elif field == "dofs":
        ctx.field_upload(wl.modes, torch.from_numpy(dofs).cuda(), kind=0)
    return wl, o, ctx, dofs, coef


def _dev(B, m):
    return B.markers_to_device(m)


def _host(md):
    return {k: v.cpu().numpy() for k, v in md.items()}


SCALES = dict(R=10.0, Z=1.0, vpar=1.0)


def _assert_state_close(got, want, tol, wscale):
    for k in ("R", "Z", "vpar"):
        e = rel_err(got[k], want[k], SCALES[k]).max()
        assert e < tol, (k, e)
    e = (wrap_diff(got["phi"], want["phi"]) / (2 * np.pi)).max()
    assert e < tol, ("phi", e)
    e = rel_err(got["w"], want["w"], wscale).max()
    assert e < tol, ("w", e)


# ----------------------------------------------------------------------------- a0
def test_geometry_table_bit_exact(B, inputs):
    for name in ("cfg1", "cfg3"):
        wl, o, ctx, _, _ = _setup(B, inputs, name, field=None)
        g = ctx.mesh_download_geom().cpu().numpy()
        assert np.array_equal(g, o.geom()), name


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5"])
def test_bell_constructor_matches_oracle(B, inputs, name):
    wl, o, ctx, dofs, coef = _setup(B, inputs, name, field="dofs")
    got = ctx.field_download_coeffs().cpu().numpy()
    scale = np.abs(coef).max(axis=2, keepdims=True)
    scale = np.maximum(scale, 1e-300)
    err = (np.abs(got - coef) / scale).max()
    assert err < 1e-11, err


def test_bell_constructor_own_properties(B, inputs):
    """The library's own table: reproduces the nodal DOFs and is C1 across edges (cfg1)."""
    wl, o, ctx, dofs, _ = _setup(B, inputs, "cfg1", field="dofs")
    coef = ctx.field_download_coeffs().cpu().numpy()
    g, tri = o.geom(), o.triangles()
    _, Rv, Zv = inputs.mesh_nodes(wl)
    ref = [(0.0, 0.0), (1.0, 0.0), (0.0, 1.0)]
    worst = 0.0
    for t in range(0, o.n_tri, 3):
        for k, (xi, eta) in enumerate(ref):
            gotd = phys_derivs(coef[t, 1], g[t], xi, eta)
            want = dofs[1, tri[t, k]]
            scale = np.maximum(np.abs(want), np.abs(dofs[1]).max(axis=0))
            worst = max(worst, float((np.abs(gotd - want) / scale).max()))
    assert worst < 1e-12, worst
    fs, gs = np.abs(dofs[..., 0]).max(), np.abs(dofs[..., 1:3]).max()
    wv = wn = 0.0
    for (va, vb), (t1, t2) in list(interior_edges(tri).items())[::2]:
        tR, tZ = Rv[vb] - Rv[va], Zv[vb] - Zv[va]
        L = math.hypot(tR, tZ)
        for s in (0.3, 0.77):
            R, Z = Rv[va] + s * tR, Zv[va] + s * tZ
            vals = []
            for t in (t1, t2):
                xi, eta = local_coords(g[t], R, Z)
                d = phys_derivs(coef[t, 1], g[t], xi, eta)
                vals.append((d[0], (tZ * d[1] - tR * d[2]) / L))
            wv = max(wv, abs(vals[0][0] - vals[1][0]) / fs)
            wn = max(wn, abs(vals[0][1] - vals[1][1]) / gs)
    assert wv < 1e-12 and wn < 1e-12, (wv, wn)


# ----------------------------------------------------------------------------- a2
def _probe_points(wl, n, seed):
    rng = np.random.default_rng(seed)
    r = np.concatenate([np.sqrt(rng.random(n)) * 1.02 * wl.a, rng.random(n // 8) * 1e-3 * wl.a,
                        wl.a * (1 - 5e-3 * rng.random(n // 8))])
    th = 2 * np.pi * rng.random(r.size)
    return wl.R0 + r * np.cos(th), r * np.sin(th)


def test_locate_bit_exact_vs_brute_force_cfg1(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", field=None)
    _, Rv, Zv = inputs.mesh_nodes(wl)
    R, Z = _probe_points(wl, 100003, 1)
    # add every vertex, every edge midpoint, and special values
    tri = o.triangles()
    em = np.array([[0.5 * (Rv[a] + Rv[b]), 0.5 * (Zv[a] + Zv[b])] for (a, b) in
                   {tuple(sorted((int(t[i]), int(t[(i + 1) % 3])))) for t in tri for i in range(3)}])
    R = np.concatenate([R, Rv, em[:, 0], [np.nan, 1e300, 10.0, 12.0]])
    Z = np.concatenate([Z, Zv, em[:, 1], [0.0, 0.0, np.nan, 0.0]])
    want = o.locate_brute(R, Z)
    got = ctx.locate(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda()).cpu().numpy()
    assert np.array_equal(got, want), np.where(got != want)[0][:10]
    assert (want < 0).sum() > 100 and (want >= 0).sum() > 90000


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg5"])
def test_locate_bit_exact_large_meshes(B, inputs, name):
    wl, o, ctx, _, _ = _setup(B, inputs, name, field=None)
    R, Z = _probe_points(wl, 400001, 2)
    want = o.locate(R, Z)                 # pinned to brute force by tests/test_oracle_locator.py
    got = ctx.locate(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda()).cpu().numpy()
    assert np.array_equal(got, want)
    # a brute-force sample as well
    idx = np.arange(0, R.size, 997)
    assert np.array_equal(got[idx], o.locate_brute(R[idx], Z[idx]))


# ----------------------------------------------------------------------------- a3
@pytest.mark.parametrize("name,n", [("cfg1", 4096 + 37), ("cfg2", 70001), ("cfg5", 30011)])
def test_gather_parity(B, inputs, name, n):
    wl, o, ctx, _, coef = _setup(B, inputs, name)
    m = inputs.markers(wl, n=n)
    want = o.gather(m["R"], m["Z"], m["phi"])
    d = _dev(B, m)
    for hint in (None, torch.from_numpy(want["cell"]).cuda(), torch.zeros(n, dtype=torch.int32, device="cuda")):
        got = ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=hint)
        for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
            scale = np.abs(want[k]).max()
            e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
            assert e < 1e-12, (k, e)


@pytest.mark.parametrize("name,n", [("cfg2", 300007), ("cfg3", 270001)])
def test_gather_large_batches_sorted_and_unsorted(B, inputs, name, n):
    """Batches of 2^18 markers and more with hints: cell-sorted markers take the lane kernel (records in shared memory,
    inputs prefetched), anything else the thread-per-marker kernel; the device decides.  Hints: none, the true cells
    (unsorted), stale, sorted, sorted with a few markers out of place and flagged ones."""
    wl, o, ctx, _, coef = _setup(B, inputs, name)
    m = inputs.markers(wl, n=n)
    m["R"][::1013] = wl.R0 + 1.5 * wl.a                       # some markers outside the mesh
    want = o.gather(m["R"], m["Z"], m["phi"])
    d = _dev(B, m)
    cells = torch.from_numpy(want["cell"]).cuda()
    keys = ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi")

    def check(got, ref):
        for k in keys:
            e = rel_err(got[k].cpu().numpy(), ref[k], np.abs(ref[k]).max()).max()
            assert e < 1e-12, (k, e)

    for hint in (None, cells, torch.zeros(n, dtype=torch.int32, device="cuda")):
        check(ctx.gather(d["R"], d["Z"], d["phi"], cell_hint=hint), want)
    key = torch.where(cells < 0, torch.full_like(cells, wl.n_tri), cells)
    order = torch.argsort(key, stable=True)
    ds = {k: d[k][order].contiguous() for k in ("R", "Z", "phi")}
    hs = cells[order].contiguous()
    on = order.cpu().numpy()
    ref = {k: want[k][on] for k in keys}
    lost = want["cell"][on] < 0
    assert lost.sum() > 100
    got = ctx.gather(ds["R"], ds["Z"], ds["phi"], cell_hint=hs)           # lost markers (hint -1) at the end
    check(got, ref)
    for k in keys:
        assert np.all(got[k].cpu().numpy()[lost] == 0.0)
    h2 = hs.clone()
    h2[::777] = 0                                                          # a few stale hints: still "sorted enough"
    check(ctx.gather(ds["R"], ds["Z"], ds["phi"], cell_hint=h2), ref)
    g3 = ctx.gather(ds["R"], ds["Z"], ds["phi"], cell_hint=hs, want_dphi=False)
    assert "dphi_dphi" not in g3
    for k in keys[:3]:
        assert rel_err(g3[k].cpu().numpy(), ref[k], np.abs(ref[k]).max()).max() < 1e-12


# ----------------------------------------------------------------------------- a4 + a5
@pytest.mark.parametrize("name,n,variant,wmode", [("cfg1", 4096, 0, 0), ("cfg1", 1000, 1, 1), ("cfg2", 50021, 0, 0),
                                                  ("cfg3", 20011, 0, 0), ("cfg5", 20011, 0, 0)])
def test_rhs_parity(B, inputs, name, n, variant, wmode):
    wl, o, ctx, _, _ = _setup(B, inputs, name)
    o.set_params(wl.params(variant, wmode))
    ctx.set_params(wl.params(variant, wmode))
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng(3).standard_normal(n) * 1e-2
    want = o.rhs(m["R"], m["Z"], m["phi"], m["vpar"], m["mu"], m["w"])
    d = _dev(B, m)
    d["cell"] = ctx.locate(d["R"], d["Z"])
    assert np.array_equal(d["cell"].cpu().numpy(), want["cell"])
    got = ctx.rhs(d)
    for k in ("dRdt", "dZdt", "dphidt", "dvpardt", "dwdt"):
        scale = np.abs(want[k]).max()
        e = rel_err(got[k].cpu().numpy(), want[k], scale).max()
        assert e < 1e-12, (k, e)
    if name == "cfg5":
        lost = want["cell"] < 0
        assert lost.sum() > 0
        for k in ("dRdt", "dwdt"):
            assert np.all(got[k].cpu().numpy()[lost] == 0.0)


# ----------------------------------------------------------------------------- a6
def _push_both(B, inputs, name, n, nsteps, dt=None, **replace):
    wl, o, ctx, _, _ = _setup(B, inputs, name, **replace)
    m = inputs.markers(wl, n=n)
    if wl.sigma_w == 0.0:
        m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    dt = wl.dt if dt is None else dt
    want = o.push(m, dt, nsteps)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, dt, nsteps)
    return wl, o, ctx, m, want, _host(d)


def test_push_one_step_cfg1(B, inputs):
    wl, o, ctx, m, want, got = _push_both(B, inputs, "cfg1", 4096, 1)
    assert np.array_equal(got["cell"], want["cell"])
    assert np.array_equal(got["mu"], m["mu"])
    _assert_state_close(got, want, 1e-12, 1e-4)


def test_push_twenty_steps_cfg1(B, inputs):
    """BASELINE.json configs[0] in full: 4096 markers, dt = 0.05, 20 steps."""
    wl, o, ctx, m, want, got = _push_both(B, inputs, "cfg1", 4096, 20)
    _assert_state_close(got, want, 1e-9, 1e-4)
    # rule L5: a cell may differ only where the oracle's marker sits within 1e-10 of an edge
    diff = got["cell"] != want["cell"]
    if diff.any():
        b = o.bary(want["cell"][diff], want["R"][diff], want["Z"][diff])
        assert b.min(axis=1).max() < 1e-10
    assert diff.sum() == 0
    assert np.array_equal(got["mu"], m["mu"])
    assert np.abs(got["w"] - m["w"]).max() > 1e-6            # the weights evolved


@pytest.mark.parametrize("name,n,nsteps", [("cfg2", (1 << 16) + 13, 3), ("cfg3", 30011, 3), ("cfg5", 40009, 5)])
def test_push_parity_itg_meshes(B, inputs, name, n, nsteps):
    wl, o, ctx, m, want, got = _push_both(B, inputs, name, n, nsteps)
    assert np.array_equal(got["cell"] < 0, want["cell"] < 0)
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10, 1e-4)
    if name == "cfg5":
        nl = (want["cell"] < 0).sum()
        assert nl > 0
        assert ctx.get_stats()["n_lost"] >= 0


def test_push_lost_markers_flagged_and_restored(B, inputs):
    """Markers driven out of the mesh: restored to start-of-step state, cell = -1, skipped later."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", modes=())
    th = np.linspace(0, 2 * np.pi, 640, endpoint=False)
    r = 0.995 * math.cos(math.pi / 32)
    n = th.size
    m = dict(R=10.0 + r * np.cos(th), Z=r * np.sin(th), phi=np.zeros(n), vpar=0.3 * np.ones(n),
             mu=400.0 * np.ones(n), w=np.zeros(n))
    want = o.push(m, 0.05, 40)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.reset_stats()
    ctx.push(d, 0.05, 25)
    ctx.push(d, 0.05, 15)                 # flagged markers are skipped by the second call
    got = _host(d)
    assert np.array_equal(got["cell"] < 0, want["cell"] < 0)
    assert 50 < (got["cell"] < 0).sum() < 600
    _assert_state_close(got, want, 1e-9, 1.0)
    assert ctx.get_stats()["n_lost"] == (got["cell"] < 0).sum()
    assert np.array_equal(got["w"], m["w"])           # no field: weights bit-identical


def test_push_without_field_modes_keeps_weights(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", modes=())
    m = inputs.markers(wl, n=1000)
    m["w"] = np.random.default_rng(1).standard_normal(1000)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, 0.05, 10)
    got = _host(d)
    assert np.array_equal(got["w"], m["w"]) and np.array_equal(got["mu"], m["mu"])
    want = o.push(m, 0.05, 10)
    _assert_state_close(got, want, 1e-10, 1.0)


def test_push_full_chain_from_dofs(B, inputs):
    """DOFs -> library's own Bell expansion -> push, against the oracle's own chain."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", field="dofs")
    m = inputs.markers(wl)
    want = o.push(m, wl.dt, 20)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 20)
    _assert_state_close(_host(d), want, 1e-9, 1e-4)


def test_stale_and_garbage_hints_do_not_change_results(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg2")
    n = 20001
    m = inputs.markers(wl, n=n)
    want = o.push(m, wl.dt, 2)
    rng = np.random.default_rng(8)
    for hint in (rng.integers(0, wl.n_tri, n), np.zeros(n), np.full(n, wl.n_tri - 1), np.full(n, 2 ** 30)):
        d = _dev(B, dict(m, cell=hint.astype(np.int32)))
        ctx.push(d, wl.dt, 2)
        got = _host(d)
        assert np.array_equal(got["cell"], want["cell"])
        _assert_state_close(got, want, 1e-10, 1e-4)


def test_non_arithmetic_mode_list(B, inputs):
    """Mode lists that are not an arithmetic progression take the per-mode sincos path."""
    wl, o, ctx, dofs, coef = _setup(B, inputs, "cfg1", field=None, modes=(0, 1, 5))
    ctx.field_upload(wl.modes, torch.from_numpy(coef).cuda(), kind=1)
    m = inputs.markers(wl, n=3000)
    want = o.gather(m["R"], m["Z"], m["phi"])
    d = _dev(B, m)
    got = ctx.gather(d["R"], d["Z"], d["phi"])
    for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
        assert rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max() < 1e-12
    # arithmetic progression not starting at zero
    wl2, o2, ctx2, _, coef2 = _setup(B, inputs, "cfg1", field="oracle", modes=(3, 7, 11))
    want = o2.gather(m["R"], m["Z"], m["phi"])
    got = ctx2.gather(d["R"], d["Z"], d["phi"])
    for k in ("dphi", "dphi_dR", "dphi_dZ", "dphi_dphi"):
        assert rel_err(got[k].cpu().numpy(), want[k], np.abs(want[k]).max()).max() < 1e-12


# ----------------------------------------------------------------------------- push-kernel schedules
@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("name,n,nsteps,sort", [("cfg1", 4096, 20, False), ("cfg1", 1777, 3, True),
                                                ("cfg2", (1 << 16) + 13, 3, True), ("cfg5", 40009, 5, True),
                                                ("cfg3", 20011, 2, False)])
def test_push_kernel_variants_match_oracle(B, inputs, variant, name, n, nsteps, sort):
    """Every schedule of trimeg_push (trimeg_set_push_kernel) against the oracle: unsorted input
    (markers of a tile spread over the whole mesh: hash bins overflow, one-marker fallback) and
    cell-sorted input (the batched path), ragged tile tails, lost markers (cfg5)."""
    wl, o, ctx, _, _ = _setup(B, inputs, name)
    ctx.set_push_kernel(variant)
    m = inputs.markers(wl, n=n)
    if wl.sigma_w == 0.0:
        m["w"] = np.random.default_rng(5).standard_normal(n) * 1e-4
    want = o.push(m, wl.dt, nsteps)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    if sort:
        perm = ctx.sort(d, want_perm=True).cpu().numpy()
        want = {k: v[perm] for k, v in want.items()}
        mu0 = m["mu"][perm]
    else:
        mu0 = m["mu"]
    ctx.reset_stats()
    outside_at_start = int((d["cell"] < 0).sum())
    ctx.push(d, wl.dt, nsteps)
    got = _host(d)
    assert np.array_equal(got["cell"], want["cell"])
    assert np.array_equal(got["mu"], mu0)
    _assert_state_close(got, want, 1e-9 if nsteps > 5 else 1e-10, 1e-4)
    assert ctx.get_stats()["n_lost"] == int((want["cell"] < 0).sum()) - outside_at_start


@pytest.mark.parametrize("variant", [1, 2])
def test_push_kernel_schedules_edge_cases(B, inputs, variant):
    """No field modes (weights bit-identical), already-lost markers on input are left untouched,
    two calls equal one, non-arithmetic mode list."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", modes=())
    ctx.set_push_kernel(variant)
    m = inputs.markers(wl, n=1000)
    m["w"] = np.random.default_rng(1).standard_normal(1000)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    d["cell"][::7] = -1
    before = _host(d)
    ctx.push(d, 0.05, 10)
    got = _host(d)
    assert np.array_equal(got["w"], m["w"])
    dead = before["cell"] < 0
    for k in ("R", "Z", "phi", "vpar", "w", "cell"):
        assert np.array_equal(got[k][dead], before[k][dead]), k
    want = o.push({k: v[~dead] for k, v in m.items()}, 0.05, 10)
    _assert_state_close({k: v[~dead] for k, v in got.items()}, want, 1e-10, 1.0)
    # two calls of 3 + 4 steps equal one call of 7; non-arithmetic mode list
    wl2, o2, ctx2, dofs, coef = _setup(B, inputs, "cfg1", field=None, modes=(0, 1, 5))
    ctx2.field_upload(wl2.modes, torch.from_numpy(coef).cuda(), kind=1)
    ctx2.set_push_kernel(variant)
    m2 = inputs.markers(wl2, n=3001)
    want2 = o2.push(m2, wl2.dt, 7)
    d2 = _dev(B, m2)
    ctx2.locate(d2["R"], d2["Z"], cell=d2["cell"])
    ctx2.sort(d2)
    ctx2.push(d2, wl2.dt, 3)
    ctx2.push(d2, wl2.dt, 4)
    got2 = _host(d2)
    order_got = np.lexsort((got2["mu"], got2["vpar"] * 0))          # mu is a unique, untouched key
    order_want = np.lexsort((want2["mu"], want2["vpar"] * 0))
    _assert_state_close({k: v[order_got] for k, v in got2.items()}, {k: v[order_want] for k, v in want2.items()}, 1e-10, 1e-4)


# ----------------------------------------------------------------------------- a1 / a6 helpers
def test_sort_is_a_valid_cell_ordered_permutation(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5")
    n = 200003
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    before = _host(d)
    perm = ctx.sort(d, want_perm=True).cpu().numpy()
    after = _host(d)
    assert np.array_equal(np.sort(perm), np.arange(n))
    for k in before:
        assert np.array_equal(after[k], before[k][perm]), k
    key = np.where(after["cell"] < 0, wl.n_tri, after["cell"])
    assert np.all(np.diff(key) >= 0)
    assert (after["cell"] < 0).sum() > 0
    # pushing the sorted set gives, per original index, the same answer as the oracle
    want = o.push(m, wl.dt, 2)
    ctx.push(d, wl.dt, 2)
    got = _host(d)
    back = {k: np.empty_like(v) for k, v in got.items()}
    for k, v in got.items():
        back[k][perm] = v
    assert np.array_equal(back["cell"], want["cell"])
    _assert_state_close(back, want, 1e-10, 1e-4)


def test_compact_is_a_stable_partition(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5", field=None)
    n = 100001
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    before = _host(d)
    na, perm = ctx.compact(d, want_perm=True)
    perm = perm.cpu().numpy()
    after = _host(d)
    act = before["cell"] >= 0
    assert na == act.sum() and 0 < na < n
    want_perm = np.concatenate([np.where(act)[0], np.where(~act)[0]])
    assert np.array_equal(perm, want_perm)
    for k in before:
        assert np.array_equal(after[k], before[k][perm]), k


def test_push_host_equals_device_push(B, inputs):
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg2")
    n = (1 << 22) + 1001          # ragged tail; one chunk at this density (129 markers per triangle)
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    ctx.push(d, wl.dt, 2)
    dev = _host(d)
    h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
    h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
    ctx.push_host(h, wl.dt, 2, locate_first=True)
    for k in ("R", "Z", "phi", "vpar", "w", "cell", "mu"):
        assert np.array_equal(h[k].numpy(), dev[k]), k
    # and a sample against the oracle
    idx = np.arange(0, n, 257)
    want = o.push({k: m[k][idx] for k in m}, wl.dt, 2)
    _assert_state_close({k: dev[k][idx] for k in dev}, want, 1e-10, 1e-4)


# ----------------------------------------------------------------------------- edge cases
def test_empty_and_error_paths(B, inputs):
    wl = inputs.WORKLOADS["cfg1"]
    ctx = B.context_for(wl, inputs)
    m = inputs.markers(wl, n=64)
    d = _dev(B, m)
    with pytest.raises(B.TrimegError) as e:
        ctx.push(d, 0.05, 1)
    assert e.value.code == B.ERR_NO_FIELD
    with pytest.raises(B.TrimegError):
        ctx.rhs(d)
    ctx.field_upload([], None, kind=1)                       # n_modes = 0 is legal
    empty = {k: v[:0].contiguous() for k, v in d.items()}
    ctx.push(empty, 0.05, 3)                                 # n = 0
    ctx.sort(empty)
    assert ctx.compact(empty)[0] == 0
    ctx.push(d, 0.05, 0)                                     # nsteps = 0: no-op
    assert np.array_equal(d["R"].cpu().numpy(), m["R"])
    # all markers flagged lost: untouched
    d["cell"].fill_(-1)
    ctx.push(d, 0.05, 3)
    assert np.array_equal(d["R"].cpu().numpy(), m["R"])
    with pytest.raises(B.TrimegError) as e:
        B.Context(2, 3, [0.0, 0.9, 1.0], wl.params())
    assert e.value.code == B.ERR_MESH


def test_library_vertices_fallback_close_to_generator(B, inputs):
    """vert_R/vert_Z = NULL: the library places the vertices itself."""
    wl = inputs.WORKLOADS["cfg1"]
    r, Rv, Zv = inputs.mesh_nodes(wl)
    ctx = B.Context(wl.n_r, wl.n_theta, r, wl.params())
    g = ctx.mesh_download_geom().cpu().numpy()
    o = oracle.from_workload(wl, inputs)
    assert np.abs(g - o.geom()).max() < 1e-9 * np.abs(o.geom()).max()


# ----------------------------------------------------------------------------- full size, sampled
@pytest.mark.parametrize("name,nsteps", [("cfg5", 4)])
def test_full_size_sampled_parity_in_bench_configuration(B, inputs, name, nsteps):
    """BASELINE.json's 2^24-marker workload in the launch configuration bench.py times
    (locate -> sort -> push), checked on every 1024-th marker against the oracle."""
    wl, o, ctx, _, _ = _setup(B, inputs, name)
    n = wl.n_markers
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    perm = ctx.sort(d, want_perm=True)
    ctx.push(d, wl.dt, nsteps)
    idx = np.arange(0, n, 1024)
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(n, device="cuda")
    pos = inv[torch.from_numpy(idx).cuda()]
    got = {k: v[pos].cpu().numpy() for k, v in d.items()}
    want = o.push({k: m[k][idx] for k in m}, wl.dt, nsteps)
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10, 1e-4)
    assert (want["cell"] < 0).sum() > 0


@pytest.mark.parametrize("variant", [1, 2])
def test_push_keeps_slots_while_markers_stay_in_their_triangles(B, inputs, variant):
    """The warp-autonomous kernels group their markers by triangle anew only at a stage where a marker of the warp has
    changed its triangle.  With a tiny time step nobody moves: one grouping per warp in 40 stages; with a large one the
    grouping runs at most stages; the oracle's result either way (cell-sorted input, 10 RK4 steps)."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5")
    ctx.set_push_kernel(variant)
    n = 12011
    m = inputs.markers(wl, n=n)
    frac = {}
    for dt in (1e-7, 0.2):
        want = o.push(m, dt, 10)
        d = _dev(B, m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        perm = ctx.sort(d, want_perm=True).cpu().numpy()
        ctx.reset_stats()
        ctx.push(d, dt, 10)
        got = _host(d)
        assert np.array_equal(got["cell"], want["cell"][perm])
        _assert_state_close(got, {k: v[perm] for k, v in want.items()}, 1e-9, 1e-4)
        t = ctx.get_tile_counters()
        assert t["n_stages"] > 0 and t["n_stages"] % 40 == 0
        frac[dt] = t["n_regroup"] / t["n_stages"]        # [1] of trimeg_get_tile_counters: groupings per warp and stage
    assert frac[1e-7] <= 2.5 / 40                           # lane kernels: one look-up round per pass (two passes per stage)
    assert frac[0.2] > 0.2


# ----------------------------------------------------------------------------- schedule selection, diagnostics
def test_automatic_schedule_selection_and_variant_range(B, inputs):
    """TRIMEG_PUSH_KERNEL_AUTO resolves by the number of uploaded modes (plain warp kernel below 12 and above 26 -- its
    128-register build up to 4 --, warp kernel with shared-memory records in between); variants outside
    -1..TRIMEG_PUSH_KERNEL_MAX are rejected; AUTO gives the oracle's result like any fixed variant."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1")
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_LANE    # 2 modes
    for bad in (-2, 3, 100):
        with pytest.raises(B.TrimegError):
            ctx.set_push_kernel(bad)
    ctx.set_push_kernel(B.PUSH_KERNEL_WCACHE)
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_WCACHE
    ctx.set_push_kernel(B.PUSH_KERNEL_AUTO)
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_LANE
    _, _, ctx8, _, _ = _setup(B, inputs, "cfg1", modes=tuple(range(0, 16, 2)))
    assert ctx8.get_push_kernel() == B.PUSH_KERNEL_WCACHE   # 8 modes
    wl5, o5, ctx5, _, _ = _setup(B, inputs, "cfg5")
    assert ctx5.get_push_kernel() == B.PUSH_KERNEL_WCACHE
    m = inputs.markers(wl5, n=30011)
    want = o5.push(m, wl5.dt, 3)
    d = _dev(B, m)
    ctx5.locate(d["R"], d["Z"], cell=d["cell"])
    ctx5.push(d, wl5.dt, 3)
    got = _host(d)
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10, 1e-4)


def test_fp64_peak_depends_on_register_operands(B, inputs):
    """The roofline denominators of bench.py: a DFMA stream with three fresh register operands per instruction runs at
    2/3 of the rate of one with a single fresh operand; two fresh operands cost (almost) nothing."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1")
    p1, p2, p3 = (ctx.measure_fp64_peak_operands(k) for k in (1, 2, 3))
    p0 = ctx.measure_fp64_peak()
    assert 25.0 < p0 < 45.0
    assert 0.85 < p1 / p0 < 1.05 and 0.80 < p2 / p0 < 1.05
    assert 0.60 < p3 / p0 < 0.72
    with pytest.raises(B.TrimegError):
        ctx.measure_fp64_peak_operands(4)


@pytest.mark.parametrize("variant", [1, 2])
def test_push_many_modes_few_record_slots(B, inputs, variant):
    """32 toroidal modes: a coefficient record is 10.8 KB, the shared-memory record table has room for a dozen of them (the
    lane kernel: 8) and sends the other triangles' markers down the one-marker path; same results as the oracle either way."""
    modes = tuple(range(0, 64, 2))
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg1", modes=modes)
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_WCACHE    # automatic choice
    ctx.set_push_kernel(variant)
    m = inputs.markers(wl, n=6007)
    m["w"] = np.random.default_rng(7).standard_normal(6007) * 1e-4
    want = o.push(m, wl.dt, 3)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    perm = ctx.sort(d, want_perm=True).cpu().numpy()
    ctx.push(d, wl.dt, 3)
    got = _host(d)
    want = {k: v[perm] for k, v in want.items()}
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10, 1e-4)


def test_schedules_agree_bit_for_bit_on_the_many_mode_config(B, inputs):
    """The three schedules put every marker through the same operations in the same order (the
    two-phase mode loop of trimeg_lane.cuh, the grouping and the lane pairs of the many-mode kernel change which lane
    evaluates a marker and what its loads cost, not its arithmetic): on the cfg5 mesh with its 16 modes, cell-sorted
    markers, 3 RK4 steps, the states are bit-identical."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5")
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_WCACHE
    m = inputs.markers(wl, n=40009)
    results = []
    for variant in (B.PUSH_KERNEL_THREAD, B.PUSH_KERNEL_LANE, B.PUSH_KERNEL_WCACHE):
        ctx.set_push_kernel(variant)
        d = _dev(B, m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        perm = ctx.sort(d, want_perm=True).cpu().numpy()    # the order inside a triangle follows an atomic cursor: undo it
        ctx.push(d, wl.dt, 3)
        h = _host(d)
        back = {}
        for k, v in h.items():
            back[k] = np.empty_like(v)
            back[k][perm] = v
        results.append(back)
    for other in results[1:]:
        for k in ("R", "Z", "phi", "vpar", "w", "mu", "cell"):
            assert np.array_equal(results[0][k], other[k]), k


# ----------------------------------------------------------------------------- configs at their own sizes and step counts
def test_cfg3_full_size_sampled_parity(B, inputs):
    """BASELINE.json configs[2] at full size: 2^26 markers (3.5 GB) in memory order as drawn (unsorted), automatic
    schedule, 2 RK4 steps; every 4096-th marker against the oracle: cells bit-exact, state to 1e-10."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg3")
    n = wl.n_markers
    assert n == 1 << 26
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    assert ctx.get_push_kernel() == B.PUSH_KERNEL_LANE
    ctx.push(d, wl.dt, 2)
    idx = np.arange(0, n, 4096)
    tidx = torch.from_numpy(idx).cuda()
    got = {k: v[tidx].cpu().numpy() for k, v in d.items()}
    want = o.push({k: m[k][idx] for k in m}, wl.dt, 2)
    assert np.array_equal(got["cell"], want["cell"])
    _assert_state_close(got, want, 1e-10, 1e-4)
    assert np.array_equal(got["mu"], m["mu"][idx])


@pytest.mark.parametrize("name,n", [("cfg2", 20011), ("cfg3", 20011), ("cfg5", 40009)])
@pytest.mark.parametrize("path", ["push_sorted", "push_host"])
def test_twenty_steps_on_the_itg_meshes(B, inputs, name, n, path, monkeypatch):
    """north_star's 20-step bar (1e-9) on the cfg2 / cfg3 / cfg5 meshes with the automatic schedule: cell-sorted
    trimeg_push of 20 fused steps, and trimeg_push_host (sort -> 10 steps -> re-sort -> 10 steps -> unsort, three chunks)."""
    wl, o, ctx, _, _ = _setup(B, inputs, name)
    m = inputs.markers(wl, n=n)
    want = o.push(m, wl.dt, 20)
    if path == "push_sorted":
        d = _dev(B, m)
        ctx.locate(d["R"], d["Z"], cell=d["cell"])
        perm = ctx.sort(d, want_perm=True).cpu().numpy()
        ctx.push(d, wl.dt, 20)
        raw = _host(d)
        got = {k: np.empty_like(v) for k, v in raw.items()}
        for k, v in raw.items():
            got[k][perm] = v
    else:
        monkeypatch.setenv("TRIMEG_HOST_CHUNKS", "3")
        h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
        h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
        ctx.push_host(h, wl.dt, 20, locate_first=True)
        got = {k: v.numpy() for k, v in h.items()}
    assert np.array_equal(got["cell"] < 0, want["cell"] < 0)
    diff = got["cell"] != want["cell"]
    if diff.any():                                       # rule L5
        b = o.bary(want["cell"][diff], want["R"][diff], want["Z"][diff])
        assert b.min(axis=1).max() < 1e-10
    assert diff.sum() == 0
    _assert_state_close(got, want, 1e-9, 1e-4)
    assert np.array_equal(got["mu"], m["mu"])
    if name == "cfg5":
        assert (want["cell"] < 0).sum() > 0


def test_push_host_resort_path_with_lost_markers(B, inputs, monkeypatch):
    """trimeg_push_host over 25 steps (sort, 10, re-sort, 10, re-sort, 5, unsort) on the cfg5 mesh with markers that
    leave the mesh on the way: equals, bit for bit and per caller index, cell sort + trimeg_push of 10 + 10 + 5 steps,
    whatever the number of chunks; a sample against the oracle."""
    wl, o, ctx, _, _ = _setup(B, inputs, "cfg5")
    n = 150001
    m = inputs.markers(wl, n=n)
    d = _dev(B, m)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    for k in (10, 10, 5):
        ctx.push(d, wl.dt, k)
    dev = _host(d)
    assert 0 < (dev["cell"] < 0).sum() < n // 10
    for chunks in ("1", "4"):
        monkeypatch.setenv("TRIMEG_HOST_CHUNKS", chunks)
        h = {k: torch.from_numpy(np.array(m[k])).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
        h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
        ctx.push_host(h, wl.dt, 25, locate_first=True)
        for k in ("R", "Z", "phi", "vpar", "w", "cell", "mu"):
            assert np.array_equal(h[k].numpy(), dev[k]), (chunks, k)
    idx = np.arange(0, n, 37)
    want = o.push({k: m[k][idx] for k in m}, wl.dt, 25)
    assert np.array_equal(dev["cell"][idx], want["cell"])
    _assert_state_close({k: dev[k][idx] for k in dev}, want, 1e-9, 1e-4)
    ctx.release_host_buffers()
    with pytest.raises(B.TrimegError):
        ctx.push_host(h, float("nan"), 1, locate_first=True)


def test_two_contexts_on_two_devices(B, inputs):
    """Function attributes (the opt-in to > 48 KB of dynamic shared memory) are per device, and every call runs on its
    context's device whatever device is current: two contexts on two GPUs in one process, many-mode kernel on both."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    wl = inputs.WORKLOADS["cfg5"]
    o = oracle.from_workload(wl, inputs)
    coef = o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    m = inputs.markers(wl, n=20011)
    want = o.push(m, wl.dt, 2)
    ctxs = []
    for dev in (0, 1):
        torch.cuda.set_device(dev)
        c = B.context_for(wl, inputs)
        c.field_upload(wl.modes, torch.from_numpy(coef).cuda(dev), kind=1)
        c.set_push_kernel(B.PUSH_KERNEL_WCACHE)
        ctxs.append(c)
    torch.cuda.set_device(0)                             # device 0 stays current for both pushes
    for dev, c in enumerate(ctxs):
        d = B.markers_to_device(m, f"cuda:{dev}")
        with torch.cuda.device(dev):
            s = torch.cuda.current_stream(dev)
        c.locate(d["R"], d["Z"], cell=d["cell"], stream=s)
        c.push(d, wl.dt, 2, stream=s)
        torch.cuda.synchronize(dev)
        got = _host(d)
        assert np.array_equal(got["cell"], want["cell"])
        _assert_state_close(got, want, 1e-10, 1e-4)
