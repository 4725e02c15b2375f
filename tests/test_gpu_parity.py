"""GPU parity: the CUDA path, called through the C ABI (include/pic.h), against the CPU oracle on
the same seeded inputs.  perm and cell_offsets bit-exact; rho, x, v within north_star's tolerances.
"""
import numpy as np
import pytest

import pic_workloads as W
from parity import TOL_RHO, TOL_XV, err_rho, err_v, err_x, to_dev, to_host

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _mods():
    import oracle as O
    import paper_1603_02886_b200 as B
    return O, B


# sizes span several radix tiles (4096) and scan tiles (2048) plus a ragged tail
SMALL = [
    ("cfg1", dict()),                                           # 2-D 64^2, 1e5, f64, p=1 (full size)
    ("cfg2", dict(N=3 * 4096 + 77)),
    ("cfg2", dict(N=200_003, n=(64, 64))),
    ("cfg3", dict(N=150_001, n=(32, 32, 32))),
    ("cfg3", dict(N=40_000, n=(16, 8, 4))),
    ("cfg4", dict(N=300_007, n=(32, 32, 32))),
    ("cfg5", dict(N=8 * 16 ** 3 + 5, n=(16, 16, 16))),
]
ORDERS = [1, 2, 3]


def _cfg(name, kw, order=None, dtype=None):
    cfg = W.CONFIGS[name]
    kw = dict(kw)
    N = kw.pop("N", cfg.N)
    cfg = cfg.scaled(N, **kw)
    if order is not None:
        cfg = cfg.scaled(N, order=order)
    if dtype is not None:
        cfg = cfg.scaled(N, dtype=dtype)
    return cfg


def _gpu_sort(B, g, wl):
    n = wl.cfg.N
    x, v = to_dev(wl.x), to_dev(wl.v)
    w = to_dev([wl.w])[0]
    xo = [torch.empty_like(a) for a in x]
    vo = [torch.empty_like(a) for a in v]
    wo = torch.empty_like(w)
    perm = torch.full((max(n, 4),), -1, dtype=torch.int32, device="cuda")
    off = torch.full((g.cells + 4,), -1, dtype=torch.int32, device="cuda")
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    B.pic_sort(g, x, v, w, xo, vo, wo, perm, off, ws)
    torch.cuda.synchronize()
    return xo, vo, wo, perm[:n], off[: g.cells + 1]


@pytest.mark.parametrize("name,kw", SMALL)
def test_sort_bit_exact(name, kw):
    O, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    ro = O.sort(O.grid_of(cfg), wl.x, wl.v, wl.w)
    xo, vo, wo, perm, off = _gpu_sort(B, B.grid_of(cfg), wl)
    assert np.array_equal(perm.cpu().numpy(), ro[3])
    assert np.array_equal(off.cpu().numpy(), ro[4])
    for c in range(cfg.dim):
        assert np.array_equal(xo[c].cpu().numpy(), ro[0][c])
        assert np.array_equal(vo[c].cpu().numpy(), ro[1][c])
    assert np.array_equal(wo.cpu().numpy(), ro[2])
    assert B.pic_last_launch_count() >= 5


@pytest.mark.parametrize("N", [0, 1, 31, 32, 33, 4095, 4096, 4097, 8192])
def test_sort_edge_sizes(N):
    O, B = _mods()
    cfg = _cfg("cfg2", dict(N=N, n=(16, 16)))
    wl = W.make_workload(cfg)
    ro = O.sort(O.grid_of(cfg), wl.x, wl.v, wl.w)
    xo, vo, wo, perm, off = _gpu_sort(B, B.grid_of(cfg), wl)
    assert np.array_equal(perm.cpu().numpy(), ro[3])
    assert np.array_equal(off.cpu().numpy(), ro[4])
    assert np.array_equal(xo[0].cpu().numpy(), ro[0][0])


def test_sort_degenerate_inputs():
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=50_000, n=(16, 16, 16)))
    wl = W.make_workload(cfg)
    # (a) every particle in one cell  (b) already sorted  (c) reverse sorted  (d) positions on cell faces and at x = L-ulp
    one = [np.full(cfg.N, 3.25, np.float32) + (np.arange(cfg.N) % 7).astype(np.float32) * 0.1 for _ in range(3)]
    for x in (one, None, "rev", "faces"):
        if x is None:
            xs, vs, wsrt, _, _ = O.sort(O.grid_of(cfg), wl.x, wl.v, wl.w)
            wl2 = W.Workload(cfg, xs, vs, wsrt, wl.E, wl.modes)
        elif isinstance(x, str) and x == "rev":
            xs, vs, wsrt, _, _ = O.sort(O.grid_of(cfg), wl.x, wl.v, wl.w)
            wl2 = W.Workload(cfg, [a[::-1].copy() for a in xs], [a[::-1].copy() for a in vs], wsrt[::-1].copy(), wl.E, wl.modes)
        elif isinstance(x, str):
            xf = [np.floor(a).astype(np.float32) for a in wl.x]
            xf[0][::3] = np.nextafter(np.float32(16.0), np.float32(0.0))
            xf[1][::5] = 0.0
            wl2 = W.Workload(cfg, xf, wl.v, wl.w, wl.E, wl.modes)
        else:
            wl2 = W.Workload(cfg, x, wl.v, wl.w, wl.E, wl.modes)
        ro = O.sort(O.grid_of(cfg), wl2.x, wl2.v, wl2.w)
        xo, vo, wo, perm, off = _gpu_sort(B, B.grid_of(cfg), wl2)
        assert np.array_equal(perm.cpu().numpy(), ro[3])
        assert np.array_equal(off.cpu().numpy(), ro[4])


def _gpu_sort_hint(B, g, x, v, w, hint):
    """pic_sort with cell_offsets pre-filled with `hint` (the library reads it as the order hint)."""
    n = w.shape[0]
    xd, vd, wd = to_dev(x), to_dev(v), to_dev([w])[0]
    xo = [torch.empty_like(a) for a in xd]
    vo = [torch.empty_like(a) for a in vd]
    wo = torch.empty_like(wd)
    perm = torch.full((max(n, 4),), -1, dtype=torch.int32, device="cuda")
    off = torch.from_numpy(np.concatenate([hint.astype(np.int32), np.zeros(3, np.int32)])).cuda()
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    B.pic_sort(g, xd, vd, wd, xo, vo, wo, perm, off, ws)
    torch.cuda.synchronize()
    return perm[:n].cpu().numpy(), off[: g.cells + 1].cpu().numpy(), xo


@pytest.mark.parametrize("name,kw", [
    ("cfg2", dict(N=200_003, n=(64, 64))),
    ("cfg3", dict(N=150_001, n=(32, 32, 32))),
    ("cfg4", dict(N=300_007, n=(32, 32, 32))),
    ("cfg5", dict(N=8 * 16 ** 3 + 5, n=(16, 16, 16))),
    ("cfg3", dict(N=5_000, n=(32, 32, 32))),          # far fewer particles than cells: long runs of empty cells
])
def test_sort_with_order_hint(name, kw):
    """Whatever cell_offsets holds on entry, the result is the unique stable permutation (R7)."""
    O, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    r1 = O.step(go, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm)            # sorted at t, pushed to t+1
    r2 = O.step(go, r1["x"], r1["v"], r1["w"], wl.E, cfg.dt, cfg.qm)    # sorted at t+1, pushed to t+2
    x, v, w = r2["x"], r2["v"], r2["w"]                                # order = cells at t+1
    ref = O.sort(go, x, v, w)
    C, n = gb.cells, cfg.N
    rng = np.random.default_rng(5)
    hints = {
        "previous offsets (steady state)": r2["cell_offsets"],
        "offsets of two steps ago": r1["cell_offsets"],
        "the new offsets themselves": ref[4],
        "all zero": np.zeros(C + 1, np.int64),
        "all N": np.full(C + 1, n, np.int64),
        "random non-decreasing": np.sort(rng.integers(0, n + 1, C + 1)),
        "random, not monotone": rng.integers(0, n + 1, C + 1),
        "out of range": np.arange(C + 1, dtype=np.int64) * 7 - 3,
        "one interval holds everything": np.concatenate([np.zeros(C // 2 + 1, np.int64), np.full(C - C // 2, n, np.int64)]),
    }
    for what, hint in hints.items():
        perm, off, xo = _gpu_sort_hint(B, gb, x, v, w, np.asarray(hint))
        assert np.array_equal(off, ref[4]), what
        assert np.array_equal(perm, ref[3]), what
        assert np.array_equal(xo[0].cpu().numpy(), ref[0][0]), what
    # an input that is already sorted, with its own offsets as the hint: identity
    xs, vs, wsrt, _, offs = ref
    perm, off, _ = _gpu_sort_hint(B, gb, xs, vs, wsrt, offs)
    assert np.array_equal(perm, np.arange(n, dtype=np.int32)) and np.array_equal(off, offs)


@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("name,kw", SMALL)
def test_deposit_parity(name, kw, order):
    O, B = _mods()
    cfg = _cfg(name, kw, order=order)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    rho_ref = O.deposit(go, wl.x, wl.w)
    x, w = to_dev(wl.x), to_dev([wl.w])[0]
    rho = torch.full((gb.cells,), 123.0, dtype=gb.torch_dtype, device="cuda")      # must be overwritten
    ws = torch.empty(B.pic_workspace_bytes(gb, cfg.N), dtype=torch.uint8, device="cuda")
    B.pic_deposit(gb, x, w, rho, B.PIC_ORDER_UNSORTED, None, ws)
    assert err_rho(rho.cpu().numpy(), rho_ref) <= TOL_RHO[cfg.dtype]
    # sorted path
    xs, vs, wsrt, perm, off = O.sort(go, wl.x, wl.v, wl.w)
    rho_ref_s = O.deposit(go, xs, wsrt)
    xd, wd = to_dev(xs), to_dev([wsrt])[0]
    offd = torch.from_numpy(np.concatenate([off, np.zeros(3, np.int32)])).cuda()
    rho.fill_(-7.0)
    B.pic_deposit(gb, xd, wd, rho, B.PIC_ORDER_SORTED, offd, ws)
    r = rho.cpu().numpy()
    assert err_rho(r, rho_ref_s) <= TOL_RHO[cfg.dtype]
    # exact conservation holds at any size: sum rho h^d = sum w
    tot = float(np.sum(wl.w.astype(np.float64)))
    assert abs(float(np.sum(r.astype(np.float64))) * cfg.h ** cfg.dim - tot) <= (1e-12 if cfg.dtype == "f64" else 2e-6) * tot


@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("name,kw", SMALL)
def test_push_parity(name, kw, order):
    O, B = _mods()
    cfg = _cfg(name, kw, order=order)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    xr, vr = O.push(go, wl.x, wl.v, wl.E, cfg.dt, cfg.qm)
    x, v, E = to_dev(wl.x), to_dev(wl.v), to_dev(wl.E)
    B.pic_push(gb, x, v, E, cfg.dt, cfg.qm)
    for c in range(cfg.dim):
        xg, vg = x[c].cpu().numpy(), v[c].cpu().numpy()
        assert err_x(xg, xr[c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(vg, vr[c]) <= TOL_XV[cfg.dtype]
        assert np.all((xg >= 0) & (xg < cfg.np_dtype(cfg.L[c])))
    # sorted input goes through the sorted path
    xs, vs, wsrt, perm, off = O.sort(go, wl.x, wl.v, wl.w)
    xr, vr = O.push(go, xs, vs, wl.E, cfg.dt, cfg.qm)
    x, v = to_dev(xs), to_dev(vs)
    offd = torch.from_numpy(np.concatenate([off, np.zeros(3, np.int32)])).cuda()
    B.pic_push(gb, x, v, E, cfg.dt, cfg.qm, B.PIC_ORDER_SORTED, offd)
    for c in range(cfg.dim):
        assert err_x(x[c].cpu().numpy(), xr[c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(v[c].cpu().numpy(), vr[c]) <= TOL_XV[cfg.dtype]


def _lockstep(cfg, steps, sort_every=1):
    """GPU step k is fed the oracle's state after step k-1 (reading R19)."""
    O, B = _mods()
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    x, v, w = wl.x, wl.v, wl.w
    E = to_dev(wl.E)
    n = cfg.N
    ws = torch.empty(B.pic_workspace_bytes(gb, n), dtype=torch.uint8, device="cuda")
    off_ref = None
    for k in range(steps):
        do_sort = (k % sort_every) == 0
        ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm, do_sort=do_sort, cell_offsets=off_ref)
        xi, vi, wi = to_dev(x), to_dev(v), to_dev([w])[0]
        xo = [torch.empty_like(a) for a in xi]
        vo = [torch.empty_like(a) for a in vi]
        wo = torch.empty_like(wi)
        perm = torch.full((max(n, 4),), -1, dtype=torch.int32, device="cuda")
        if do_sort or off_ref is None:
            off = torch.full((gb.cells + 4,), -1, dtype=torch.int32, device="cuda")
        else:
            off = torch.from_numpy(np.concatenate([off_ref, np.zeros(3, np.int32)])).cuda()
        rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
        B.pic_step(gb, xi, vi, wi, xo, vo, wo, perm, off if (do_sort or off_ref is not None) else None, rho, E,
                   cfg.dt, cfg.qm, do_sort, ws)
        torch.cuda.synchronize()
        if do_sort:
            assert np.array_equal(perm[:n].cpu().numpy(), ref["perm"]), "perm differs at step %d" % k
            assert np.array_equal(off[: gb.cells + 1].cpu().numpy(), ref["cell_offsets"])
            off_ref = ref["cell_offsets"]
        assert err_rho(rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[cfg.dtype], "rho at step %d" % k
        for c in range(cfg.dim):
            assert err_x(xo[c].cpu().numpy(), ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype], "x at step %d" % k
            assert err_v(vo[c].cpu().numpy(), ref["v"][c]) <= TOL_XV[cfg.dtype], "v at step %d" % k
        assert np.array_equal(wo.cpu().numpy(), ref["w"])
        x, v, w = ref["x"], ref["v"], ref["w"]


@pytest.mark.parametrize("name,kw,steps", [
    ("cfg1", dict(), 1),
    ("cfg2", dict(N=300_000, n=(64, 64)), 10),
    ("cfg3", dict(N=400_000, n=(32, 32, 32)), 10),
    ("cfg4", dict(N=400_000, n=(32, 32, 32)), 10),
    ("cfg5", dict(N=32 * 16 ** 3, n=(16, 16, 16)), 6),
])
def test_step_lockstep(name, kw, steps):
    _lockstep(_cfg(name, kw), steps)


@pytest.mark.parametrize("k", [4, 16])
def test_step_lockstep_sort_every_k(k):
    # config 5's sort-every-k arm: steps between sorts run on the stale order and must stay exact
    _lockstep(_cfg("cfg5", dict(N=8 * 16 ** 3, n=(16, 16, 16))), 18, sort_every=k)


@pytest.mark.parametrize("name,kw", [("cfg2", dict(N=200_000, n=(64, 64))), ("cfg3", dict(N=300_000, n=(32, 32, 32)))])
def test_step_free_running_by_particle_id(name, kw):
    """10 steps without re-feeding the oracle state: compare by particle identity (composition of perms)."""
    O, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    st = B.Stepper(gb, wl.x, wl.v, wl.w, wl.E)
    ident_g = torch.arange(cfg.N, device="cuda")
    x, v, w = wl.x, wl.v, wl.w
    ident_r = np.arange(cfg.N)
    for _ in range(10):
        st.step(cfg.dt, cfg.qm, True)
        ident_g = ident_g[st.perm[: cfg.N].long()]
        r = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        ident_r = ident_r[r["perm"]]
        x, v, w = r["x"], r["v"], r["w"]
    ig = ident_g.cpu().numpy()
    inv_g, inv_r = np.empty_like(ig), np.empty_like(ident_r)
    inv_g[ig] = np.arange(cfg.N)
    inv_r[ident_r] = np.arange(cfg.N)
    # a 1-ulp difference can move a particle across a cell face and change later perms; x and v by id must still agree
    # (ten free-running steps: still within the stated one-step tolerance -- achieved on B200 2.2e-16 / 2.8e-16 in
    # fp64 and 1.8e-7 / 1.5e-7 in fp32 (round 3; it was 10 x the tolerance before).  The achieved error is printed:
    # pytest -s or -rP shows it)
    ex = max(err_x(st.cur["x"][c].cpu().numpy()[inv_g], x[c][inv_r], cfg.L[c]) for c in range(cfg.dim))
    ev = max(err_v(st.cur["v"][c].cpu().numpy()[inv_g], v[c][inv_r]) for c in range(cfg.dim))
    print("free-running %s: achieved err_x %.3g, err_v %.3g; tolerance %.0e"
          % (name, ex, ev, TOL_XV[cfg.dtype]))
    assert ex <= TOL_XV[cfg.dtype]
    assert ev <= TOL_XV[cfg.dtype]
    mism = int(np.sum(ig != ident_r))
    assert mism <= (0 if cfg.dtype == "f64" else cfg.N // 1000), "order mismatches: %d" % mism


def test_step_host_entry_point():
    O, B = _mods()
    cfg = _cfg("cfg2", dict(N=50_001, n=(32, 32)))
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    ref = O.step(go, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm)
    xo = [np.empty_like(a) for a in wl.x]
    vo = [np.empty_like(a) for a in wl.v]
    wo = np.empty_like(wl.w)
    perm = np.empty(cfg.N, np.int32)
    off = np.empty(gb.cells + 1, np.int32)
    rho = np.empty(gb.cells, cfg.np_dtype)
    dws = torch.empty(B.pic_step_host_bytes(gb, cfg.N), dtype=torch.uint8, device="cuda")
    B.pic_step_host(gb, wl.x, wl.v, wl.w, xo, vo, wo, perm, off, rho, wl.E, cfg.dt, cfg.qm, True, dws)
    assert np.array_equal(perm, ref["perm"]) and np.array_equal(off, ref["cell_offsets"])
    assert err_rho(rho, ref["rho"]) <= TOL_RHO[cfg.dtype]
    for c in range(cfg.dim):
        assert err_x(xo[c], ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(vo[c], ref["v"][c]) <= TOL_XV[cfg.dtype]


def test_argument_validation():
    O, B = _mods()
    g = B.Grid(2, (16, 16), (1.0, 1.0), 1, "f64")
    n = 100
    x = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    w = torch.ones(n, dtype=torch.float64, device="cuda")
    rho = torch.zeros(g.cells, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PicError):
        B.pic_deposit(B.Grid(2, (16, 16), (1.0, 1.0), 4, "f64"), x, w, rho)          # order 4
    with pytest.raises(B.PicError):
        B.pic_deposit(B.Grid(2, (2, 16), (1.0, 1.0), 3, "f64"), x, w, torch.zeros(32, dtype=torch.float64, device="cuda"))
    with pytest.raises(B.PicError):
        B.pic_deposit(B.Grid(2, (16, 16), (0.0, 1.0), 1, "f64"), x, w, rho)          # h = 0
    ws = torch.empty(16, dtype=torch.uint8, device="cuda")                            # workspace too small
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    off = torch.empty(g.cells + 1, dtype=torch.int32, device="cuda")
    with pytest.raises(B.PicError, match="workspace"):
        B.pic_sort(g, x, x, w, [torch.empty_like(a) for a in x], [torch.empty_like(a) for a in x],
                   torch.empty_like(w), perm, off, ws)
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    with pytest.raises(B.PicError):                                                   # in aliases out
        B.pic_sort(g, x, x, w, x, x, w, perm, off, ws)


@pytest.mark.parametrize("kind", ["garbage", "not_covering", "stale"])
def test_step_without_sort_any_cell_offsets(kind):
    """pic_step(do_sort = 0) must be exact whatever cell_offsets holds: the step kernel finds the runs of equal
    cell key itself (cell_offsets only says "the order is that of an earlier sort") and sets the particles
    that sit alone between other cells' particles aside for the threads-on-particles kernel."""
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=150_000, n=(32, 32, 32)))
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    x, v, w = wl.x, wl.v, wl.w
    if kind == "stale":                       # sort, then advance twice without telling the offsets
        r = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        off_host = r["cell_offsets"].copy()
        x, v, w = r["x"], r["v"], r["w"]
        r = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm, do_sort=False, cell_offsets=off_host)
        x, v, w = r["x"], r["v"], r["w"]
    elif kind == "garbage":
        off_host = np.random.default_rng(3).integers(-5, n + 5, gb.cells + 1).astype(np.int32)
    else:                                     # non-decreasing but off[C] != N: would skip particles
        off_host = np.sort(np.random.default_rng(4).integers(0, n // 2, gb.cells + 1)).astype(np.int32)
        off_host[0] = 0
    ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm, do_sort=False, cell_offsets=off_host)
    xi, vi, wi = to_dev(x), to_dev(v), to_dev([w])[0]
    off = torch.from_numpy(np.concatenate([off_host, np.zeros(3, np.int32)])).cuda()
    rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
    ws = torch.empty(B.pic_workspace_bytes(gb, n), dtype=torch.uint8, device="cuda")
    B.pic_step(gb, xi, vi, wi, xi, vi, wi, None, off, rho, to_dev(wl.E), cfg.dt, cfg.qm, False, ws)
    torch.cuda.synchronize()
    assert np.array_equal(off[: gb.cells + 1].cpu().numpy(), off_host)          # not modified
    assert err_rho(rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[cfg.dtype]
    for c in range(cfg.dim):
        assert err_x(xi[c].cpu().numpy(), ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(vi[c].cpu().numpy(), ref["v"][c]) <= TOL_XV[cfg.dtype]


@pytest.mark.parametrize("drift_dt", [0.1, 0.6])
@pytest.mark.parametrize("name,kw,order", [
    ("cfg2", dict(N=150_000, n=(48, 40)), 2),
    ("cfg3", dict(N=200_000, n=(24, 20, 12)), 3),
    ("cfg3", dict(N=120_000, n=(16, 16, 16), dtype="f64"), 1),
    ("cfg5", dict(N=60 * 12 ** 3, n=(12, 12, 12)), 2),
])
def test_stale_order_deposit_push_step(name, kw, order, drift_dt):
    """PIC_ORDER_STALE on pic_deposit and pic_push, and pic_step(do_sort = 0): particles sorted three pushes ago.
    With drift_dt = 0.1 about half of them have left their cell (config 5's sort-every-4 arm); with 0.6 nearly
    all have, so almost every particle is a lone stray between others (the k_strays path).  Results do not depend
    on the order: the oracle's deposit / push / step on the same arrays are the reference."""
    O, B = _mods()
    cfg = _cfg(name, kw, order=order)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    x, v, w, perm, off_host = O.sort(go, wl.x, wl.v, wl.w)
    for _ in range(3):
        x, v = O.push(go, x, v, wl.E, drift_dt, cfg.qm)
    E = to_dev(wl.E)
    off = torch.from_numpy(np.concatenate([off_host, np.zeros(3, np.int32)])).cuda()
    ws = torch.empty(B.pic_workspace_bytes(gb, n), dtype=torch.uint8, device="cuda")
    rho = torch.full((gb.cells,), 9.0, dtype=gb.torch_dtype, device="cuda")
    # deposit
    B.pic_deposit(gb, to_dev(x), to_dev([w])[0], rho, B.PIC_ORDER_STALE, off, ws)
    rho_ref = O.deposit(go, x, w)
    assert err_rho(rho.cpu().numpy(), rho_ref) <= TOL_RHO[cfg.dtype]
    # push
    xr, vr = O.push(go, x, v, wl.E, cfg.dt, cfg.qm)
    xd, vd = to_dev(x), to_dev(v)
    B.pic_push(gb, xd, vd, E, cfg.dt, cfg.qm, B.PIC_ORDER_STALE, off)
    for c in range(cfg.dim):
        assert err_x(xd[c].cpu().numpy(), xr[c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(vd[c].cpu().numpy(), vr[c]) <= TOL_XV[cfg.dtype]
    # step without sort, in place
    ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm, do_sort=False, cell_offsets=off_host)
    xi, vi, wi = to_dev(x), to_dev(v), to_dev([w])[0]
    rho.fill_(-3.0)
    B.pic_step(gb, xi, vi, wi, xi, vi, wi, None, off, rho, E, cfg.dt, cfg.qm, False, ws)
    torch.cuda.synchronize()
    assert err_rho(rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[cfg.dtype]
    tot = float(np.sum(w.astype(np.float64)))
    assert abs(float(rho.double().sum()) * cfg.h ** cfg.dim - tot) <= (1e-12 if cfg.dtype == "f64" else 2e-6) * tot
    for c in range(cfg.dim):
        assert err_x(xi[c].cpu().numpy(), ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
        assert err_v(vi[c].cpu().numpy(), ref["v"][c]) <= TOL_XV[cfg.dtype]
    assert np.array_equal(wi.cpu().numpy(), w)


@pytest.mark.parametrize("h", [0.5, 0.3, 3.0])
@pytest.mark.parametrize("name,kw", [("cfg2", dict(N=60_000, n=(48, 40))), ("cfg3", dict(N=90_000, n=(24, 20, 12)))])
def test_step_lockstep_grid_spacing(name, kw, h):
    """Spacing h != 1 (reading R13): a power of two takes the multiply path, 0.3 and 3.0 the IEEE division
    in the storage precision; grids whose sizes are not powers of two; three steps in lockstep."""
    _lockstep(_cfg(name, dict(kw, h=h)), 3)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("case", ["one_cell", "minimal_grid", "fast", "edges"])
def test_step_degenerate(case, dtype):
    """The degenerate cases of the method: every particle in one cell (one long run cut into pieces), the
    smallest legal grid (n = p + 1: the stencil covers the whole grid), velocities that cross many boxes per
    step, particles exactly on 0 and on the last representable position below L."""
    O, B = _mods()
    rng = np.random.default_rng(5)
    dt_np = np.float64 if dtype == "f64" else np.float32
    order = 3
    n = (4, 4, 4) if case == "minimal_grid" else (12, 10, 8)
    N = 20_000
    cfg = W.CONFIGS["cfg3"].scaled(N, n=n, dtype=dtype, order=order)
    L = np.array(n, np.float64)
    x = [(rng.random(N) * L[c]).astype(dt_np) for c in range(3)]
    v = [rng.normal(0, 1, N).astype(dt_np) for c in range(3)]
    if case == "one_cell":
        x = [(3.0 + rng.random(N)).astype(dt_np) for c in range(3)]
    if case == "fast":
        # many boxes per step (a particle that leaves the box is advanced in double and rounded once, like O4)
        v = [rng.normal(0, 400, N).astype(dt_np) for c in range(3)]
    if case == "edges":
        for c in range(3):
            x[c][0::4] = 0
            x[c][1::4] = np.nextafter(dt_np(L[c]), dt_np(0))
    for c in range(3):
        x[c][x[c] >= L[c]] = 0
    w = (0.5 + rng.random(N)).astype(dt_np)
    E = [rng.normal(0, 1, cfg.cells).astype(dt_np) for c in range(3)]
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    ref = O.step(go, x, v, w, E, cfg.dt, cfg.qm)
    xi, vi, wi = to_dev(x), to_dev(v), to_dev([w])[0]
    xo, vo, wo = [torch.empty_like(a) for a in xi], [torch.empty_like(a) for a in vi], torch.empty_like(wi)
    perm = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    off = torch.full((gb.cells + 4,), -1, dtype=torch.int32, device="cuda")
    rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
    ws = torch.empty(B.pic_workspace_bytes(gb, N), dtype=torch.uint8, device="cuda")
    for rep in range(2):          # second call: cell_offsets now holds a valid hint for the same input
        B.pic_step(gb, xi, vi, wi, xo, vo, wo, perm, off, rho, to_dev(E), cfg.dt, cfg.qm, True, ws)
        torch.cuda.synchronize()
        assert np.array_equal(perm.cpu().numpy(), ref["perm"])
        assert np.array_equal(off[: gb.cells + 1].cpu().numpy(), ref["cell_offsets"])
        assert err_rho(rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[dtype]
        for c in range(3):
            assert err_x(xo[c].cpu().numpy(), ref["x"][c], L[c]) <= TOL_XV[dtype]
            assert err_v(vo[c].cpu().numpy(), ref["v"][c], sigma_v=max(1.0, float(np.max(np.abs(ref["v"][c]))))) <= TOL_XV[dtype]
            xs = xo[c].cpu().numpy()
            assert xs.min() >= 0 and xs.max() < L[c]


@pytest.mark.parametrize("seed", range(24))
def test_step_random_shapes(seed):
    """Seeded random combinations of dimension, spline order, dtype, grid sizes (down to n = p + 1, odd sizes),
    spacing, particle count (ragged tails), clustered or uniform: two steps in lockstep against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    dim = int(rng.integers(2, 4))
    order = int(rng.integers(1, 4))
    dtype = "f64" if rng.random() < 0.5 else "f32"
    n = tuple(int(rng.integers(order + 1, 40 if dim == 2 else 14)) for _ in range(dim))
    N = int(rng.integers(1, 60_000))
    h = float(rng.choice([1.0, 0.25, 0.7]))
    base = "cfg2" if dim == 2 else ("cfg4" if rng.random() < 0.3 and min(n) >= 8 else "cfg3")
    cfg = W.CONFIGS[base].scaled(N, n=n, order=order, dtype=dtype, h=h, seed=seed)
    _lockstep(cfg, 2)


def test_step_fields_host_entry_point():
    """pic_step_fields_host: particles on the device, E and rho on the host; two steps (ping-pong) against the oracle."""
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=70_001, n=(16, 16, 16)))
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    a = dict(x=to_dev(wl.x), v=to_dev(wl.v), w=to_dev([wl.w])[0])
    b = dict(x=[torch.empty_like(t) for t in a["x"]], v=[torch.empty_like(t) for t in a["v"]], w=torch.empty_like(a["w"]))
    perm = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    off = torch.full((gb.cells + 4,), -1, dtype=torch.int32, device="cuda")
    ws = torch.empty(B.pic_step_fields_host_bytes(gb, n), dtype=torch.uint8, device="cuda")
    rho = np.empty(gb.cells, cfg.np_dtype)
    x, v, w = wl.x, wl.v, wl.w
    for step in range(2):
        ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        B.pic_step_fields_host(gb, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], perm, off, rho, wl.E,
                               cfg.dt, cfg.qm, True, ws)
        assert B.pic_last_launch_count() > 0
        assert np.array_equal(perm.cpu().numpy(), ref["perm"])
        assert err_rho(rho, ref["rho"]) <= TOL_RHO[cfg.dtype]
        for c in range(cfg.dim):
            assert err_x(b["x"][c].cpu().numpy(), ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
            assert err_v(b["v"][c].cpu().numpy(), ref["v"][c]) <= TOL_XV[cfg.dtype]
        # lockstep: the next step starts from the oracle's state
        x, v, w = ref["x"], ref["v"], ref["w"]
        a = dict(x=to_dev(x), v=to_dev(v), w=to_dev([w])[0])
    with pytest.raises(B.PicError, match="workspace"):
        B.pic_step_fields_host(gb, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], perm, off, rho, wl.E,
                               cfg.dt, cfg.qm, True, ws[: 4096])


# ---------------------------------------------------------------------------------------------------------------
# PIC_SORT_CHAINED (row a8: the step kernel emits the next step's keys, histogram and mover list).  The chained
# sort must give, bit for bit, what the sort from the positions gives; the latter is compared with the oracle in
# lockstep above, the former also directly below.
CHAIN_CASES = [
    ("cfg2", dict(N=200_003, n=(64, 64))),
    ("cfg3", dict(N=150_001, n=(32, 32, 32))),
    ("cfg3", dict(N=3 * 2048 + 1, n=(8, 8, 8))),
    ("cfg4", dict(N=300_007, n=(32, 32, 32))),
    ("cfg5", dict(N=8 * 16 ** 3 + 5, n=(16, 16, 16))),
    ("cfg1", dict()),
]


def _same_state(a, b, n, cells, what):
    assert torch.equal(a.perm[:n], b.perm[:n]), "perm, " + what
    assert torch.equal(a.cell_offsets[: cells + 1], b.cell_offsets[: cells + 1]), "cell_offsets, " + what
    for c in range(len(a.cur["x"])):
        assert torch.equal(a.cur["x"][c], b.cur["x"][c]), "x[%d], %s" % (c, what)
        assert torch.equal(a.cur["v"][c], b.cur["v"][c]), "v[%d], %s" % (c, what)
    assert torch.equal(a.cur["w"], b.cur["w"]), "w, " + what


@pytest.mark.parametrize("name,kw", CHAIN_CASES)
def test_chained_steps_equal_unchained_bit_for_bit(name, kw):
    O, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    g = B.grid_of(cfg)
    a = B.Stepper(g, wl.x, wl.v, wl.w, wl.E)
    b = B.Stepper(g, wl.x, wl.v, wl.w, wl.E)
    # sorted steps, an unsorted one in between (which breaks the chain), sorted steps again
    plan = [True, True, True, False, True, True, True, True]
    for k, do_sort in enumerate(plan):
        a.step(cfg.dt, cfg.qm, do_sort, chained=True)
        b.step(cfg.dt, cfg.qm, do_sort, chained=False)
        torch.cuda.synchronize()
        if do_sort:
            _same_state(a, b, cfg.N, g.cells, "step %d" % k)
        ra, rb = a.rho.double(), b.rho.double()
        assert float((ra - rb).abs().max()) <= TOL_RHO[cfg.dtype] * float(rb.abs().max()), "rho, step %d" % k


@pytest.mark.parametrize("name,kw", [("cfg3", dict(N=150_001, n=(32, 32, 32))), ("cfg5", dict(N=8 * 16 ** 3 + 5, n=(16, 16, 16)))])
def test_chained_steps_against_oracle_lockstep_by_id(name, kw):
    """A free-running chained GPU run and the oracle, step by step: while no particle sits within rounding of a cell
    face the two orders are identical, and then perm and cell_offsets must agree bit for bit at every step."""
    O, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    go, g = O.grid_of(cfg), B.grid_of(cfg)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E)
    x, v, w = wl.x, wl.v, wl.w
    for k in range(6):
        # the oracle steps from the GPU's own state: the chain is not touched (nothing is written to the device)
        st.step(cfg.dt, cfg.qm, True, chained=True)
        r = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        torch.cuda.synchronize()
        assert np.array_equal(st.perm[: cfg.N].cpu().numpy(), r["perm"]), "perm, step %d" % k
        assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), r["cell_offsets"]), "cell_offsets, step %d" % k
        assert err_rho(st.rho.cpu().numpy(), r["rho"]) <= TOL_RHO[cfg.dtype]
        x = [a.cpu().numpy() for a in st.cur["x"]]
        v = [a.cpu().numpy() for a in st.cur["v"]]
        w = st.cur["w"].cpu().numpy()
        for c in range(cfg.dim):
            assert err_x(x[c], r["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
            assert err_v(v[c], r["v"][c]) <= TOL_XV[cfg.dtype]


def test_chain_flag_on_foreign_arrays_falls_back():
    """PIC_SORT_CHAINED on arrays the workspace's emission does not belong to (other addresses, another sort in
    between) must behave like PIC_SORT: the device-side check of the chain signature."""
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=60_001, n=(16, 16, 16)))
    wl = W.make_workload(cfg)
    go, g = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E)
    st.step(cfg.dt, cfg.qm, True)
    st.step(cfg.dt, cfg.qm, True)
    torch.cuda.synchronize()
    # (1) other arrays, same workspace, chained flag
    wl2 = W.make_workload(cfg.scaled(n, seed=cfg.seed + 7))
    ref = O.step(go, wl2.x, wl2.v, wl2.w, wl2.E, cfg.dt, cfg.qm)
    x, v, w = to_dev(wl2.x), to_dev(wl2.v), to_dev([wl2.w])[0]
    xo, vo, wo = [torch.empty_like(a) for a in x], [torch.empty_like(a) for a in v], torch.empty_like(w)
    E = to_dev(wl2.E)
    B.pic_step(g, x, v, w, xo, vo, wo, st.perm, st.cell_offsets, st.rho, E, cfg.dt, cfg.qm, B.PIC_SORT_CHAINED, st.ws)
    torch.cuda.synchronize()
    assert np.array_equal(st.perm[:n].cpu().numpy(), ref["perm"])
    assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), ref["cell_offsets"])
    # (2) that call has left an emission for (xo, vo, wo); a pic_sort on the same workspace voids it
    perm2 = torch.empty_like(st.perm)
    off2 = torch.zeros_like(st.cell_offsets)
    B.pic_sort(g, x, v, w, [torch.empty_like(a) for a in x], [torch.empty_like(a) for a in v], torch.empty_like(w), perm2, off2, st.ws)
    ref2 = O.step(go, to_host(xo), to_host(vo), wo.cpu().numpy(), wl2.E, cfg.dt, cfg.qm)   # from the GPU's own state
    x2, v2, w2 = [torch.empty_like(a) for a in x], [torch.empty_like(a) for a in v], torch.empty_like(w)
    B.pic_step(g, xo, vo, wo, x2, v2, w2, st.perm, st.cell_offsets, st.rho, E, cfg.dt, cfg.qm, B.PIC_SORT_CHAINED, st.ws)
    torch.cuda.synchronize()
    assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), ref2["cell_offsets"])
    assert np.array_equal(st.perm[:n].cpu().numpy(), ref2["perm"])


def test_pic_step_do_sort_values_and_checks_before_any_copy():
    """any non-zero do_sort sorts (only PIC_SORT_CHAINED means more); and a bad argument is reported before
    anything is enqueued -- with do_sort = 0 and distinct out arrays that includes the device-to-device copies."""
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=30_001, n=(16, 16, 16)))
    wl = W.make_workload(cfg)
    go, g = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    ref = O.step(go, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm)
    x, v, w, E = to_dev(wl.x), to_dev(wl.v), to_dev([wl.w])[0], to_dev(wl.E)
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    rho = torch.empty(g.cells, dtype=g.torch_dtype, device="cuda")
    for do_sort in (2, 7, -1, True):
        xo, vo, wo = [torch.empty_like(a) for a in x], [torch.empty_like(a) for a in v], torch.empty_like(w)
        perm = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        off = torch.zeros(g.cells + 4, dtype=torch.int32, device="cuda")
        B.pic_step(g, x, v, w, xo, vo, wo, perm, off, rho, E, cfg.dt, cfg.qm, do_sort, ws)
        torch.cuda.synchronize()
        assert np.array_equal(perm.cpu().numpy(), ref["perm"]), do_sort
        assert np.array_equal(off[: g.cells + 1].cpu().numpy(), ref["cell_offsets"]), do_sort
        assert err_x(xo[0].cpu().numpy(), ref["x"][0], cfg.L[0]) <= TOL_XV[cfg.dtype]
    # do_sort = 0 with a misaligned cell_offsets: refused, and `out` has not been written
    xo, vo, wo = [torch.full_like(a, -1.0) for a in x], [torch.full_like(a, -1.0) for a in v], torch.full_like(w, -1.0)
    off = torch.zeros(g.cells + 8, dtype=torch.int32, device="cuda")
    with pytest.raises(B.PicError, match="invalid argument"):
        B.pic_step(g, x, v, w, xo, vo, wo, None, off[1:], rho, E, cfg.dt, cfg.qm, 0, ws)
    torch.cuda.synchronize()
    assert all(torch.all(a == -1.0).item() for a in xo + vo + [wo])


@pytest.mark.parametrize("foreign", ["field_solve", "deposit_other_n", "deposit_nodes_other_n", "replicated_other_n"])
def test_chain_ends_when_the_workspace_is_used_for_something_else(foreign):
    """Between two chained steps another call is given the same workspace and writes over the emission (the field
    solve's arrays start at the front; a deposit carved for another particle count puts its double grid in the middle
    of the staged keys).  Each of these calls voids the chain signature in the first bytes of the workspace, so the
    next PIC_SORT_CHAINED step must sort from the positions and still give the oracle's perm and offsets."""
    O, B = _mods()
    cfg = _cfg("cfg3", dict(N=40_000, n=(32, 32, 32)))          # field arrays (32 C bytes) cover keys, idx and pkey of N
    wl = W.make_workload(cfg)
    go, g = O.grid_of(cfg), B.grid_of(cfg)
    n = cfg.N
    big = torch.empty(max(B.pic_workspace_bytes(g, n), B.pic_field_solve_bytes(g), B.pic_deposit_replicated_bytes(g, 1000)) + 4096,
                      dtype=torch.uint8, device="cuda")
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E)
    st.ws = big
    st.step(cfg.dt, cfg.qm, True)
    st.step(cfg.dt, cfg.qm, True)                              # chained; leaves an emission for the third step
    torch.cuda.synchronize()
    small = W.make_workload(cfg.scaled(1000, seed=3))
    xs, ws_ = to_dev(small.x), to_dev([small.w])[0]
    rho = torch.empty(g.cells, dtype=torch.float32, device="cuda")
    if foreign == "field_solve":
        rho.copy_(st.rho)
        B.pic_field_solve(g, rho, [torch.empty_like(rho) for _ in range(3)], None, big)
    elif foreign == "deposit_other_n":
        B.pic_deposit(g, xs, ws_, rho, B.PIC_ORDER_UNSORTED, None, big)
    else:
        sx, _, sw, _, off = O.sort(go, small.x, small.v, small.w)
        offd = torch.from_numpy(np.concatenate([off, np.zeros(3, np.int32)]).astype(np.int32)).cuda()
        dep = B.pic_deposit_nodes if foreign == "deposit_nodes_other_n" else B.pic_deposit_replicated
        dep(g, to_dev(sx), to_dev([sw])[0], rho, offd, big)
    torch.cuda.synchronize()
    ref = O.step(go, to_host(st.cur["x"]), to_host(st.cur["v"]), st.cur["w"].cpu().numpy(), wl.E, cfg.dt, cfg.qm)
    st.step(cfg.dt, cfg.qm, True)                              # asks for PIC_SORT_CHAINED
    torch.cuda.synchronize()
    assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), ref["cell_offsets"])
    assert np.array_equal(st.perm[:n].cpu().numpy(), ref["perm"])
    assert err_rho(st.rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[cfg.dtype]
    for c in range(cfg.dim):
        assert err_x(st.cur["x"][c].cpu().numpy(), ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
    # and the chain picks up again afterwards: one more chained step, still the oracle's order
    ref2 = O.step(go, to_host(st.cur["x"]), to_host(st.cur["v"]), st.cur["w"].cpu().numpy(), wl.E, cfg.dt, cfg.qm)
    st.step(cfg.dt, cfg.qm, True)
    torch.cuda.synchronize()
    assert np.array_equal(st.perm[:n].cpu().numpy(), ref2["perm"])


@pytest.mark.parametrize("name,kw,mode", [("cfg1", dict(), "plain"), ("cfg3", dict(N=200_000, n=(32, 32, 32)), "plain"),
                                          ("cfg5", dict(N=8 * 16 ** 3, n=(16, 16, 16)), "closed"),
                                          ("cfg2", dict(N=100_000, n=(32, 32)), "bucket")])
def test_graph_replay_equals_plain_stepping(name, kw, mode):
    """Stepper(graph=True) replays the sort steps from CUDA graphs (launch-bound problems).  Every choice inside a step is
    made on the device, so the replayed steps must be the plain ones bit for bit -- perm, offsets, x, v, w -- over 7 steps
    (first sort, pre-ordered sorts, both ping-pong directions)."""
    _, B = _mods()
    cfg = _cfg(name, kw)
    wl = W.make_workload(cfg)
    g = B.grid_of(cfg)
    extra = dict(closed_loop=True) if mode == "closed" else (dict(bucket=(4, 2)) if mode == "bucket" else {})
    a = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, **extra)
    b = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, graph=True, **extra)
    for k in range(7):
        a.step(cfg.dt, cfg.qm, True)
        b.step(cfg.dt, cfg.qm, True)
        torch.cuda.synchronize()
        if mode == "closed":
            # the field comes from rho, whose reductions have no fixed order: two runs agree to rounding, not bit for bit
            for c in range(cfg.dim):
                assert err_x(b.cur["x"][c].cpu().numpy(), a.cur["x"][c].cpu().numpy(), cfg.L[c]) <= 1e-12
            continue
        assert torch.equal(a.perm[: cfg.N], b.perm[: cfg.N]), "perm at step %d" % k
        assert torch.equal(a.cell_offsets, b.cell_offsets)
        for c in range(cfg.dim):
            assert torch.equal(a.cur["x"][c], b.cur["x"][c]) and torch.equal(a.cur["v"][c], b.cur["v"][c])
        assert torch.equal(a.cur["w"], b.cur["w"])
        assert err_rho(b.rho.cpu().numpy(), a.rho.cpu().numpy()) <= 1e-6
    assert b.last_launches > 0 and len(b._graphs) == 2
