"""GPU parity of the multi-cell bucket sort and step
against the oracle's pic_ref_sort_buckets (+ deposit and push on the bucket-ordered arrays), through the C ABI.
perm and bucket_offsets bit-exact for every bucket shape; rho, x, v within north_star's tolerances."""
import numpy as np
import pytest

import pic_workloads as W
from parity import TOL_RHO, TOL_XV, err_rho, err_v, err_x, to_dev

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _mods():
    import oracle as O
    import paper_1603_02886_b200 as B
    return O, B


def _cfg(name, N, **kw):
    return W.CONFIGS[name].scaled(N, **kw)


CASES = [
    # (config, N, grid, bucket)
    ("cfg2", 200_003, (64, 64), (1, 1)),            # unit buckets: the cell sort
    ("cfg2", 200_003, (64, 64), (2, 2)),
    ("cfg2", 200_003, (64, 64), (8, 4)),
    ("cfg2", 150_001, (48, 40), (5, 7)),            # bucket sizes that do not divide the grid: ragged last buckets
    ("cfg2", 100_000, (64, 64), (64, 64)),          # ONE bucket: the identity permutation
    ("cfg2", 100_000, (64, 64), (64, 1)),           # buckets = grid rows
    ("cfg3", 150_001, (32, 32, 32), (2, 2, 2)),
    ("cfg3", 150_001, (32, 32, 32), (4, 4, 4)),
    ("cfg3", 150_001, (32, 16, 8), (8, 2, 3)),
    ("cfg4", 300_007, (32, 32, 32), (4, 4, 4)),     # clustered: a few buckets hold most particles
    ("cfg5", 8 * 16 ** 3 + 5, (16, 16, 16), (4, 2, 1)),
    ("cfg1", 100_000, (64, 64), (32, 16)),          # the paper's optimum in buckets per dimension (2 x 4 buckets here)
]


def _gpu_sort_buckets(B, g, bucket, wl, hint=None):
    n = wl.cfg.N
    x, v = to_dev(wl.x), to_dev(wl.v)
    w = to_dev([wl.w])[0]
    xo = [torch.empty_like(a) for a in x]
    vo = [torch.empty_like(a) for a in v]
    wo = torch.empty_like(w)
    nb = B.pic_bucket_count(g, bucket)
    perm = torch.full((max(n, 4),), -1, dtype=torch.int32, device="cuda")
    off = torch.full((nb + 4,), -1, dtype=torch.int32, device="cuda")
    if hint is not None:
        off[: nb + 1] = torch.from_numpy(hint.astype(np.int32)).cuda()
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    B.pic_sort_buckets(g, bucket, x, v, w, xo, vo, wo, perm, off, ws)
    torch.cuda.synchronize()
    return xo, vo, wo, perm[:n].cpu().numpy(), off[: nb + 1].cpu().numpy()


@pytest.mark.parametrize("name,N,n,bucket", CASES)
def test_sort_buckets_bit_exact(name, N, n, bucket):
    O, B = _mods()
    cfg = _cfg(name, N, n=n)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    assert B.pic_bucket_count(gb, bucket) == O.bucket_count(go, bucket)
    ro = O.sort_buckets(go, wl.x, wl.v, wl.w, bucket)
    xo, vo, wo, perm, off = _gpu_sort_buckets(B, gb, bucket, wl)
    assert np.array_equal(perm, ro[3])
    assert np.array_equal(off, ro[4])
    for c in range(cfg.dim):
        assert np.array_equal(xo[c].cpu().numpy(), ro[0][c])
        assert np.array_equal(vo[c].cpu().numpy(), ro[1][c])
    assert np.array_equal(wo.cpu().numpy(), ro[2])


@pytest.mark.parametrize("bucket", [(2, 2, 2), (4, 8, 1)])
def test_sort_buckets_with_hints(bucket):
    """bucket_offsets on entry is an order hint: the previous offsets (pre-ordered particles), garbage, zeros --
    the permutation never depends on it."""
    O, B = _mods()
    cfg = _cfg("cfg3", 120_001, n=(32, 32, 32))
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    xs, vs, wsrt, _, off0 = O.sort_buckets(go, wl.x, wl.v, wl.w, bucket)
    x1, v1 = O.push(go, xs, vs, wl.E, cfg.dt, cfg.qm)               # pre-ordered: one push after a bucket sort
    wl1 = W.Workload(cfg, x1, v1, wsrt, wl.E, wl.modes)
    ro = O.sort_buckets(go, x1, v1, wsrt, bucket)
    rng = np.random.default_rng(5)
    nb = off0.size - 1
    hints = [off0, np.zeros(nb + 1, np.int64), rng.integers(-5, cfg.N + 5, nb + 1), np.sort(rng.integers(0, cfg.N + 1, nb + 1)),
             np.full(nb + 1, cfg.N)]
    for h in hints:
        _, _, _, perm, off = _gpu_sort_buckets(B, gb, bucket, wl1, hint=np.asarray(h))
        assert np.array_equal(perm, ro[3])
        assert np.array_equal(off, ro[4])


@pytest.mark.parametrize("N", [0, 1, 33, 4097])
def test_sort_buckets_edge_sizes(N):
    O, B = _mods()
    cfg = _cfg("cfg2", N, n=(16, 16))
    wl = W.make_workload(cfg)
    ro = O.sort_buckets(O.grid_of(cfg), wl.x, wl.v, wl.w, (4, 4))
    _, _, _, perm, off = _gpu_sort_buckets(B, B.grid_of(cfg), (4, 4), wl)
    assert np.array_equal(perm, ro[3])
    assert np.array_equal(off, ro[4])


def test_bucket_arguments_are_validated():
    _, B = _mods()
    g = B.Grid(2, (16, 16), (1.0, 1.0), 1, "f64")
    for bad in ((0, 1), (17, 1), (1, -3)):
        with pytest.raises(B.PicError, match="invalid argument"):
            B.pic_bucket_count(g, bad)
    assert B.pic_bucket_count(g, (16, 16)) == 1
    assert B.pic_bucket_count(g, (5, 3)) == 4 * 6


STEP_CASES = [
    ("cfg2", 200_003, (64, 64), (1, 1)),
    ("cfg2", 200_003, (64, 64), (4, 4)),
    ("cfg3", 150_001, (32, 32, 32), (2, 2, 2)),
    ("cfg3", 150_001, (32, 32, 32), (4, 4, 4)),
    ("cfg4", 200_007, (32, 32, 32), (2, 2, 2)),
    ("cfg5", 8 * 16 ** 3 + 5, (16, 16, 16), (4, 4, 2)),
    ("cfg1", 100_000, (64, 64), (8, 8)),
    ("cfg3", 60_000, (16, 16, 16), (16, 16, 16)),   # one bucket: the step runs on the source order (137 KB tile: still shared memory)
    ("cfg3", 90_000, (32, 32, 32), (32, 32, 16)),   # tile too large for shared memory: the run kernel with strays takes over
    ("cfg2", 120_000, (96, 80), (96, 80)),          # the same in 2-D, fp64
    ("cfg5", 50_000, (12, 10, 14), (5, 3, 4)),      # ragged buckets, quadratic, fp64
    ("cfg1", 100_000, (64, 64), (64, 32)),          # linear splines, two buckets (R blocks per bucket)
]


@pytest.mark.parametrize("name,N,n,bucket", STEP_CASES)
def test_step_buckets_lockstep(name, N, n, bucket):
    """Three steps of pic_step_buckets, each fed the oracle's state: perm / bucket_offsets bit-exact, rho and the
    advanced particles (in bucket order) within tolerance.  Buckets whose grid tile fits in shared memory go through the
    tile kernel (pic_tile.cuh), the others through the run kernel; the first step takes the reorder-first arm of both."""
    O, B = _mods()
    cfg = _cfg(name, N, n=n)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    nb = B.pic_bucket_count(gb, bucket)
    E = to_dev(wl.E)
    ws = torch.empty(B.pic_workspace_bytes(gb, N), dtype=torch.uint8, device="cuda")
    perm = torch.full((max(N, 4),), -1, dtype=torch.int32, device="cuda")
    off = torch.zeros(nb + 4, dtype=torch.int32, device="cuda")
    rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
    x, v, w = wl.x, wl.v, wl.w
    for k in range(3):
        xs, vs, wsrt, rperm, roff = O.sort_buckets(go, x, v, w, bucket)
        rrho = O.deposit(go, xs, wsrt)
        rx, rv = O.push(go, xs, vs, wl.E, cfg.dt, cfg.qm)
        xd, vd, wd = to_dev(x), to_dev(v), to_dev([w])[0]
        xo = [torch.empty_like(a) for a in xd]
        vo = [torch.empty_like(a) for a in vd]
        wo = torch.empty_like(wd)
        B.pic_step_buckets(gb, bucket, xd, vd, wd, xo, vo, wo, perm, off, rho, E, cfg.dt, cfg.qm, ws)
        torch.cuda.synchronize()
        assert np.array_equal(perm[:N].cpu().numpy(), rperm), "perm at step %d" % k
        assert np.array_equal(off[: nb + 1].cpu().numpy(), roff), "offsets at step %d" % k
        assert err_rho(rho.cpu().numpy(), rrho) <= TOL_RHO[cfg.dtype], "rho at step %d" % k
        for c in range(cfg.dim):
            assert err_x(xo[c].cpu().numpy(), rx[c], cfg.L[c]) <= TOL_XV[cfg.dtype], "x at step %d" % k
            assert err_v(vo[c].cpu().numpy(), rv[c]) <= TOL_XV[cfg.dtype], "v at step %d" % k
        assert np.array_equal(wo.cpu().numpy(), wsrt)
        x, v, w = rx, rv, wsrt


def test_unit_buckets_equal_the_cell_step():
    """bucket = (1,1,1) is pic_step(PIC_SORT): same perm, offsets, and bit-identical particles."""
    _, B = _mods()
    cfg = _cfg("cfg3", 100_003, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    gb = B.grid_of(cfg)
    N = cfg.N
    E = to_dev(wl.E)
    outs = []
    for mode in ("cells", "buckets"):
        xd, vd, wd = to_dev(wl.x), to_dev(wl.v), to_dev([wl.w])[0]
        xo = [torch.empty_like(a) for a in xd]
        vo = [torch.empty_like(a) for a in vd]
        wo = torch.empty_like(wd)
        ws = torch.empty(B.pic_workspace_bytes(gb, N), dtype=torch.uint8, device="cuda")
        perm = torch.full((N,), -1, dtype=torch.int32, device="cuda")
        off = torch.zeros(gb.cells + 4, dtype=torch.int32, device="cuda")
        rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
        if mode == "cells":
            B.pic_step(gb, xd, vd, wd, xo, vo, wo, perm, off, rho, E, cfg.dt, cfg.qm, True, ws)
        else:
            B.pic_step_buckets(gb, (1, 1, 1), xd, vd, wd, xo, vo, wo, perm, off, rho, E, cfg.dt, cfg.qm, ws)
        torch.cuda.synchronize()
        outs.append((perm.cpu().numpy(), off[: gb.cells + 1].cpu().numpy(), [a.cpu().numpy() for a in xo + vo]))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    for a, b in zip(outs[0][2], outs[1][2]):
        assert np.array_equal(a, b)


# ---- pic_sort_buckets_inplace: Alg. 2, only misplaced particles move ------------------------
INPLACE_CASES = [
    ("cfg2", 200_003, (64, 64), (8, 8), True), ("cfg2", 200_003, (64, 64), (1, 1), True), ("cfg2", 150_001, (48, 40), (5, 7), True),
    ("cfg3", 150_001, (32, 32, 32), (4, 4, 4), True), ("cfg3", 150_001, (32, 32, 32), (1, 1, 1), True),
    ("cfg3", 150_001, (32, 32, 32), (8, 8, 8), False),        # random order: nearly everything is misplaced
    ("cfg4", 300_007, (32, 32, 32), (4, 4, 4), True), ("cfg5", 8 * 16 ** 3 + 5, (16, 16, 16), (4, 2, 1), True),
    ("cfg1", 100_000, (64, 64), (32, 16), True), ("cfg3", 60_000, (16, 16, 16), (16, 16, 16), False),   # one bucket: nothing moves
]


@pytest.mark.parametrize("name,N,n,bucket,presort", INPLACE_CASES)
def test_sort_buckets_inplace_bit_exact(name, N, n, bucket, presort):
    """The whole particle arrays, the offsets and the number of moved particles equal the oracle's Alg. 2 bit for bit
    (slots in ascending position make the result unique, R24)."""
    O, B = _mods()
    cfg = _cfg(name, N, n=n)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    x, v, w = wl.x, wl.v, wl.w
    if presort:
        x, v, w, _, _ = O.sort_buckets(go, x, v, w, bucket)
        x, v = O.push(go, x, v, wl.E, cfg.dt, cfg.qm)
    rx, rv, rw, roff, rmoved = O.sort_buckets_inplace(go, x, v, w, bucket)
    xd, vd, wd = to_dev(x), to_dev(v), to_dev([w])[0]
    nb = B.pic_bucket_count(gb, bucket)
    off = torch.full((nb + 4,), -7, dtype=torch.int32, device="cuda")
    moved = torch.full((4,), -1, dtype=torch.int32, device="cuda")
    ws = torch.full((B.pic_sort_buckets_inplace_bytes(gb, N),), 0x5C, dtype=torch.uint8, device="cuda")
    B.pic_sort_buckets_inplace(gb, bucket, xd, vd, wd, off, moved, ws)
    torch.cuda.synchronize()
    assert int(moved[0].item()) == rmoved
    assert np.array_equal(off[: nb + 1].cpu().numpy(), roff)
    for c in range(cfg.dim):
        assert np.array_equal(xd[c].cpu().numpy(), rx[c]) and np.array_equal(vd[c].cpu().numpy(), rv[c])
    assert np.array_equal(wd.cpu().numpy(), rw)
    if nb == 1:
        assert rmoved == 0


@pytest.mark.parametrize("N", [0, 1, 33, 4097])
def test_sort_buckets_inplace_edge_sizes(N):
    O, B = _mods()
    cfg = _cfg("cfg2", N, n=(16, 16))
    wl = W.make_workload(cfg)
    rx, rv, rw, roff, rmoved = O.sort_buckets_inplace(O.grid_of(cfg), wl.x, wl.v, wl.w, (4, 4))
    gb = B.grid_of(cfg)
    xd, vd, wd = to_dev(wl.x), to_dev(wl.v), to_dev([wl.w])[0]
    off = torch.zeros(16 + 4, dtype=torch.int32, device="cuda")
    moved = torch.zeros(4, dtype=torch.int32, device="cuda")
    ws = torch.empty(B.pic_sort_buckets_inplace_bytes(gb, N), dtype=torch.uint8, device="cuda")
    B.pic_sort_buckets_inplace(gb, (4, 4), xd, vd, wd, off, moved, ws)
    torch.cuda.synchronize()
    assert int(moved[0].item()) == rmoved and np.array_equal(off[:17].cpu().numpy(), roff)
    if N:
        assert np.array_equal(xd[0].cpu().numpy(), rx[0]) and np.array_equal(wd.cpu().numpy(), rw)
