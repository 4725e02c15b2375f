"""Pins of the oracle's bucket sort (NEXT-2: buckets of several cells):
a hand-written numpy key with numpy's stable argsort, the special cases that reduce to the
cell sort and to the identity, and the invariants of a stable counting sort."""
import numpy as np
import pytest

import oracle as O
import pic_workloads as W


def cfg_of(dim, dtype, N, n, seed=0):
    return W.Config("t", dim, tuple(n), N, dtype, 1, "uniform", 3, 1, seed=seed)


def numpy_bucket_key(cfg, x, bucket):
    """b_c = floor(cell_c / bucket_c), key = b_x + nb_x (b_y + nb_y b_z): bins x fastest."""
    key = np.zeros(cfg.N, np.int64)
    stride = 1
    for c in range(cfg.dim):
        cell = np.clip(np.floor(x[c] / cfg.np_dtype(cfg.h)).astype(np.int64), 0, cfg.n[c] - 1)
        key += stride * (cell // bucket[c])
        stride *= -(-cfg.n[c] // bucket[c])
    return key, stride


CASES = [
    (2, "f64", (16, 16), (4, 2)),
    (2, "f32", (32, 16), (16, 16)),      # the paper's 512x256 grid in 32x16 buckets, scaled down
    (3, "f32", (8, 8, 8), (2, 2, 2)),
    (3, "f64", (8, 8, 8), (4, 4, 4)),
    (3, "f64", (10, 6, 7), (3, 4, 2)),   # bucket sizes that do not divide the grid: ragged last buckets
    (3, "f32", (8, 8, 8), (8, 1, 1)),    # whole x rows
]


@pytest.mark.parametrize("dim,dtype,n,bucket", CASES)
def test_bucket_sort_equals_numpy_stable_argsort(dim, dtype, n, bucket):
    cfg = cfg_of(dim, dtype, 20011, n)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    key, B = numpy_bucket_key(cfg, wl.x, bucket)
    assert O.bucket_count(g, bucket) == B
    assert np.array_equal(O.bucket_keys(g, wl.x, bucket), key.astype(np.int32))
    xo, vo, wo, perm, off = O.sort_buckets(g, wl.x, wl.v, wl.w, bucket)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.int32))
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(key, minlength=B))]).astype(np.int32))
    assert np.array_equal(np.sort(perm), np.arange(cfg.N, dtype=np.int32))
    ks = key[perm]
    assert np.all(np.diff(ks) >= 0)
    assert np.all(np.diff(perm.astype(np.int64))[np.diff(ks) == 0] > 0)      # ties keep the source order
    for c in range(dim):
        assert np.array_equal(xo[c], wl.x[c][perm]) and np.array_equal(vo[c], wl.v[c][perm])
    assert np.array_equal(wo, wl.w[perm])


@pytest.mark.parametrize("dim,n", [(2, (16, 16)), (3, (8, 8, 8))])
def test_unit_buckets_are_the_cell_sort_and_one_bucket_is_the_identity(dim, n):
    cfg = cfg_of(dim, "f64", 7001, n, seed=3)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    ones = (1,) * dim
    a = O.sort(g, wl.x, wl.v, wl.w)
    b = O.sort_buckets(g, wl.x, wl.v, wl.w, ones)
    assert np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])
    assert np.array_equal(O.keys(g, wl.x), O.bucket_keys(g, wl.x, ones))
    # one bucket holding the whole grid: nothing moves
    _, _, _, perm, off = O.sort_buckets(g, wl.x, wl.v, wl.w, n)
    assert np.array_equal(perm, np.arange(cfg.N, dtype=np.int32))
    assert np.array_equal(off, np.array([0, cfg.N], np.int32))


def test_bucket_order_refines_to_cell_order():
    """Sorting by cell inside every bucket of a bucket-sorted array gives, bucket by bucket, the same particle
    sets as the cell sort restricted to the cells of that bucket (a bucket is a union of cells)."""
    cfg = cfg_of(3, "f32", 30011, (8, 8, 8), seed=5)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    bucket = (4, 2, 2)
    _, _, _, perm_b, off_b = O.sort_buckets(g, wl.x, wl.v, wl.w, bucket)
    cell = O.keys(g, wl.x)
    bkey = O.bucket_keys(g, wl.x, bucket)
    for k in range(off_b.size - 1):
        ids = perm_b[off_b[k]: off_b[k + 1]]
        assert np.all(bkey[ids] == k)
        cx, cy, cz = cell[ids] % 8, (cell[ids] // 8) % 8, cell[ids] // 64
        assert np.all(cx // 4 + 2 * (cy // 2 + 4 * (cz // 2)) == k)
    assert off_b[-1] == cfg.N


def test_bad_bucket_sizes_are_rejected():
    cfg = cfg_of(2, "f64", 10, (8, 8))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    for bad in [(0, 1), (9, 1), (1, -2)]:
        with pytest.raises(Exception):
            O.sort_buckets(g, wl.x, wl.v, wl.w, bad)


# ---- Alg. 2: sort for pre-ordered particles, in place ---------------------------------------
def _alg2_transcription(key, nb, rng):
    """The paper's listing transcribed line by line in Python, buffer slots handed out in RANDOM order (its atomic
    counters fix none): returns the array of particle ids after the sort, and the holes."""
    n = key.size
    sizes = np.bincount(key, minlength=nb)
    off = np.concatenate([[0], np.cumsum(sizes)])
    bucket_num = np.repeat(np.arange(nb), sizes)                       # l.6-10
    ids = np.arange(n)
    mis = np.nonzero(bucket_num != key)[0]                             # l.13-17
    out = ids.copy()
    for b in range(nb):                                                # l.31-35, per bucket
        holes = mis[bucket_num[mis] == b]
        incoming = mis[key[mis] == b]
        assert holes.size == incoming.size
        out[rng.permutation(holes)] = ids[incoming]
    return out, off, mis


@pytest.mark.parametrize("name,N,n,bucket,presort", [
    ("cfg2", 30_000, (32, 32), (4, 4), False), ("cfg2", 30_000, (32, 32), (4, 4), True), ("cfg2", 20_000, (30, 28), (7, 5), True),
    ("cfg3", 40_000, (16, 16, 16), (1, 1, 1), True), ("cfg3", 40_000, (16, 16, 16), (4, 4, 4), True),
    ("cfg4", 40_000, (16, 16, 16), (2, 4, 8), True), ("cfg5", 20_000, (12, 10, 14), (12, 10, 14), False)])
def test_inplace_sort_is_alg2(name, N, n, bucket, presort):
    cfg = W.CONFIGS[name].scaled(N, n=n)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    x, v, w = wl.x, wl.v, wl.w
    if presort:                                   # pre-ordered: sorted once, then pushed (the paper's situation, ~20 % misplaced)
        x, v, w, _, _ = O.sort_buckets(g, x, v, w, bucket)
        x, v = O.push(g, x, v, wl.E, cfg.dt, cfg.qm)
    ident = np.arange(N, dtype=cfg.np_dtype) if cfg.dtype == "f64" else np.arange(N, dtype=np.float32)
    assert np.array_equal(ident.astype(np.int64), np.arange(N))       # ids survive as the weight attribute
    xo, vo, wo, off, moved = O.sort_buckets_inplace(g, x, v, ident, bucket)
    key = O.bucket_keys(g, x, bucket).astype(np.int64)
    nb = O.bucket_count(g, bucket)
    got_ids = wo.astype(np.int64)
    # (1) a sort: keys of the result non-decreasing; offsets = prefix sum of the histogram (what the stable sort gives)
    assert np.all(np.diff(O.bucket_keys(g, xo, bucket)) >= 0)
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(np.bincount(key, minlength=nb))]))
    assert np.array_equal(off, O.sort_buckets(g, x, v, w, bucket)[4])
    # (2) attributes travel together, bit for bit
    for c in range(cfg.dim):
        assert np.array_equal(xo[c], x[c][got_ids]) and np.array_equal(vo[c], v[c][got_ids])
    # (3) only misplaced particles moved, and all of them: the others sit where they sat
    ref_ids, roff, mis = _alg2_transcription(key, nb, np.random.default_rng(1))
    assert moved == mis.size == int(np.sum(got_ids != np.arange(N)) + np.sum((got_ids == np.arange(N))[mis]))
    stay = np.ones(N, bool); stay[mis] = False
    assert np.array_equal(got_ids[stay], np.arange(N)[stay])
    # (4) same buckets as the paper's listing with arbitrary slot order: equal multisets of ids per bucket
    for b in range(nb):
        assert np.array_equal(np.sort(got_ids[off[b]:off[b + 1]]), np.sort(ref_ids[roff[b]:roff[b + 1]]))
    # (5) the slot rule of R24: holes in ascending position take the misplaced particles in stable key order
    order = mis[np.argsort(key[mis], kind="stable")]
    assert np.array_equal(got_ids[mis], order)
    if presort and int(np.prod(bucket)) >= 32:
        assert 0.02 * N < moved < 0.6 * N         # large buckets: the particles that crossed a bucket face, plus boundary drift
    if presort and int(np.prod(bucket)) == 1:
        # one cell per bucket: "misplaced" is judged against the NEW offsets, and the boundary of a cell shifts by the sum of
        # the count changes of all cells below it -- most particles lie outside their own cell's region although only
        # about a fifth of them changed cell (why the hot path does not sort this way)
        changed = int(np.sum(key != O.bucket_keys(g, O.sort_buckets(g, wl.x, wl.v, wl.w, bucket)[0], bucket)))
        assert changed < 0.3 * N and moved > 0.5 * N


def test_inplace_sort_of_sorted_particles_moves_nothing():
    cfg = W.CONFIGS["cfg3"].scaled(20_000, n=(8, 8, 8))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    xs, vs, ws_, _, off0 = O.sort_buckets(g, wl.x, wl.v, wl.w, (2, 2, 2))
    xo, vo, wo, off, moved = O.sort_buckets_inplace(g, xs, vs, ws_, (2, 2, 2))
    assert moved == 0 and np.array_equal(off, off0)
    for c in range(3):
        assert np.array_equal(xo[c], xs[c]) and np.array_equal(vo[c], vs[c])
