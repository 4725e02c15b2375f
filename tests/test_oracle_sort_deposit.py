"""Pins of the oracle's sort (O2) and deposit (O3): library special cases, invariants,
closed forms and the all-pairs brute force (the paper's threads-on-grid definition,
PAPER.md:447-469)."""
import math

import numpy as np
import pytest

import oracle as O
import pic_workloads as W


def small_cfg(dim, p, dtype, N, n=8, seed=0, **kw):
    base = W.CONFIGS["cfg1"]
    return W.Config("t", dim, tuple([n] * dim), N, dtype, p, "uniform", 3, 1, seed=seed, **kw)


# --------------------------------------------------------------------------- sort
@pytest.mark.parametrize("dim,dtype", [(2, "f64"), (3, "f32"), (3, "f64"), (2, "f32")])
def test_sort_equals_numpy_stable_argsort(dim, dtype):
    cfg = small_cfg(dim, 1, dtype, 20011, n=16 if dim == 2 else 8)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    xo, vo, wo, perm, off = O.sort(g, wl.x, wl.v, wl.w)
    # key definition by hand: x fastest, floor in storage precision, clamped
    key = np.zeros(cfg.N, np.int64)
    stride = 1
    for c in range(dim):
        cell = np.clip(np.floor(wl.x[c] / cfg.np_dtype(cfg.h)).astype(np.int64), 0, cfg.n[c] - 1)
        key += stride * cell
        stride *= cfg.n[c]
    assert np.array_equal(O.keys(g, wl.x), key.astype(np.int32))
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.int32))
    counts = np.bincount(key, minlength=cfg.cells)
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(counts)]).astype(np.int32))
    # bijection, grouped, ties by ascending source index
    assert np.array_equal(np.sort(perm), np.arange(cfg.N, dtype=np.int32))
    ks = key[perm]
    assert np.all(np.diff(ks) >= 0)
    same = np.diff(ks) == 0
    assert np.all(np.diff(perm.astype(np.int64))[same] > 0)
    # attributes moved bit for bit
    for c in range(dim):
        assert np.array_equal(xo[c], wl.x[c][perm]) and np.array_equal(vo[c], wl.v[c][perm])
    assert np.array_equal(wo, wl.w[perm])


def test_sort_of_sorted_input_is_identity_and_handles_empty():
    cfg = small_cfg(3, 2, "f64", 5000)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    xo, vo, wo, perm, off = O.sort(g, wl.x, wl.v, wl.w)
    xo2, vo2, wo2, perm2, off2 = O.sort(g, xo, vo, wo)
    assert np.array_equal(perm2, np.arange(cfg.N, dtype=np.int32))
    assert np.array_equal(off2, off)
    e = [np.empty(0, np.float64)] * 3
    _, _, _, p0, off0 = O.sort(g, e, e, np.empty(0, np.float64))
    assert p0.size == 0 and np.all(off0 == 0) and off0.size == g.cells + 1


def test_sort_all_particles_in_one_cell():
    g = O.Grid(2, (8, 8), (1.0, 1.0), 1, "f64")
    N = 777
    rng = np.random.default_rng(1)
    x = [3.0 + rng.random(N), 5.0 + rng.random(N)]
    v = [rng.random(N), rng.random(N)]
    w = rng.random(N)
    _, _, _, perm, off = O.sort(g, x, v, w)
    assert np.array_equal(perm, np.arange(N, dtype=np.int32))
    k = 3 + 8 * 5
    assert np.all(off[: k + 1] == 0) and np.all(off[k + 1:] == N)


# ------------------------------------------------------------------------ deposit
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("p", [1, 2, 3])
@pytest.mark.parametrize("dim", [2, 3])
def test_deposit_equals_allpairs_bruteforce(dim, p, dtype):
    n = 6 if dim == 3 else 8
    cfg = small_cfg(dim, p, dtype, 90, n=n, seed=11 * dim + p)
    wl = W.make_workload(cfg)
    # force particles into the first and last cell of every dimension to exercise the fold
    for c in range(dim):
        wl.x[c][0] = 0.0
        wl.x[c][1] = cfg.np_dtype(0.01)
        wl.x[c][2] = np.nextafter(cfg.np_dtype(n), cfg.np_dtype(0))
        wl.x[c][3] = cfg.np_dtype(n - 0.5)
    g = O.grid_of(cfg)
    a = O.deposit(g, wl.x, wl.w)
    b = O.deposit(g, wl.x, wl.w, allpairs=True)
    assert np.max(np.abs(a - b)) <= 4e-15 * np.max(np.abs(b))


def test_deposit_allpairs_nonunit_spacing():
    g = O.Grid(3, (6, 5, 7), (0.5, 2.0, 1.25), 2, "f64")
    rng = np.random.default_rng(5)
    N = 60
    x = [rng.random(N) * g.n[c] * g.h[c] for c in range(3)]
    w = rng.random(N) + 0.5
    a = O.deposit(g, x, w)
    b = O.deposit(g, x, w, allpairs=True)
    assert np.max(np.abs(a - b)) <= 4e-15 * np.max(np.abs(b))
    vol = 0.5 * 2.0 * 1.25
    assert math.fsum(a) * vol == pytest.approx(math.fsum(w), rel=1e-14)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_charge_conservation(name):
    cfg = W.CONFIGS[name].scaled(60000)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    rho = O.deposit(g, wl.x, wl.w)
    tot_w = math.fsum(wl.w.astype(np.float64))
    assert abs(math.fsum(rho) * cfg.h ** cfg.dim - tot_w) <= 1e-13 * tot_w
    assert np.all(rho >= 0.0)


@pytest.mark.parametrize("p", [1, 2, 3])
def test_single_particle_is_tensor_product_of_1d_weights(p):
    n = 8
    g = O.Grid(3, (n, n, n), (1.0, 1.0, 1.0), p, "f64")
    pos = (5.25, 0.5, 7.75)
    x = [np.array([t]) for t in pos]
    rho = O.deposit(g, x, np.array([2.5])).reshape(n, n, n)
    want = np.zeros((n, n, n))
    sten = [O.stencil_1d(g, c, x[c]) for c in range(3)]
    for kz, wz in zip(*sten[2]):
        for ky, wy in zip(*sten[1]):
            for kx, wx in zip(*sten[0]):
                want[kz, ky, kx] += 2.5 * wx * wy * wz
    assert np.allclose(rho, want, atol=1e-16)
    assert np.count_nonzero(rho) <= (p + 1) ** 3


@pytest.mark.parametrize("p", [1, 2, 3])
def test_one_particle_per_node_gives_uniform_density(p):
    n, h = 8, 0.5
    g = O.Grid(2, (n, n), (h, h), p, "f64")
    jj, ii = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    x = [np.ascontiguousarray((ii.ravel() * h).astype(np.float64)),
         np.ascontiguousarray((jj.ravel() * h).astype(np.float64))]
    rho = O.deposit(g, x, np.full(n * n, 3.0))
    assert np.allclose(rho, 3.0 / h ** 2, rtol=1e-15)


@pytest.mark.parametrize("p", [1, 2, 3])
def test_shift_by_one_cell_rolls_rho_exactly(p):
    cfg = small_cfg(2, p, "f64", 4000, n=16, seed=3)
    wl = W.make_workload(cfg)
    # positions on a 2^-20 lattice, so x+1 (mod 16) is exactly representable
    x = [np.floor(a * 2 ** 20) / 2 ** 20 for a in wl.x]
    g = O.grid_of(cfg)
    rho = O.deposit(g, x, wl.w).reshape(16, 16)
    xs = [np.mod(x[0] + 1.0, 16.0), x[1]]
    rho_s = O.deposit(g, xs, wl.w).reshape(16, 16)
    assert np.array_equal(rho_s, np.roll(rho, 1, axis=1))
    ys = [x[0], np.mod(x[1] + 1.0, 16.0)]
    assert np.array_equal(O.deposit(g, ys, wl.w).reshape(16, 16), np.roll(rho, 1, axis=0))


@pytest.mark.parametrize("p", [1, 2, 3])
def test_first_moment_away_from_the_seam(p):
    n = 16
    g = O.Grid(2, (n, n), (1.0, 1.0), p, "f64")
    rng = np.random.default_rng(7)
    N = 3000
    x = [3.0 + 10.0 * rng.random(N), 3.0 + 10.0 * rng.random(N)]
    w = rng.random(N)
    rho = O.deposit(g, x, w).reshape(n, n)
    jx = np.arange(n, dtype=np.float64)
    assert math.fsum((rho * jx[None, :]).ravel()) == pytest.approx(math.fsum(w * x[0]), rel=1e-13)
    assert math.fsum((rho * jx[:, None]).ravel()) == pytest.approx(math.fsum(w * x[1]), rel=1e-13)


def test_deposit_is_order_independent_to_rounding():
    cfg = W.CONFIGS["cfg3"].scaled(50000, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    rho_u = O.deposit(g, wl.x, wl.w)
    xo, vo, wo, perm, off = O.sort(g, wl.x, wl.v, wl.w)
    rho_s = O.deposit(g, xo, wo)
    assert np.max(np.abs(rho_u - rho_s)) <= 1e-13 * np.max(rho_u)
