"""Pins of the oracle's gather + accel + push (O4) and of the composed step (O5)."""
import math

import numpy as np
import pytest

import oracle as O
import pic_workloads as W


def small_cfg(dim, p, dtype, N, n=8, seed=0, modes=3):
    return W.Config("t", dim, tuple([n] * dim), N, dtype, p, "uniform", modes, 1, seed=seed)


# ------------------------------------------------------------------------- gather
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("p", [1, 2, 3])
@pytest.mark.parametrize("dim", [2, 3])
def test_gather_equals_allnodes_bruteforce(dim, p, dtype):
    n = 6 if dim == 3 else 8
    cfg = small_cfg(dim, p, dtype, 70, n=n, seed=5 * dim + p)
    wl = W.make_workload(cfg)
    for c in range(dim):
        wl.x[c][0] = 0.0
        wl.x[c][1] = np.nextafter(cfg.np_dtype(n), cfg.np_dtype(0))
    g = O.grid_of(cfg)
    a = O.gather(g, wl.x, wl.E)
    b = O.gather(g, wl.x, wl.E, allnodes=True)
    for c in range(dim):
        assert np.max(np.abs(a[c] - b[c])) <= 1e-15


@pytest.mark.parametrize("p", [1, 2, 3])
def test_gather_reproduces_constants_and_linear_fields(p):
    n = 16
    g = O.Grid(3, (n, n, n), (1.0, 1.0, 1.0), p, "f64")
    rng = np.random.default_rng(2)
    N = 500
    x = [3.0 + 10.0 * rng.random(N) for _ in range(3)]
    const = [np.full(g.cells, 0.375), np.full(g.cells, -2.0), np.full(g.cells, 7.0)]
    Ep = O.gather(g, x, const)
    for c, val in enumerate((0.375, -2.0, 7.0)):
        assert np.max(np.abs(Ep[c] - val)) <= 4e-15 * abs(val)      # partition of unity
    jz, jy, jx = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    lin = [np.ascontiguousarray((1.0 + 2.0 * jx - 0.5 * jy + 0.25 * jz).ravel().astype(np.float64))] * 3
    Ep = O.gather(g, x, lin)
    want = 1.0 + 2.0 * x[0] - 0.5 * x[1] + 0.25 * x[2]
    assert np.max(np.abs(Ep[0] - want)) <= 1e-13                      # first moment


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5"])
def test_gather_is_the_adjoint_of_deposit(name):
    cfg = W.CONFIGS[name].scaled(20000)
    if cfg.dim == 3:
        cfg = cfg.scaled(20000, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    rho = O.deposit(g, wl.x, wl.w)
    Ep = O.gather(g, wl.x, wl.E)
    w = wl.w.astype(np.float64)
    for c in range(cfg.dim):
        lhs = math.fsum(w * Ep[c])
        rhs = math.fsum(rho * wl.E[c].astype(np.float64)) * cfg.h ** cfg.dim
        scale = math.fsum(np.abs(w * Ep[c]))
        assert abs(lhs - rhs) <= 1e-13 * scale


# --------------------------------------------------------------------------- push
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_push_with_zero_field_is_free_streaming(dtype):
    cfg = small_cfg(3, 2, dtype, 5000, seed=4)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    Z = [np.zeros(g.cells, cfg.np_dtype)] * 3
    xn, vn = O.push(g, wl.x, wl.v, Z, 0.1, 1.0)
    for c in range(3):
        assert np.array_equal(vn[c], wl.v[c])
        want = wl.x[c].astype(np.float64) + 0.1 * wl.v[c].astype(np.float64)
        want = (want - 8.0 * np.floor(want / 8.0)).astype(cfg.np_dtype)
        want[(want >= 8.0) | (want < 0)] = 0
        assert np.array_equal(xn[c], want)
        assert np.all((xn[c] >= 0) & (xn[c] < cfg.np_dtype(8.0)))


def test_push_with_constant_field():
    cfg = small_cfg(2, 3, "f64", 3000, seed=6)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    Ec = [np.full(g.cells, 0.5), np.full(g.cells, -0.25)]
    xn, vn = O.push(g, wl.x, wl.v, Ec, 0.1, 2.0)
    for c, e0 in enumerate((0.5, -0.25)):
        assert np.max(np.abs(vn[c] - (wl.v[c] + 2.0 * 0.1 * e0))) <= 1e-15
        want = wl.x[c] + 0.1 * vn[c]
        want -= 8.0 * np.floor(want / 8.0)
        assert np.max(np.abs(xn[c] - want)) <= 2e-15


def test_push_uses_the_new_velocity_and_the_field_at_the_old_position():
    # v(t+1) = v(t) + dt E(t);  x(t+1) = x(t) + dt v(t+1)
    n = 8
    g = O.Grid(2, (n, n), (1.0, 1.0), 1, "f64")
    Ex = np.tile(np.arange(n, dtype=np.float64), n)     # E_x[j] = j_x: linear in x
    Ey = np.zeros(g.cells)
    x = [np.array([2.5]), np.array([4.0])]
    v = [np.array([1.0]), np.array([0.0])]
    xn, vn = O.push(g, x, v, [Ex, Ey], 0.5, 2.0)
    assert vn[0][0] == 1.0 + 2.0 * 0.5 * 2.5            # E at the OLD x = 2.5
    assert xn[0][0] == 2.5 + 0.5 * vn[0][0]             # moved with the NEW v
    assert vn[1][0] == 0.0 and xn[1][0] == 4.0


def test_push_periodic_wrap_edge_cases():
    n = 8
    for dtype in ("f64", "f32"):
        g = O.Grid(2, (n, n), (1.0, 1.0), 1, dtype)
        dt_ = g.np_dtype
        Z = [np.zeros(g.cells, dt_)] * 2
        x = [np.array([0.05, 7.95, 1e-9, 0.0, 7.999999], dt_), np.full(5, 4.0, dt_)]
        v = [np.array([-1.0, 1.0, -1.000001e-7, -80.0, 0.25], dt_), np.zeros(5, dt_)]
        xn, _ = O.push(g, x, v, Z, 0.1, 1.0)
        assert xn[0][0] == pytest.approx(7.95, abs=1e-6)
        assert xn[0][1] == pytest.approx(0.05, abs=1e-6)
        assert 0.0 <= xn[0][2] < 8.0            # -1e-15 + 8 rounds to 8 -> stored as 0
        assert xn[0][3] == 0.0                  # exactly one box length to the left
        assert np.all((xn[0] >= 0) & (xn[0] < dt_(8.0)))


@pytest.mark.parametrize("p", [1, 2, 3])
def test_single_fourier_mode_projection_is_sinc_power(p):
    """Config 1's field E_x[j] = sin(2 pi j_x/n_x).  The interpolated field is
    sum_j W_p(x-j) sin(k j); its projection on the fundamental is exactly
    sinc(k h/2)^(p+1) (Fourier transform of the B-spline)."""
    n = 64
    cfg = W.Config("t", 2, (n, n), 1, "f64", p, "one", 0, 1)
    E, _ = W.make_field(cfg)
    assert np.max(np.abs(E[1])) == 0.0
    assert np.allclose(E[0].reshape(n, n)[5], np.sin(2 * np.pi * np.arange(n) / n), atol=1e-15)
    g = O.grid_of(cfg)
    M = 32                                              # samples per cell, uniform lattice
    xs = (np.arange(n * M) + 0.5) / M
    x = [xs, np.full(xs.size, 17.3)]
    Ep = O.gather(g, x, E)[0]
    k = 2 * np.pi / n
    proj = 2.0 * np.mean(Ep * np.sin(k * xs))
    s = math.sin(k / 2) / (k / 2)
    assert proj == pytest.approx(s ** (p + 1), abs=1e-6)
    if p == 1:
        assert s ** 2 == pytest.approx(0.999197, abs=1e-6)
        assert np.max(np.abs(Ep - np.sin(k * xs))) <= k * k / 8 * 1.0001   # linear interpolation bound
    # and the push built on it: v' - v = qm dt E(x), x' = x + dt v'
    v = [np.full(xs.size, 0.3), np.full(xs.size, -0.2)]
    xn, vn = O.push(g, x, v, E, 0.1, 1.0)
    assert np.max(np.abs((vn[0] - 0.3) / 0.1 - Ep)) <= 1e-14
    assert np.max(np.abs(vn[0] - 0.3 - 0.1 * s ** (p + 1) * np.sin(k * xs))) <= 0.1 * 2 * (1 - s ** (p + 1)) + 1e-4
    want = xs + 0.1 * vn[0]
    want -= n * np.floor(want / n)
    assert np.max(np.abs(xn[0] - want)) <= 1e-13
    assert np.array_equal(vn[1], v[1])


def test_interpolation_error_falls_4x_per_grid_doubling():
    errs = []
    for n in (32, 64, 128):
        cfg = W.Config("t", 2, (n, n), 1, "f64", 1, "one", 0, 1)
        E, _ = W.make_field(cfg)
        g = O.grid_of(cfg)
        xs = (np.arange(n * 8) + 0.5) / 8
        Ep = O.gather(g, [xs, np.full(xs.size, 1.0)], E)[0]
        errs.append(np.max(np.abs(Ep - np.sin(2 * np.pi * xs / n))))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.02)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.02)


# --------------------------------------------------------------------------- step
@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_step_is_sort_then_deposit_then_push(name):
    cfg = W.CONFIGS[name].scaled(30000)
    if cfg.dim == 3:
        cfg = cfg.scaled(30000, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    r = O.step(g, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm)
    xo, vo, wo, perm, off = O.sort(g, wl.x, wl.v, wl.w)
    assert np.array_equal(r["perm"], perm) and np.array_equal(r["cell_offsets"], off)
    assert np.array_equal(r["rho"], O.deposit(g, xo, wo))
    xn, vn = O.push(g, xo, vo, wl.E, cfg.dt, cfg.qm)
    xu, vu = O.push(g, wl.x, wl.v, wl.E, cfg.dt, cfg.qm)          # push commutes with the permutation
    for c in range(cfg.dim):
        assert np.array_equal(r["x"][c], xn[c]) and np.array_equal(r["v"][c], vn[c])
        assert np.array_equal(r["x"][c], xu[c][perm]) and np.array_equal(r["v"][c], vu[c][perm])
    assert np.array_equal(r["w"], wl.w[perm])
    rho_u = O.deposit(g, wl.x, wl.w)
    assert np.max(np.abs(r["rho"] - rho_u)) <= 1e-13 * np.max(rho_u)
    # do_sort = 0: same particles in the given order
    r0 = O.step(g, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm, do_sort=False)
    assert np.array_equal(r0["perm"], np.arange(cfg.N, dtype=np.int32))
    assert np.array_equal(r0["rho"], rho_u)
    for c in range(cfg.dim):
        assert np.array_equal(r0["x"][c], xu[c])


def test_multi_step_identity_is_the_composition_of_perms():
    cfg = W.CONFIGS["cfg2"].scaled(5000, n=(16, 16))
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    x, v, w = wl.x, wl.v, wl.w
    ident = np.arange(cfg.N)
    xu, vu = [a.copy() for a in wl.x], [a.copy() for a in wl.v]
    for _ in range(4):
        r = O.step(g, x, v, w, wl.E, cfg.dt, cfg.qm)
        ident = ident[r["perm"]]
        x, v, w = r["x"], r["v"], r["w"]
        xu, vu = O.push(g, xu, vu, wl.E, cfg.dt, cfg.qm)          # never sorted
    for c in range(cfg.dim):
        assert np.array_equal(x[c], xu[c][ident]) and np.array_equal(v[c], vu[c][ident])
    assert np.array_equal(w, wl.w[ident])
