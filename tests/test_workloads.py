"""The seeded input generators (pic_workloads): RNG cross-check against an independent
numpy statement of splitmix64, distribution shape, and the regime the paper quotes
("23 % of particles are misplaced")."""
import math

import numpy as np
import pytest

import pic_workloads as W

G = np.uint64(0x9E3779B97F4A7C15)


def _mix64(z):
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def np_uniform01(seed, stream, i0, n):
    with np.errstate(over="ignore"):
        key = _mix64(np.array([seed], np.uint64) + G * np.uint64(stream + 1))[0]
        i = np.arange(i0, i0 + n, dtype=np.uint64)
        r = _mix64(key + G * (i + np.uint64(1)))
    return (r >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def test_rng_matches_numpy_splitmix64():
    for seed, stream, i0 in [(0, 0, 0), (0, 20, 12345), (7, 3, 10 ** 9), (2 ** 40 + 1, 54, 5)]:
        a = W.uniform01(seed, stream, i0, 1000)
        b = np_uniform01(seed, stream, i0, 1000)
        assert np.array_equal(a, b)
        assert np.all((a >= 0) & (a < 1))
    # splitmix64 reference outputs for state seed 0 (first output = mix64(G))
    assert int(_mix64(np.array([G], np.uint64))[0]) == 0xE220A8397B1DCDAF


def test_streams_are_distinct_and_uniform():
    a = W.uniform01(0, 0, 0, 200000)
    b = W.uniform01(0, 1, 0, 200000)
    assert abs(a.mean() - 0.5) < 3e-3 and abs(a.var() - 1 / 12) < 2e-3
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.01
    assert abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 0.01


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg5"])
def test_workload_shapes_and_ranges(name):
    cfg = W.CONFIGS[name].scaled(100000)
    wl = W.make_workload(cfg)
    assert len(wl.x) == len(wl.v) == len(wl.E) == cfg.dim
    for c in range(cfg.dim):
        assert wl.x[c].dtype == cfg.np_dtype and wl.x[c].shape == (cfg.N,)
        assert np.all(wl.x[c] >= 0) and np.all(wl.x[c] < cfg.np_dtype(cfg.L[c]))
        assert abs(wl.x[c].mean() / cfg.L[c] - 0.5) < 0.01
        assert abs(wl.v[c].mean()) < 0.02 and abs(wl.v[c].std() - 1.0) < 0.02
        assert wl.E[c].shape == (cfg.cells,) and wl.E[c].dtype == cfg.np_dtype
    if cfg.weights == "inv_n":
        assert np.all(wl.w == 1.0 / cfg.N)
    elif cfg.weights == "uniform":
        assert wl.w.min() >= 0.5 and wl.w.max() < 1.5 and abs(wl.w.mean() - 1.0) < 0.01
    else:
        assert np.all(wl.w == 1.0)
    # deterministic
    wl2 = W.make_workload(cfg)
    assert all(np.array_equal(a, b) for a, b in zip(wl.x + wl.v, wl2.x + wl2.v))
    # a prefix of a larger workload is the smaller workload (index addressable)
    wl3 = W.make_workload(cfg.scaled(1000))
    assert np.array_equal(wl3.x[0], wl.x[0][:1000]) and np.array_equal(wl3.v[1], wl.v[1][:1000])


def test_fraction_of_particles_changing_cell_matches_the_papers_regime():
    # dt = 0.1, sigma_v = 1, h = 1: 8.0 % cross a face per dimension, 22.1 % change cell in 3-D
    cfg = W.CONFIGS["cfg3"].scaled(400000)
    wl = W.make_workload(cfg)
    moved = np.zeros(cfg.N, bool)
    for c in range(3):
        xn = wl.x[c].astype(np.float64) + cfg.dt * wl.v[c].astype(np.float64)
        moved |= np.floor(xn) != np.floor(wl.x[c].astype(np.float64))
    per_dim = cfg.dt * math.sqrt(2 / math.pi)            # E|v| dt / h
    assert per_dim == pytest.approx(0.0798, abs=1e-4)
    assert moved.mean() == pytest.approx(1 - (1 - per_dim) ** 3, abs=0.004)
    assert 0.21 < moved.mean() < 0.24                    # "23 % misplaced"


def test_clustered_config_has_a_dense_centre():
    cfg = W.CONFIGS["cfg4"].scaled(1_000_000)
    wl = W.make_workload(cfg)
    for c in range(3):
        assert np.all(wl.x[c] >= 0) and np.all(wl.x[c] < np.float32(128.0))
    r2 = sum((wl.x[c].astype(np.float64) - 64.0) ** 2 for c in range(3))
    # 70 % Gaussian sigma = 4: P(r < 8) = chi3 cdf(2 sigma) = 0.7385; uniform background adds ~0.03 %
    assert (r2 < 64.0).mean() == pytest.approx(0.7 * 0.7385, abs=0.004)
    centre = (np.floor(wl.x[0]) == 64) & (np.floor(wl.x[1]) == 64) & (np.floor(wl.x[2]) == 64)
    want = 0.7 * cfg.N * (math.erf(1 / (4 * math.sqrt(2))) / 2) ** 3      # one cell next to the centre
    assert centre.sum() == pytest.approx(want, rel=0.15)


def test_field_modes_are_low_k_and_electrostatic():
    cfg = W.CONFIGS["cfg3"]
    m = W.field_modes(cfg)
    assert m["k"].shape == (8, 3) and np.all(np.abs(m["k"]) <= 2) and np.all(np.any(m["k"] != 0, axis=1))
    assert np.allclose(np.linalg.norm(m["dir"], axis=1), 1.0)
    assert np.all((m["amp"] >= 0.5 / 8) & (m["amp"] < 1.0 / 8))
    small = cfg.scaled(10, n=(8, 8, 8))
    E, mm = W.make_field(small)
    jz, jy, jx = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    want = np.zeros((8, 8, 8))
    for a in range(8):
        ph = (mm["k"][a, 0] * jx + mm["k"][a, 1] * jy + mm["k"][a, 2] * jz) / 8.0
        want += mm["amp"][a] * mm["dir"][a, 1] * np.sin(2 * np.pi * ph + mm["phase"][a])
    assert np.allclose(E[1].reshape(8, 8, 8), want, atol=1e-6)
