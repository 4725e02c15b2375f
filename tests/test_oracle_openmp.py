"""The OpenMP build of the oracle (oracle.build_openmp(): the same source with -fopenmp, timed by bench.py's
cpu_baseline and never used for parity) must compute what the plain build computes: perm, cell offsets and the pushed
x, v bit for bit (those loops are only split over threads); rho to rounding (one private grid per thread, added up
node by node, so the order of the additions differs from particle order)."""
import os

import numpy as np
import pytest

import oracle as O
import pic_workloads as W


def _omp_or_skip():
    try:
        O.build_openmp()
        import ctypes
        ctypes.CDLL("libgomp.so.1")
    except Exception as e:                      # no OpenMP runtime / compiler support on this box
        pytest.skip("OpenMP build unavailable: %s" % e)


@pytest.mark.parametrize("name,N,kw,threads", [
    ("cfg1", 100_000, dict(), 4),
    ("cfg2", 60_001, dict(n=(64, 64)), 3),
    ("cfg3", 120_001, dict(n=(32, 32, 32)), 7),
    ("cfg4", 90_000, dict(n=(16, 16, 16)), 16),
    ("cfg5", 8 * 16 ** 3 + 5, dict(n=(16, 16, 16)), 2),
    ("cfg3", 5, dict(n=(8, 8, 8)), 8),          # fewer particles than threads
])
def test_openmp_build_equals_plain_build(name, N, kw, threads):
    _omp_or_skip()
    cfg = W.CONFIGS[name].scaled(N, **kw)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    a = O.step(g, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm)
    b = O.step_openmp(g, wl.x, wl.v, wl.w, wl.E, cfg.dt, cfg.qm, threads)
    assert np.array_equal(a["perm"], b["perm"])
    assert np.array_equal(a["cell_offsets"], b["cell_offsets"])
    for c in range(cfg.dim):
        assert np.array_equal(a["x"][c], b["x"][c]) and np.array_equal(a["v"][c], b["v"][c])
    assert np.array_equal(a["w"], b["w"])
    assert np.max(np.abs(a["rho"] - b["rho"])) <= 1e-13 * np.max(np.abs(a["rho"]))
    # a second step from the first one's output (the steady-state leg bench.py times)
    a2 = O.step(g, a["x"], a["v"], a["w"], wl.E, cfg.dt, cfg.qm)
    b2 = O.step_openmp(g, b["x"], b["v"], b["w"], wl.E, cfg.dt, cfg.qm, threads)
    assert np.array_equal(a2["perm"], b2["perm"]) and np.array_equal(a2["cell_offsets"], b2["cell_offsets"])
    assert np.max(np.abs(a2["rho"] - b2["rho"])) <= 1e-13 * np.max(np.abs(a2["rho"]))
