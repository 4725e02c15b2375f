"""pic_deposit_static: the deposit for callers that cannot allocate device memory.

Some users of the library are only handed their input and output buffers: a plug-in inside an application that owns
the device heap, code on a latency budget where cudaMalloc / cudaFree are ruled out because they may synchronise the
device, a process that starts after all GPU memory went into pools.  pic_deposit needs a caller-allocated workspace on
fp32 grids (the double-precision sums); pic_deposit_static keeps those sums in a fixed 16 MiB array inside the library
instead and takes no workspace.  These tests check that it gives the density of the existing path, pic_deposit with a
workspace, within the tolerance the other deposit tests use (parity.TOL_RHO), and that of the oracle.

The array is shared by all calls and keeps the last call's sums, so every case makes TWO calls in a row -- on different
particles and on grids of different sizes, the larger first -- and checks both: a call that did not clear what it
uses, or cleared too little, fails the second comparison.

This file is named to be collected last: pytest -x stops at the first failure, and a failure here must not hide the
parity tests.  It passes on its own in a fresh process (the first call does the one-time address look-up) and after
the rest of the suite.
"""
import numpy as np
import pytest

import pic_workloads as W
from parity import TOL_RHO, err_rho, to_dev

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _mods():
    import oracle as O
    import paper_1603_02886_b200 as B
    return O, B


def _case(name, N, n, order, seed):
    cfg = W.CONFIGS[name].scaled(N, n=n, order=order, dtype="f32", seed=seed)
    return cfg, W.make_workload(cfg)


def _both_paths(O, B, cfg, wl):
    """rho of the existing path (workspace), of the no-allocation path, and of the oracle, for one particle set."""
    g = B.grid_of(cfg)
    x, w = to_dev(wl.x), to_dev([wl.w])[0]
    ws = torch.empty(B.pic_workspace_bytes(g, cfg.N), dtype=torch.uint8, device="cuda")
    rho_ws = torch.full((g.cells,), 5.0, dtype=torch.float32, device="cuda")          # must be overwritten
    B.pic_deposit(g, x, w, rho_ws, B.PIC_ORDER_UNSORTED, None, ws)
    rho_st = torch.full((g.cells,), -3.0, dtype=torch.float32, device="cuda")
    B.pic_deposit_static(g, x, w, rho_st)
    assert B.pic_last_launch_count() == 2          # the deposit kernel and the rounding kernel
    torch.cuda.synchronize()
    return rho_ws.cpu().numpy(), rho_st.cpu().numpy(), O.deposit(O.grid_of(cfg), wl.x, wl.w)


# (first call, second call): the second grid is smaller, or the same size with other particles, so stale sums of the
# first call sit exactly where the second one adds
PAIRS = [
    (("cfg3", 150_001, (32, 32, 32), 3, 1), ("cfg3", 40_003, (16, 8, 4), 3, 2)),
    (("cfg3", 60_000, (32, 16, 8), 1, 3), ("cfg4", 90_001, (32, 16, 8), 2, 4)),
    (("cfg2", 200_003, (64, 64), 2, 5), ("cfg1", 50_000, (64, 64), 1, 6)),
    (("cfg2", 30_000, (96, 40), 3, 7), ("cfg2", 31, (8, 4), 3, 8)),
]


@pytest.mark.parametrize("first,second", PAIRS)
def test_static_deposit_matches_workspace_deposit_twice_in_a_row(first, second):
    O, B = _mods()
    for spec in (first, second):
        cfg, wl = _case(*spec)
        rho_ws, rho_st, rho_ref = _both_paths(O, B, cfg, wl)
        tol = TOL_RHO["f32"]
        assert err_rho(rho_st, rho_ws) <= tol, spec
        assert err_rho(rho_st, rho_ref) <= tol, spec
        # both round the same double sums once: they differ at most in the last bit of a float
        assert np.max(np.abs(rho_st.astype(np.float64) - rho_ws)) <= 2.0 ** -23 * np.max(np.abs(rho_ws)), spec
        tot = float(np.sum(wl.w.astype(np.float64)))
        assert abs(float(np.sum(rho_st.astype(np.float64))) * cfg.h ** cfg.dim - tot) <= 2e-6 * tot, spec


def test_static_deposit_same_particles_twice_gives_the_same_density():
    """The second of two identical calls must not see the first one's sums (it would give 2 rho)."""
    O, B = _mods()
    cfg, wl = _case("cfg3", 100_000, (32, 32, 32), 3, 11)
    g = B.grid_of(cfg)
    x, w = to_dev(wl.x), to_dev([wl.w])[0]
    rho_ref = O.deposit(O.grid_of(cfg), wl.x, wl.w)
    rho = torch.empty((g.cells,), dtype=torch.float32, device="cuda")
    for _ in range(2):
        rho.fill_(9.0)
        B.pic_deposit_static(g, x, w, rho)
        assert err_rho(rho.cpu().numpy(), rho_ref) <= TOL_RHO["f32"]


def test_static_deposit_empty_particle_set_clears_rho():
    _, B = _mods()
    cfg, wl = _case("cfg3", 5_000, (16, 16, 16), 2, 12)
    g = B.grid_of(cfg)
    x, w = to_dev(wl.x), to_dev([wl.w])[0]
    rho = torch.empty((g.cells,), dtype=torch.float32, device="cuda")
    B.pic_deposit_static(g, x, w, rho)                      # leaves sums behind
    empty = [torch.empty(0, dtype=torch.float32, device="cuda") for _ in range(3)]
    rho.fill_(4.0)
    B.pic_deposit_static(g, empty, torch.empty(0, dtype=torch.float32, device="cuda"), rho)
    assert torch.count_nonzero(rho).item() == 0


def test_static_deposit_at_the_maximum_grid():
    """128^3 nodes = PIC_DEPOSIT_STATIC_MAX_NODES exactly: accepted, and the whole array is usable."""
    O, B = _mods()
    cfg, wl = _case("cfg3", 400_000, (128, 128, 128), 3, 13)
    assert B.grid_of(cfg).cells == B.PIC_DEPOSIT_STATIC_MAX_NODES
    rho_ws, rho_st, rho_ref = _both_paths(O, B, cfg, wl)
    assert err_rho(rho_st, rho_ws) <= TOL_RHO["f32"]
    assert err_rho(rho_st, rho_ref) <= TOL_RHO["f32"]


def test_static_deposit_rejects_what_it_cannot_do():
    _, B = _mods()
    # one node more than the array holds: a clear error, and rho is not touched
    big = B.Grid(3, (128, 128, 129), (1.0, 1.0, 1.0), 1, "f32")
    x = [torch.zeros(4, dtype=torch.float32, device="cuda") for _ in range(3)]
    w = torch.ones(4, dtype=torch.float32, device="cuda")
    rho = torch.full((big.cells,), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(B.PicError, match="PIC_DEPOSIT_STATIC_MAX_NODES"):
        B.pic_deposit_static(big, x, w, rho)
    torch.cuda.synchronize()
    assert torch.all(rho == 7.0).item()
    # fp64 grids need no scratch at all: pic_deposit(ws=None) is the call for them
    g64 = B.Grid(2, (16, 16), (1.0, 1.0), 1, "f64")
    x64 = [torch.zeros(4, dtype=torch.float64, device="cuda") for _ in range(2)]
    with pytest.raises(B.PicError, match="unsupported"):
        B.pic_deposit_static(g64, x64, torch.ones(4, dtype=torch.float64, device="cuda"),
                             torch.zeros(256, dtype=torch.float64, device="cuda"))
