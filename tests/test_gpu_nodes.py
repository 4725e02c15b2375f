"""GPU parity of pic_deposit_nodes, the collision-free "threads on splines" deposit (
PAPER.md:202-204 section 3.3.1, Fig. 6, App. B 447-469).  Its additions happen in a fixed order -- ascending position
of the sorted particles -- in individually rounded double operations, which is exactly what the oracle's pic_ref_deposit
does on the sorted arrays (oracle/pic_ref.c: particle order, gcc -ffp-contract=off).  So the bar here is BIT-EXACT:
rho (fp64) equal to the oracle's double sum, rho (fp32) equal to that sum rounded once."""
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


def _sorted_inputs(O, cfg, wl=None):
    wl = wl or W.make_workload(cfg)
    xs, vs, ws, perm, off = O.sort(O.grid_of(cfg), wl.x, wl.v, wl.w)
    return xs, ws, off


def _gpu_nodes(B, g, xs, wsrt, off):
    n = wsrt.shape[0]
    x = to_dev(xs)
    w = to_dev([wsrt])[0]
    offd = torch.from_numpy(np.concatenate([off.astype(np.int32), np.zeros(3, np.int32)])).cuda()
    rho = torch.full((g.cells,), float("nan"), dtype=g.torch_dtype, device="cuda")
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    B.pic_deposit_nodes(g, x, w, rho, offd, ws)
    torch.cuda.synchronize()
    return rho.cpu().numpy()


def _bits(a):
    a = np.ascontiguousarray(a)
    return a.view(np.uint64 if a.dtype == np.float64 else np.uint32)


CASES = []
for dtype in ("f64", "f32"):
    for order in (1, 2, 3):
        CASES += [("cfg2", 60_003, dict(n=(32, 24)), order, dtype),
                  ("cfg3", 70_001, dict(n=(16, 12, 8)), order, dtype),
                  ("cfg3", 3_000, dict(n=(order + 1, order + 1, order + 1)), order, dtype),     # the smallest legal grid
                  ("cfg2", 2_000, dict(n=(order + 1, order + 2)), order, dtype)]


@pytest.mark.parametrize("name,N,kw,order,dtype", CASES)
def test_nodes_bit_exact(name, N, kw, order, dtype):
    O, B = _mods()
    cfg = W.CONFIGS[name].scaled(N, order=order, dtype=dtype, **kw)
    xs, wsrt, off = _sorted_inputs(O, cfg)
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)                   # double, particle order
    got = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)
    want = ref if dtype == "f64" else ref.astype(np.float32)
    assert np.array_equal(_bits(got), _bits(want)), "max rel diff %g" % err_rho(got, ref)


@pytest.mark.parametrize("h", [0.5, 0.3, 3.0])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_nodes_bit_exact_spacing(h, dtype):
    """h != 1: the power-of-two (multiply) and the general (division) form of t = x/h (R13), 1/prod(h) as the oracle forms it."""
    O, B = _mods()
    cfg = W.CONFIGS["cfg3"].scaled(50_000, n=(12, 10, 14), h=h, order=2, dtype=dtype)
    xs, wsrt, off = _sorted_inputs(O, cfg)
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)
    got = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)
    want = ref if dtype == "f64" else ref.astype(np.float32)
    assert np.array_equal(_bits(got), _bits(want))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_nodes_clustered_uses_the_warp_path(dtype):
    """cfg4's blob: nodes with far more than 4096 particles around them are summed by a warp, in the same order."""
    O, B = _mods()
    cfg = W.CONFIGS["cfg4"].scaled(400_000, n=(16, 16, 16), dtype=dtype)
    xs, wsrt, off = _sorted_inputs(O, cfg)
    cnt = np.diff(off).reshape(16, 16, 16)
    assert cnt[6:10, 6:10, 6:10].sum() > 4096                  # the 4^3 cells around a central node
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)
    got = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)
    want = ref if dtype == "f64" else ref.astype(np.float32)
    assert np.array_equal(_bits(got), _bits(want))
    again = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)        # run to run
    assert np.array_equal(_bits(got), _bits(again))


def test_nodes_negative_weights_and_edge_positions():
    O, B = _mods()
    cfg = W.CONFIGS["cfg5"].scaled(40_000, n=(8, 8, 8))
    wl = W.make_workload(cfg)
    w = wl.w.copy()
    w[::3] *= -1.0                                              # charges of both signs: sums cancel
    x = [a.copy() for a in wl.x]
    x[0][::7] = 0.0
    x[1][::11] = np.nextafter(8.0, 0.0)
    x[2][::13] = np.floor(x[2][::13])
    wl2 = W.Workload(cfg, x, wl.v, w, wl.E, wl.modes)
    xs, wsrt, off = _sorted_inputs(O, cfg, wl2)
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)
    got = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)
    assert np.array_equal(_bits(got), _bits(ref))


@pytest.mark.parametrize("N", [0, 1, 33])
def test_nodes_tiny(N):
    O, B = _mods()
    cfg = W.CONFIGS["cfg2"].scaled(N, n=(8, 8))
    xs, wsrt, off = _sorted_inputs(O, cfg)
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)
    got = _gpu_nodes(B, B.grid_of(cfg), xs, wsrt, off)
    assert np.array_equal(_bits(got), _bits(ref))


@pytest.mark.parametrize("what", ["unsorted", "garbage", "shifted"])
def test_nodes_offsets_that_do_not_describe_the_order(what):
    """The call stays correct (within the deposit tolerance) when cell_offsets is not the order of p."""
    O, B = _mods()
    cfg = W.CONFIGS["cfg3"].scaled(80_000, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    go = O.grid_of(cfg)
    xs, vs, wsrt, perm, off = O.sort(go, wl.x, wl.v, wl.w)
    if what == "unsorted":
        x, w, o = wl.x, wl.w, off                                # valid offsets, particles in random order
    elif what == "garbage":
        rng = np.random.default_rng(3)
        x, w, o = xs, wsrt, rng.integers(-10, cfg.N + 10, off.size)
    else:
        x, w = xs, wsrt                                          # walkable but wrong: every boundary one particle late
        o = np.minimum(off + 1, cfg.N)
        o[0] = 0
    ref = O.deposit(go, x, w)
    got = _gpu_nodes(B, B.grid_of(cfg), x, w, np.asarray(o))
    assert err_rho(got, ref) <= TOL_RHO[cfg.dtype]


# ---- pic_deposit_replicated: threads on buckets with data replication (setrho 3.3.3) ----------------
def _gpu_replicated(B, g, xs, wsrt, off):
    n = wsrt.shape[0]
    x = to_dev(xs)
    w = to_dev([wsrt])[0]
    offd = torch.from_numpy(np.concatenate([off.astype(np.int32), np.zeros(3, np.int32)])).cuda()
    rho = torch.full((g.cells,), float("nan"), dtype=g.torch_dtype, device="cuda")
    ws = torch.full((B.pic_deposit_replicated_bytes(g, n),), 0xA5, dtype=torch.uint8, device="cuda")
    B.pic_deposit_replicated(g, x, w, rho, offd, ws)
    torch.cuda.synchronize()
    return rho.cpu().numpy()


@pytest.mark.parametrize("name,N,kw,order,dtype", CASES)
def test_replicated_parity_and_reproducibility(name, N, kw, order, dtype):
    """Within the deposit tolerance of the oracle (the association differs: sums per cell first), and bit-identical from run
    to run (no atomics, fixed order)."""
    O, B = _mods()
    cfg = W.CONFIGS[name].scaled(N, order=order, dtype=dtype, **kw)
    xs, wsrt, off = _sorted_inputs(O, cfg)
    ref = O.deposit(O.grid_of(cfg), xs, wsrt)
    got = _gpu_replicated(B, B.grid_of(cfg), xs, wsrt, off)
    assert err_rho(got, ref) <= TOL_RHO[dtype]
    again = _gpu_replicated(B, B.grid_of(cfg), xs, wsrt, off)
    assert np.array_equal(_bits(got), _bits(again))
    scale = np.prod([cfg.h] * cfg.dim)
    assert abs(np.sum(got.astype(np.float64)) * scale - np.sum(wsrt.astype(np.float64))) <= (1e-12 if dtype == "f64" else 2e-6) * np.sum(np.abs(wsrt))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_replicated_clustered_and_spacing(dtype):
    O, B = _mods()
    for cfg in (W.CONFIGS["cfg4"].scaled(400_000, n=(16, 16, 16), dtype=dtype),
                W.CONFIGS["cfg3"].scaled(50_000, n=(12, 10, 14), h=0.3, order=2, dtype=dtype)):
        xs, wsrt, off = _sorted_inputs(O, cfg)
        ref = O.deposit(O.grid_of(cfg), xs, wsrt)
        got = _gpu_replicated(B, B.grid_of(cfg), xs, wsrt, off)
        assert err_rho(got, ref) <= TOL_RHO[dtype]


@pytest.mark.parametrize("what", ["unsorted", "garbage", "shifted"])
def test_replicated_offsets_that_do_not_describe_the_order(what):
    O, B = _mods()
    cfg = W.CONFIGS["cfg3"].scaled(80_000, n=(16, 16, 16))
    wl = W.make_workload(cfg)
    go = O.grid_of(cfg)
    xs, vs, wsrt, perm, off = O.sort(go, wl.x, wl.v, wl.w)
    if what == "unsorted":
        x, w, o = wl.x, wl.w, off
    elif what == "garbage":
        x, w, o = xs, wsrt, np.random.default_rng(3).integers(-10, cfg.N + 10, off.size)
    else:
        x, w = xs, wsrt
        o = np.minimum(off + 1, cfg.N)
        o[0] = 0
    ref = O.deposit(go, x, w)
    got = _gpu_replicated(B, B.grid_of(cfg), x, w, np.asarray(o))
    assert err_rho(got, ref) <= TOL_RHO[cfg.dtype]
