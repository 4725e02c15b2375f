"""GPU parity of pic_field_solve and pic_step_selfconsistent (PAPER.md:81 step ii, 86, 88) against
oracle.field_solve / oracle.step_selfconsistent through the C ABI.  Floating point both sides (double arithmetic,
different transform algorithms): E and phi within 1e-12 of max |.| for fp64 grids, 1e-6 for fp32 grids (one rounding of
the stored rho and of the stored result); the closed-loop step at north_star's tolerances for rho, x, v."""
import numpy as np
import pytest

import pic_workloads as W
from parity import TOL_RHO, TOL_XV, err_rho, err_v, err_x, to_dev

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL_FIELD = {"f64": 1e-12, "f32": 1e-6}


def _mods():
    import oracle as O
    import paper_1603_02886_b200 as B
    return O, B


def _solve(B, g, rho, want_phi=True):
    r = torch.from_numpy(np.ascontiguousarray(rho)).cuda()
    E = [torch.full((g.cells,), float("nan"), dtype=g.torch_dtype, device="cuda") for _ in range(g.dim)]
    phi = torch.full((g.cells,), float("nan"), dtype=g.torch_dtype, device="cuda") if want_phi else None
    ws = torch.empty(B.pic_field_solve_bytes(g), dtype=torch.uint8, device="cuda")
    B.pic_field_solve(g, r, E, phi, ws)
    torch.cuda.synchronize()
    return (phi.cpu().numpy() if want_phi else None), [e.cpu().numpy() for e in E]


SHAPES = [((64, 64), (1.0, 1.0)), ((16, 128), (0.5, 0.25)), ((12, 10), (1.0, 0.3)), ((9, 7), (1.0, 1.0)),      # powers of two, others, odd
          ((32, 32, 32), (1.0, 1.0, 1.0)), ((8, 16, 4), (1.0, 2.0, 0.5)), ((12, 10, 14), (0.3, 1.0, 0.7)), ((5, 4, 3), (1.0, 1.0, 1.0)),
          ((2048, 4), (1.0, 1.0)), ((4, 1000), (1.0, 1.0))]                                                   # long lines: few lines per block


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n,h", SHAPES)
def test_field_solve_parity(n, h, dtype):
    O, B = _mods()
    d = len(n)
    go = O.Grid(d, n, h, 1, dtype)
    gb = B.Grid(d, n, h, 1, dtype)
    rng = np.random.default_rng(7)
    rho = (rng.normal(size=go.cells) + 2.5).astype(go.np_dtype)       # non-zero mean: dropped
    phi_r, E_r = O.field_solve(go, rho)
    phi_g, E_g = _solve(B, gb, rho)
    tol = TOL_FIELD[dtype]
    assert np.max(np.abs(phi_g - phi_r)) <= tol * np.max(np.abs(phi_r))
    for c in range(d):
        assert np.max(np.abs(E_g[c] - E_r[c])) <= tol * max(np.max(np.abs(e)) for e in E_r)


def test_field_solve_single_mode_closed_form():
    """Independent of the oracle: rho = A cos(k.x)  =>  E = A k/|k|^2 sin(k.x)."""
    _, B = _mods()
    n, h = (64, 32, 16), (1.0, 0.5, 2.0)
    g = B.Grid(3, n, h, 1, "f64")
    idx = np.indices((n[2], n[1], n[0]))
    X = [idx[2 - c].reshape(-1) * h[c] for c in range(3)]
    m = (3, -2, 1)
    k = [2 * np.pi * m[c] / (n[c] * h[c]) for c in range(3)]
    ph = sum(k[c] * X[c] for c in range(3)) + 0.2
    rho = 0.7 * np.cos(ph) - 1.0
    _, E = _solve(B, g, rho, want_phi=False)
    k2 = sum(kc * kc for kc in k)
    for c in range(3):
        assert np.max(np.abs(E[c] - 0.7 * k[c] / k2 * np.sin(ph))) <= 1e-12 * 0.7 / np.sqrt(k2)


def test_field_solve_rejects_what_it_cannot_do():
    _, B = _mods()
    g = B.Grid(2, (8192, 4), (1.0, 1.0), 1, "f64")
    rho = torch.zeros(g.cells, dtype=torch.float64, device="cuda")
    E = [torch.zeros_like(rho), torch.zeros_like(rho)]
    ws = torch.empty(2 * 16 * g.cells + 1024, dtype=torch.uint8, device="cuda")
    for call in (lambda: B.pic_field_solve_bytes(g), lambda: B.pic_step_selfconsistent_bytes(g, 10),
                 lambda: B.pic_field_solve(g, rho, E, None, ws)):
        with pytest.raises(B.PicError, match="unsupported"):
            call()
    # the documented bound is the enforced one: 4096 is taken, 4097 is not (the check comes before any launch)
    B.pic_field_solve_bytes(B.Grid(2, (4096, 4), (1.0, 1.0), 1, "f64"))
    with pytest.raises(B.PicError, match="unsupported"):
        B.pic_field_solve_bytes(B.Grid(2, (4, 4097), (1.0, 1.0), 1, "f64"))
    # the closed loop refuses BEFORE the sort and the deposit: out, perm and rho keep what they held
    gc = B.Grid(2, (8192, 4), (1.0, 1.0), 1, "f64")
    n = 64
    x = [torch.rand(n, dtype=torch.float64, device="cuda") * 4 for _ in range(2)]
    v = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    w = torch.ones(n, dtype=torch.float64, device="cuda")
    xo = [torch.full((n,), -1.0, dtype=torch.float64, device="cuda") for _ in range(2)]
    vo = [torch.full((n,), -1.0, dtype=torch.float64, device="cuda") for _ in range(2)]
    wo = torch.full((n,), -1.0, dtype=torch.float64, device="cuda")
    perm = torch.full((n,), -5, dtype=torch.int32, device="cuda")
    off = torch.zeros(gc.cells + 4, dtype=torch.int32, device="cuda")
    rho_c = torch.full((gc.cells,), -2.0, dtype=torch.float64, device="cuda")
    Ec = [torch.zeros(gc.cells, dtype=torch.float64, device="cuda") for _ in range(2)]
    wsc = torch.empty(B.pic_workspace_bytes(gc, n) + 2 * 16 * gc.cells + 1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.PicError, match="unsupported"):
        B.pic_step_selfconsistent(gc, x, v, w, xo, vo, wo, perm, off, rho_c, Ec, 0.1, 1.0, wsc)
    torch.cuda.synchronize()
    assert torch.all(perm == -5).item() and torch.all(rho_c == -2.0).item() and torch.all(wo == -1.0).item()
    g2 = B.Grid(2, (16, 16), (1.0, 1.0), 1, "f64")
    with pytest.raises(B.PicError, match="workspace"):
        B.pic_field_solve(g2, rho[:256], [E[0][:256], E[1][:256]], None, ws[:64])


CLOSED = [("cfg1", 100_000, dict()), ("cfg2", 200_003, dict(n=(64, 64))), ("cfg3", 150_001, dict(n=(32, 32, 32))),
          ("cfg4", 200_000, dict(n=(32, 32, 32))), ("cfg5", 8 * 16 ** 3 + 5, dict(n=(16, 16, 16))), ("cfg3", 60_000, dict(n=(12, 10, 14), order=2))]


@pytest.mark.parametrize("name,N,kw", CLOSED)
def test_closed_loop_lockstep(name, N, kw):
    """Four steps of the closed loop, each fed the oracle's state: perm / offsets bit-exact; rho, E, x, v within tolerance."""
    O, B = _mods()
    cfg = W.CONFIGS[name].scaled(N, **kw)
    wl = W.make_workload(cfg)
    go, gb = O.grid_of(cfg), B.grid_of(cfg)
    ws = torch.empty(B.pic_step_selfconsistent_bytes(gb, N), dtype=torch.uint8, device="cuda")
    perm = torch.full((max(N, 4),), -1, dtype=torch.int32, device="cuda")
    off = torch.zeros(gb.cells + 4, dtype=torch.int32, device="cuda")
    rho = torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda")
    E = [torch.empty(gb.cells, dtype=gb.torch_dtype, device="cuda") for _ in range(cfg.dim)]
    x, v = wl.x, wl.v
    w = (wl.w * (cfg.cells / N)).astype(wl.w.dtype)                  # mean density 1: fields of order one
    for k in range(4):
        ref = O.step_selfconsistent(go, x, v, w, cfg.dt, cfg.qm)
        xd, vd, wd = to_dev(x), to_dev(v), to_dev([w])[0]
        xo = [torch.empty_like(a) for a in xd]
        vo = [torch.empty_like(a) for a in vd]
        wo = torch.empty_like(wd)
        B.pic_step_selfconsistent(gb, xd, vd, wd, xo, vo, wo, perm, off, rho, E, cfg.dt, cfg.qm, ws)
        torch.cuda.synchronize()
        assert np.array_equal(perm[:N].cpu().numpy(), ref["perm"]), "perm at step %d" % k
        assert np.array_equal(off[: gb.cells + 1].cpu().numpy(), ref["cell_offsets"])
        assert err_rho(rho.cpu().numpy(), ref["rho"]) <= TOL_RHO[cfg.dtype]
        emax = max(np.max(np.abs(e.astype(np.float64))) for e in ref["E"])
        # E inherits the deposit's rounding (rho is stored in the grid dtype before the solve), x and v inherit E's; all
        # stay within the STATED tolerances (achieved on B200, round 3: E 8e-15 / 3.2e-7, x 2.2e-16 / 9.5e-8, v 2e-16 /
        # 1.7e-7 in fp64 / fp32; the bounds were 10 x the tolerances before).  Printed: pytest -s or -rP shows them
        eE = max(np.max(np.abs(E[c].cpu().numpy().astype(np.float64) - ref["E"][c].astype(np.float64))) for c in range(cfg.dim)) / emax
        ex = max(err_x(xo[c].cpu().numpy(), ref["x"][c], cfg.L[c]) for c in range(cfg.dim))
        ev = max(err_v(vo[c].cpu().numpy(), ref["v"][c]) for c in range(cfg.dim))
        print("closed loop %s step %d: achieved E %.3g (bound %.0e), x %.3g, v %.3g (bound %.0e)"
              % (name, k, eE, TOL_RHO[cfg.dtype], ex, ev, TOL_XV[cfg.dtype]))
        assert eE <= TOL_RHO[cfg.dtype]
        assert ex <= TOL_XV[cfg.dtype], "x at step %d" % k
        assert ev <= TOL_XV[cfg.dtype], "v at step %d" % k
        x, v, w = ref["x"], ref["v"], ref["w"]


def test_closed_loop_plasma_oscillation_on_the_gpu():
    """The physics pin of tests/test_oracle_field.py, run free on the GPU: cold lattice + small sine displacement oscillates at
    omega_p [sinc(kh/2)]^(p+1) (independent of the oracle)."""
    _, B = _mods()
    n, ppc, order = (32, 4), 16, 1
    g = B.Grid(2, n, (1.0, 1.0), order, "f64")
    N = n[0] * n[1] * ppc
    ix = (np.arange(N) % (n[0] * 4) + 0.5) / 4.0
    iy = (np.arange(N) // (n[0] * 4) + 0.5) / 4.0
    k = 2 * np.pi / n[0]
    amp, rho0, qm, dt = 1e-3, 0.25, 1.0, 0.2
    x = [np.mod(ix + amp * np.sin(k * ix), n[0]), iy.copy()]
    cur = dict(x=to_dev(x), v=to_dev([np.zeros(N), np.zeros(N)]), w=to_dev([np.full(N, rho0 / ppc)])[0])
    nxt = dict(x=[torch.empty_like(a) for a in cur["x"]], v=[torch.empty_like(a) for a in cur["v"]], w=torch.empty_like(cur["w"]))
    ws = torch.empty(B.pic_step_selfconsistent_bytes(g, N), dtype=torch.uint8, device="cuda")
    perm = torch.empty(N, dtype=torch.int32, device="cuda")
    off = torch.zeros(g.cells + 4, dtype=torch.int32, device="cuda")
    rho = torch.empty(g.cells, dtype=torch.float64, device="cuda")
    E = [torch.empty(g.cells, dtype=torch.float64, device="cuda") for _ in range(2)]
    a = []
    for s in range(64):
        B.pic_step_selfconsistent(g, cur["x"], cur["v"], cur["w"], nxt["x"], nxt["v"], nxt["w"], perm, off, rho, E, dt, qm, ws)
        rr = rho.cpu().numpy().reshape(n[1], n[0]).mean(axis=0)
        a.append(2.0 * np.mean(rr * np.cos(k * np.arange(n[0]))))
        cur, nxt = nxt, cur
    a = np.array(a)
    omega = np.sqrt(qm * rho0) * np.sinc(k / 2 / np.pi) ** (order + 1)
    assert np.max(np.abs(a - a[0] * np.cos(omega * dt * np.arange(64)))) < 0.08 * abs(a[0])
