"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (Stepper with
ping-pong buffers, sort every step): cfg2, cfg3 (the headline), cfg4 (clustered) and cfg5 at 128 ppc.

test_full_size_elementwise runs the WHOLE oracle step on cfg3 and cfg4 (about 45 s of one host core per
step) and compares every output element: perm, cell_offsets, every node of rho, every x, v, w.  The other
tests check (i) what is unique and cheap to verify exactly at any size -- perm is a bijection, the keys
of the reordered input are non-decreasing, perm is increasing inside every cell (stability),
cell_offsets is the exclusive scan of the key histogram -- (ii) exact invariants -- charge conservation
-- and (iii) sampled outputs the oracle computes one by one: the push of sampled particles, and rho on
the nodes of a sub-box from the particles of the cells around it.
"""
import gc

import numpy as np
import pytest

import pic_workloads as W
from parity import TOL_RHO, TOL_XV, err_v, err_x

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _keys_torch(x, n):
    # h = 1: floor(x) clamped, x fastest.  (A test-side restatement for the property checks only.)
    k = None
    mul = 1
    for c in range(len(x)):
        cc = torch.clamp(torch.floor(x[c]).to(torch.int64), 0, n[c] - 1)
        k = cc * mul if k is None else k + cc * mul
        mul *= n[c]
    return k


def _full_cfg(name):
    return W.cfg5(128, 1) if name == "cfg5" else W.CONFIGS[name]


@pytest.mark.timeout(1800)
@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_size_elementwise(name):
    """One full oracle step against pic_step at full size, EVERY element (north_star: "on all five configs"; cfg1
    runs at full size in test_gpu_parity, cfg2 and cfg5 element-wise below).  Step 1 starts from the seeded random
    order (every particle moves: the reorder-first arm); step 2 starts from the GPU's own output of step 1, so it
    exercises the incremental sort and the one-pass kernel, and is compared with the oracle's step from that same
    state.  cfg4: the comparison includes the peak cell of the blob (about 7e4 particles on one stencil)."""
    import oracle as O
    import paper_1603_02886_b200 as B

    cfg = W.CONFIGS[name]
    n, d = cfg.N, cfg.dim
    wl = W.make_workload(cfg)
    g, go = B.grid_of(cfg), O.grid_of(cfg)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, device="cuda:0")
    x, v, w = wl.x, wl.v, wl.w
    for step in range(2):
        ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        st.step(cfg.dt, cfg.qm, True)
        torch.cuda.synchronize()
        assert np.array_equal(st.perm[:n].cpu().numpy(), ref["perm"]), "perm, step %d" % step
        assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), ref["cell_offsets"]), "cell_offsets, step %d" % step
        counts = np.diff(ref["cell_offsets"])
        if cfg.clustered:
            assert counts.max() > 5e4                  # the peak cell is part of the comparison
        rho = st.rho.cpu().numpy().astype(np.float64)
        assert np.max(np.abs(rho - ref["rho"])) <= TOL_RHO[cfg.dtype] * np.max(np.abs(ref["rho"])), "rho, step %d" % step
        out = dict(x=[a.cpu().numpy() for a in st.cur["x"]], v=[a.cpu().numpy() for a in st.cur["v"]], w=st.cur["w"].cpu().numpy())
        for c in range(d):
            assert err_x(out["x"][c], ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype], "x[%d], step %d" % (c, step)
            assert err_v(out["v"][c], ref["v"][c]) <= TOL_XV[cfg.dtype], "v[%d], step %d" % (c, step)
        assert np.array_equal(out["w"], ref["w"]), "w, step %d" % step
        del ref, rho
        x, v, w = out["x"], out["v"], out["w"]        # the next oracle step starts from the GPU's state
    del st
    gc.collect()
    torch.cuda.empty_cache()


@pytest.mark.timeout(1200)
@pytest.mark.parametrize("name", ["cfg2", "cfg5_8", "cfg5_512"])
def test_full_size_elementwise_fp64(name):
    """The fp64 configs at full size, every element, one step from the seeded order and one from the GPU's state:
    cfg2 (1e7 particles) and cfg5 at 8 particles per cell (2.1e6); cfg5 at 512 per cell (1.34e8 particles, the largest
    configuration of BASELINE.json; sort every step) for ONE step from the seeded order -- the oracle needs about a
    minute for it."""
    import oracle as O
    import paper_1603_02886_b200 as B

    cfg = W.cfg5(512, 1) if name == "cfg5_512" else (W.cfg5(8, 1) if name == "cfg5_8" else W.CONFIGS[name])
    n, d = cfg.N, cfg.dim
    wl = W.make_workload(cfg)
    g, go = B.grid_of(cfg), O.grid_of(cfg)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, device="cuda:0")
    x, v, w = wl.x, wl.v, wl.w
    for step in range(1 if name == "cfg5_512" else 2):
        ref = O.step(go, x, v, w, wl.E, cfg.dt, cfg.qm)
        st.step(cfg.dt, cfg.qm, True)
        torch.cuda.synchronize()
        assert np.array_equal(st.perm[:n].cpu().numpy(), ref["perm"])
        assert np.array_equal(st.cell_offsets[: g.cells + 1].cpu().numpy(), ref["cell_offsets"])
        rho = st.rho.cpu().numpy().astype(np.float64)
        assert np.max(np.abs(rho - ref["rho"])) <= TOL_RHO[cfg.dtype] * np.max(np.abs(ref["rho"]))
        out = dict(x=[a.cpu().numpy() for a in st.cur["x"]], v=[a.cpu().numpy() for a in st.cur["v"]], w=st.cur["w"].cpu().numpy())
        for c in range(d):
            assert err_x(out["x"][c], ref["x"][c], cfg.L[c]) <= TOL_XV[cfg.dtype]
            assert err_v(out["v"][c], ref["v"][c]) <= TOL_XV[cfg.dtype]
        assert np.array_equal(out["w"], ref["w"])
        x, v, w = out["x"], out["v"], out["w"]
        del ref, rho
    del st, wl, out, x, v, w
    gc.collect()
    torch.cuda.empty_cache()


@pytest.mark.timeout(1200)
@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_full_size_two_steps(name):
    import oracle as O
    import paper_1603_02886_b200 as B

    cfg = _full_cfg(name)
    n, d = cfg.N, cfg.dim
    wl = W.make_workload(cfg)
    g, go = B.grid_of(cfg), O.grid_of(cfg)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, device="cuda:0")
    rng = np.random.default_rng(7)

    for step in range(2):                       # step 0: random order; step 1: the incremental (movers-only) sort
        before = dict(x=[a.clone() for a in st.cur["x"]], v=[a.clone() for a in st.cur["v"]], w=st.cur["w"].clone())
        st.step(cfg.dt, cfg.qm, True)
        torch.cuda.synchronize()
        perm = st.perm[:n].to(torch.int64)
        off = st.cell_offsets[: g.cells + 1].to(torch.int64)

        # (i) sort post-conditions, exact
        seen = torch.zeros(n, dtype=torch.uint8, device="cuda")
        seen[perm] = 1
        assert int(seen.sum()) == n, "perm is not a bijection"
        del seen
        keys_in = _keys_torch(before["x"], cfg.n)
        skey = keys_in[perm]
        assert bool((skey[1:] >= skey[:-1]).all()), "keys of the reordered input are not sorted"
        same = skey[1:] == skey[:-1]
        assert bool((perm[1:][same] > perm[:-1][same]).all()), "sort is not stable"
        cnt = torch.bincount(keys_in, minlength=g.cells)
        ref_off = torch.zeros(g.cells + 1, dtype=torch.int64, device="cuda")
        ref_off[1:] = torch.cumsum(cnt, 0)
        assert torch.equal(off, ref_off), "cell_offsets is not the scan of the histogram"
        del keys_in, skey, same, cnt, ref_off

        # (ii) charge conservation: sum rho h^d = sum w (fp32 rho rounded once per node)
        tot_w = float(before["w"].double().sum())
        tot_rho = float(st.rho.double().sum())
        assert abs(tot_rho - tot_w) <= (1e-6 if cfg.dtype == "f32" else 1e-12) * tot_w

        # (iii-a) sampled particles: slot j of the output = pushed particle perm[j] of the input
        js = torch.from_numpy(rng.choice(n, 4096, replace=False)).cuda()
        src = perm[js]
        xs = [before["x"][c][src].cpu().numpy() for c in range(d)]
        vs = [before["v"][c][src].cpu().numpy() for c in range(d)]
        ref = O.push(go, xs, vs, wl.E, cfg.dt, cfg.qm)
        rx, rv = (ref["x"], ref["v"]) if isinstance(ref, dict) else ref
        for c in range(d):
            assert err_x(st.cur["x"][c][js].cpu().numpy(), rx[c], cfg.L[c]) <= TOL_XV[cfg.dtype]
            assert err_v(st.cur["v"][c][js].cpu().numpy(), rv[c]) <= TOL_XV[cfg.dtype]
        assert torch.equal(st.cur["w"][js], before["w"][src])

        # (iii-b) rho on the nodes of a sub-box, from the particles of the cells around it (the box
        #          crosses the periodic seam in the last dimension; cfg4: it sits inside the dense blob)
        size, halo = 6, 3
        nn = list(cfg.n) + [1] * (3 - d)
        lo = [5 + 40 * step if nn[0] > 64 else 5 + 20 * step, nn[1] // 2 - 3, nn[2] - 3 if d == 3 else 0]
        if d == 2:
            lo[1] = nn[1] - 3
        if cfg.clustered:                        # 1.5 sigma off the blob centre: a few thousand particles per cell
            lo = [70, 70, 70 - 6 * step]
        rng_z = range(lo[2] - halo, lo[2] + size + halo) if d == 3 else [0]
        cells = []
        for kz in rng_z:
            for ky in range(lo[1] - halo, lo[1] + size + halo):
                base = (ky % nn[1]) * nn[0] + (kz % nn[2]) * nn[0] * nn[1]
                for kx in range(lo[0] - halo, lo[0] + size + halo):
                    cells.append(base + kx % nn[0])
        cells = torch.tensor(sorted(set(cells)), device="cuda")
        a, b = off[cells], off[cells + 1]
        idx = torch.cat([perm[int(s):int(e)] for s, e in zip(a.tolist(), b.tolist())])
        xs = [before["x"][c][idx].cpu().numpy() for c in range(d)]
        ws = before["w"][idx].cpu().numpy()
        rho_ref = O.deposit(go, xs, ws).reshape(nn[2], nn[1], nn[0])
        rho_gpu = st.rho.cpu().numpy().astype(np.float64).reshape(nn[2], nn[1], nn[0])
        zz = [(lo[2] + k) % nn[2] for k in range(size if d == 3 else 1)]
        yy = [(lo[1] + k) % nn[1] for k in range(size)]
        sub_ref = rho_ref[zz][:, yy][:, :, lo[0]:lo[0] + size]
        sub_gpu = rho_gpu[zz][:, yy][:, :, lo[0]:lo[0] + size]
        assert np.max(np.abs(sub_gpu - sub_ref)) <= TOL_RHO[cfg.dtype] * np.max(np.abs(rho_gpu))
        del before


@pytest.mark.timeout(1800)
@pytest.mark.parametrize("ppc", [8, 32, 128, 512])
@pytest.mark.parametrize("k", [1, 4, 16])
def test_cfg5_sweep_17_steps(ppc, k):
    """Config 5 at full size: ppc in {8, 32, 128, 512} x sort every k in {1, 4, 16} steps, 17 steps (one
    re-sort at k = 16 is crossed).  Every step: exact charge conservation of rho; on sort steps the sort
    post-conditions; on the last two steps (one of them a step without sort for k > 1) sampled particles
    against the oracle's push."""
    import oracle as O
    import paper_1603_02886_b200 as B

    cfg = W.cfg5(ppc, k)
    n, d = cfg.N, cfg.dim
    wl = W.make_workload(cfg)
    g, go = B.grid_of(cfg), O.grid_of(cfg)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, device="cuda:0")
    tot_w = float(st.cur["w"].double().sum())
    rng = np.random.default_rng(11)
    for step in range(17):
        do_sort = step % k == 0
        check = step >= 15
        if check:
            js = torch.from_numpy(rng.choice(n, 2048, replace=False)).cuda()
            if do_sort:
                x_in = [a.clone() for a in st.cur["x"]]
                v_in = [a.clone() for a in st.cur["v"]]
            else:
                x_in = [a[js].clone() for a in st.cur["x"]]
                v_in = [a[js].clone() for a in st.cur["v"]]
        st.step(cfg.dt, cfg.qm, do_sort)
        torch.cuda.synchronize()
        assert abs(float(st.rho.double().sum()) - tot_w) <= 1e-12 * tot_w, "charge not conserved at step %d" % step
        if do_sort and (step == 0 or check):
            perm = st.perm[:n].to(torch.int64)
            seen = torch.zeros(n, dtype=torch.uint8, device="cuda")
            seen[perm] = 1
            assert int(seen.sum()) == n
            off = st.cell_offsets[: g.cells + 1].to(torch.int64)
            assert int(off[0]) == 0 and int(off[-1]) == n and bool((off[1:] >= off[:-1]).all())
        if check:
            if do_sort:
                src = st.perm[:n].to(torch.int64)[js]
                xs = [a[src].cpu().numpy() for a in x_in]
                vs = [a[src].cpu().numpy() for a in v_in]
            else:
                xs = [a.cpu().numpy() for a in x_in]
                vs = [a.cpu().numpy() for a in v_in]
            rx, rv = O.push(go, xs, vs, wl.E, cfg.dt, cfg.qm)
            for c in range(d):
                assert err_x(st.cur["x"][c][js].cpu().numpy(), rx[c], cfg.L[c]) <= TOL_XV[cfg.dtype]
                assert err_v(st.cur["v"][c][js].cpu().numpy(), rv[c]) <= TOL_XV[cfg.dtype]


@pytest.mark.timeout(1800)
def test_maximum_particle_count():
    """N = 2^30 - 1, the largest count the C ABI accepts (32-bit indices): fp32, 3-D 256^3, linear splines, inputs
    drawn on the device (test-only: no oracle value is involved).  Two steps -- all particles movers, then the
    incremental sort -- checked by what is exact at any size: perm is a bijection, cell_offsets is the scan of the
    key histogram, keys of the reordered input are sorted, charge is conserved."""
    import paper_1603_02886_b200 as B

    gc.collect()
    torch.cuda.empty_cache()                    # blocks cached by the tests before this one count as used memory
    free, total = torch.cuda.mem_get_info()
    if total < 150e9:
        pytest.skip("needs a device with about 130 GB of memory")
    assert free > 135e9, "device memory is held by something else: %.0f GB free" % (free / 1e9)
    n = (1 << 30) - 1
    g = B.Grid(3, (256, 256, 256), (1.0, 1.0, 1.0), 1, "f32")
    gen = torch.Generator(device="cuda").manual_seed(1)
    mk = lambda scale: torch.rand(n, device="cuda", generator=gen, dtype=torch.float32) * scale
    a = dict(x=[mk(256.0).clamp_(max=255.99998) for _ in range(3)],
             v=[torch.randn(n, device="cuda", generator=gen, dtype=torch.float32) for _ in range(3)], w=mk(1.0) + 0.5)
    b = dict(x=[torch.empty_like(t) for t in a["x"]], v=[torch.empty_like(t) for t in a["v"]], w=torch.empty_like(a["w"]))
    E = [torch.randn(g.cells, device="cuda", generator=gen, dtype=torch.float32) * 0.1 for _ in range(3)]
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    off = torch.zeros(g.cells + 4, dtype=torch.int32, device="cuda")
    rho = torch.empty(g.cells, dtype=torch.float32, device="cuda")
    ws = torch.empty(B.pic_workspace_bytes(g, n), dtype=torch.uint8, device="cuda")
    for step in range(2):
        keys = None
        for c, m in zip(range(3), (1, 256, 65536)):
            kc = torch.floor(a["x"][c]).to(torch.int32).clamp_(0, 255) * m
            keys = kc if keys is None else keys.add_(kc)
            del kc
        tot_w = float(a["w"].sum(dtype=torch.float64))
        B.pic_step(g, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], perm, off, rho, E, 0.1, 1.0, True, ws)
        torch.cuda.synchronize()
        cnt = torch.bincount(keys, minlength=g.cells)
        assert torch.equal(off[1: g.cells + 1].to(torch.int64), torch.cumsum(cnt, 0)) and int(off[0]) == 0
        del cnt
        seen = torch.zeros(n, dtype=torch.uint8, device="cuda")
        seen[perm.to(torch.int64)] = 1
        assert int(seen.sum(dtype=torch.int64)) == n, "perm is not a bijection"
        del seen
        skey = keys[perm.to(torch.int64)]
        del keys
        assert bool((skey[1:] >= skey[:-1]).all())
        del skey
        assert abs(float(rho.sum(dtype=torch.float64)) - tot_w) <= 2e-6 * tot_w
        for c in range(3):
            assert float(b["x"][c].min()) >= 0.0 and float(b["x"][c].max()) < 256.0
        a, b = b, a
