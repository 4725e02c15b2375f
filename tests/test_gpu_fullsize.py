"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (cfg3: 3-D 128^3,
1e8 particles, fp32, cubic, Stepper with ping-pong buffers, sort every step).

The oracle cannot run 1e8 particles in seconds, so this checks (i) what is unique and cheap to verify
exactly at any size -- perm is a bijection, the keys of the reordered input are non-decreasing, perm is
increasing inside every cell (stability), cell_offsets is the exclusive scan of the key histogram --
(ii) exact invariants -- charge conservation -- and (iii) sampled outputs the oracle computes one by
one: the push of sampled particles, and rho on the nodes of a sub-box from the particles of the cells
around it (the only particles whose stencils reach those nodes).
"""
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


@pytest.mark.timeout(1200)
def test_cfg3_full_size_two_steps():
    import oracle as O
    import paper_1603_02886_b200 as B

    cfg = W.CONFIGS["cfg3"]
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
        assert abs(tot_rho - tot_w) <= 1e-6 * tot_w

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

        # (iii-b) rho on the nodes of a sub-box, from the particles of the cells around it
        lo, size, halo = (5 + 40 * step, 60, 125), 6, 3      # crosses nothing / the periodic seam in z
        cells = []
        for kz in range(lo[2] - halo, lo[2] + size + halo):
            for ky in range(lo[1] - halo, lo[1] + size + halo):
                base = (ky % cfg.n[1]) * cfg.n[0] + (kz % cfg.n[2]) * cfg.n[0] * cfg.n[1]
                for kx in range(lo[0] - halo, lo[0] + size + halo):
                    cells.append(base + kx % cfg.n[0])
        cells = torch.tensor(sorted(set(cells)), device="cuda")
        a, b = off[cells], off[cells + 1]
        idx = torch.cat([perm[int(s):int(e)] for s, e in zip(a.tolist(), b.tolist())])
        xs = [before["x"][c][idx].cpu().numpy() for c in range(d)]
        ws = before["w"][idx].cpu().numpy()
        rho_ref = O.deposit(go, xs, ws).reshape(cfg.n[2], cfg.n[1], cfg.n[0])
        rho_gpu = st.rho.cpu().numpy().astype(np.float64).reshape(cfg.n[2], cfg.n[1], cfg.n[0])
        zz = [(lo[2] + k) % cfg.n[2] for k in range(size)]
        sub_ref = rho_ref[zz][:, lo[1]:lo[1] + size, lo[0]:lo[0] + size]
        sub_gpu = rho_gpu[zz][:, lo[1]:lo[1] + size, lo[0]:lo[0] + size]
        assert np.max(np.abs(sub_gpu - sub_ref)) <= TOL_RHO[cfg.dtype] * np.max(np.abs(rho_gpu))
        del before
