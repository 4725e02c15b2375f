#!/usr/bin/env python
"""bench.py -- particle-steps/s of the fused hot path (sort + deposit + push) on B200.

Contract (one JSON line on stdout, rank 0):
  python bench.py --gpus N --steps K --warmup W [--config cfg3] [--impl ours|reference]

A "step" is one pass of the whole hot path (pic_step: cell keys, histogram, prefix sum, stable
scatter, reorder, B-spline deposit, gather + accel + push) over all N_p particles of the workload.
Default workload: BASELINE.json configs[2] (3-D 128^3, 1e8 particles, fp32, cubic), the
configuration the metric is quoted on.  The simulation runs continuously from the seeded, unsorted
initial condition: the W warm-up steps include the first (random-order) sort; the K timed steps are
the steady state ("10 steps, sort every step").  The first-step time is reported separately.

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -- "replicas only":
every rank runs an independent replica with its own seed; value = all particle-steps / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "particle-steps/s (sort+deposit+push)"
UNIT = "particle-steps/s"


def algorithmic_bytes(cfg):
    """compulsory bytes per particle-step (integer side arrays are overhead)."""
    d, s = cfg.dim, (8 if cfg.dtype == "f64" else 4)
    A = 2 * d + 1
    return {
        "step": (9 * d + 3) * s,            # sort (d + 2A) + one pass reading A, writing 2d
        "nosort_step": (4 * d + 1) * s,
        "keys": d * s,
        "reorder": 2 * A * s,
        "deposit": (d + 1) * s,
        "push": 4 * d * s,
        "fused": (4 * d + 1) * s,
    }


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_sources_sha256():
    """Hash of the CUDA sources: ties a committed ncu traffic figure to the code it was captured on."""
    import hashlib
    d = os.path.join(ROOT, "paper_1603_02886_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def ncu_traffic(cfg_name, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` capture listed in profiles/ncu_traffic.json -- only if that capture was taken on exactly
    these kernel sources (sha256 recorded beside it); otherwise null, with the reason."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    try:
        rec = json.load(open(p)).get("%s:%s" % (cfg_name, kernel))
    except Exception:
        rec = None
    if not rec:
        return None, "no ncu capture committed for this config and kernel"
    if rec.get("sources_sha256") != kernel_sources_sha256():
        return None, "stale: %s was captured on other kernel sources" % rec.get("source")
    return float(rec["traffic_bytes"]), "%s (same kernel sources, sha256 %s)" % (rec.get("source"), rec["sources_sha256"][:12])


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.index = index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for k, nme in enumerate(names):
                    if r[3 + k].strip().lower() == "active":
                        reasons.add(nme)
            except Exception:
                continue
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


def run_reference(args, cfg_full):
    """--impl reference: the CPU oracle as it stands, on the box's host cores, bounded sample."""
    import oracle as O
    import pic_workloads as W
    sample = min(cfg_full.N, args.ref_particles)
    cfg = cfg_full.scaled(sample)
    wl = W.make_workload(cfg)
    g = O.grid_of(cfg)
    x, v, w = wl.x, wl.v, wl.w
    for _ in range(args.warmup):
        r = O.step(g, x, v, w, wl.E, cfg.dt, cfg.qm)
        x, v, w = r["x"], r["v"], r["w"]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = O.step(g, x, v, w, wl.E, cfg.dt, cfg.qm)
        x, v, w = r["x"], r["v"], r["w"]
    el = time.perf_counter() - t0
    val = sample * args.steps / el
    desc = "first %d particles of %s on the full %s grid, %d steps (sort every step)" % (
        sample, cfg_full.name, "x".join(map(str, cfg.n)), args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype,
            "data": "synthetic", "config": workload_config(cfg_full, args, sample=sample),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(cfg, args, sample=None):
    return {"workload": "%s: %dD periodic %s grid, %.3g particles, %s, B-spline order %d, %s, sort every %d step(s)" % (
                cfg.name, cfg.dim, "x".join(map(str, cfg.n)), cfg.N, cfg.dtype, cfg.order,
                "clustered" if cfg.clustered else "uniform", cfg.sort_every),
            "particles": cfg.N if sample is None else sample, "grid": list(cfg.n), "order": cfg.order,
            "sort_every": cfg.sort_every, "parallelism": "replicas" if args.gpus > 1 else "single",
            "l2": "inputs larger than L2 (no flush needed)" if cfg.N * (2 * cfg.dim + 1) * (8 if cfg.dtype == "f64" else 4) > 256e6
                  else "working set fits L2; rho/ws rewritten between steps",
            "timed": "steady state after warm-up steps that include the first random-order sort"}


def max_over_ranks(value, dist, device):
    """Max of a per-rank scalar over all ranks (the timing rule: max over ranks); identity without dist."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(n_per_rank, world, steps, ms_total_max):
    """Replicas only: every rank advances its own n_per_rank particles; value = all particle-steps / max time."""
    return n_per_rank * world * steps / (ms_total_max * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--repeats", type=int, default=3,
                    help="how many times the warm-up + K-step region is run from the restored initial state; the median region is reported")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--particles", type=int, default=0, help="override N (debug; invalidates the headline)")
    ap.add_argument("--grid", default="", help="override the grid, e.g. 512,256 (the paper's Fig. 9 / Fig. 14 shape; not the headline)")
    ap.add_argument("--sort-every", type=int, default=0)
    ap.add_argument("--ppc", type=int, default=0, help="config 5: particles per cell")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cold", action="store_true")
    ap.add_argument("--bucket", default="", help="cells per bucket, e.g. 2,2,2: the sort steps are pic_step_buckets "
                    "(the paper's bucket-size sweep, PAPER.md:336-350; not the headline)")
    ap.add_argument("--graph", action="store_true",
                    help="replay the steps from CUDA graphs (small, launch-bound problems; no per-phase times)")
    ap.add_argument("--closed-loop", action="store_true",
                    help="the timed step is pic_step_selfconsistent: sort, deposit, Poisson solve, accel, push (not the headline)")
    ap.add_argument("--sort-compare", action="store_true",
                    help="with --bucket: also time pic_sort_buckets (stable, out of place) against pic_sort_buckets_inplace "
                         "(Alg. 2) on the pre-ordered particles of the run")
    ap.add_argument("--deposit-compare", action="store_true",
                    help="also time pic_deposit (sorted / never sorted) and pic_deposit_nodes on this workload")
    ap.add_argument("--ref-particles", type=int, default=2_000_000)
    ap.add_argument("--cpu-particles", type=int, default=30_000_000)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    import pic_workloads as W
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    cfg = W.CONFIGS[args.config]
    if args.config == "cfg5":
        cfg = W.cfg5(args.ppc or 128, args.sort_every or 1)
    if args.grid:
        cfg = cfg.scaled(cfg.N, n=tuple(int(k) for k in args.grid.split(",")))
    if args.particles:
        cfg = cfg.scaled(args.particles)
    if args.sort_every:
        cfg = cfg.scaled(cfg.N, sort_every=args.sort_every)

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    import paper_1603_02886_b200 as B

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg_rank = cfg.scaled(cfg.N, seed=cfg.seed + rank)          # replicas only: independent seeds
    g = B.grid_of(cfg_rank)
    wl = W.make_workload(cfg_rank)
    # load every kernel of this configuration once on a scrap problem of the same shape, so that the first timed
    # step below measures the step and not the lazy loading of the CUDA modules
    tiny = cfg_rank.scaled(min(cfg_rank.N, 50_000))
    wt = W.make_workload(tiny)
    stt = B.Stepper(B.grid_of(tiny), wt.x, wt.v, wt.w, wt.E, device=dev)
    for k in range(2):
        stt.step(tiny.dt, tiny.qm, True)
    stt.step(tiny.dt, tiny.qm, False)
    torch.cuda.synchronize()
    del stt, wt
    bucket = tuple(int(b) for b in args.bucket.split(",")) if args.bucket else None
    if args.closed_loop:       # mean charge density one, so that the self-consistent field is of order one
        wl.w = (wl.w * (cfg.cells / cfg.N)).astype(wl.w.dtype)
    st = B.Stepper(g, wl.x, wl.v, wl.w, wl.E, device=dev, bucket=bucket, closed_loop=args.closed_loop, graph=args.graph)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # SURVEY 8(d) protocol: the warm-up + K-step region is run `repeats` times, each from the restored initial state
    # (Stepper.reset: the seeded particles, no order hint), and the MEDIAN region is the one reported -- ms_per_step x
    # steps is what that one region took; the others are listed in `repeat_ms_per_step`.
    regions = []
    for rep in range(max(1, args.repeats)):
        if rep > 0:
            st.reset(wl.x, wl.v, wl.w)
            torch.cuda.synchronize()
        # ---- warm-up: includes the first, random-order step (timed separately)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        step_no = 0
        first_ms = None
        for k in range(args.warmup):
            e0.record()
            st.step(cfg.dt, cfg.qm, do_sort=(step_no % cfg.sort_every == 0))
            e1.record()
            torch.cuda.synchronize()
            if k == 0:
                first_ms = e0.elapsed_time(e1)
            step_no += 1

        # ---- timed region: exactly K steps, device-timed, with per-phase events
        K = args.steps
        phase_ev = [[torch.cuda.Event(enable_timing=True) for _ in B.PHASES] for _ in range(K)]
        for evs in phase_ev:
            for e in evs:
                e.record()
        launches = 0
        sorts = 0
        sampler = ClockSampler(local_rank)
        barrier()
        sampler.start()
        t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_begin.record()
        for k in range(K):
            do_sort = (step_no % cfg.sort_every == 0)
            if not args.graph:
                B.pic_set_phase_events(phase_ev[k])
            st.step(cfg.dt, cfg.qm, do_sort=do_sort)
            launches += (st.last_launches if (args.graph and do_sort and st.last_launches) else B.pic_last_launch_count())
            sorts += int(do_sort)
            step_no += 1
        t_end.record()
        B.pic_set_phase_events(None)
        barrier()
        clocks = sampler.stop()
        ms_total = t_begin.elapsed_time(t_end)
        ms_total = max_over_ranks(ms_total, dist if world > 1 else None, dev)
        ms_step = ms_total / K
        value = replica_throughput(cfg.N, world, K, ms_total)

        regions.append(dict(ms_total=ms_total, first_ms=first_ms, phase_ev=phase_ev, launches=launches, sorts=sorts,
                            clocks=clocks, step_no=step_no))
    order = sorted(range(len(regions)), key=lambda r: regions[r]["ms_total"])
    med = regions[order[len(order) // 2]]
    repeat_ms = [r["ms_total"] / K for r in regions]
    ms_total, first_ms, phase_ev, launches, sorts, clocks, step_no = (med[k] for k in ("ms_total", "first_ms", "phase_ev", "launches",
                                                                                      "sorts", "clocks", "step_no"))
    ms_step = ms_total / K
    value = replica_throughput(cfg.N, world, K, ms_total)

    # ---- per-phase durations from the events recorded inside the timed region
    phases = {}
    for k in range(K):
        evs, prev = phase_ev[k], phase_ev[k][0]
        for name, e in list(zip(B.PHASES, evs))[1:]:
            try:
                dt_ms = prev.elapsed_time(e)
            except Exception:
                continue
            if dt_ms > 0:
                phases.setdefault(name, []).append(dt_ms)
                prev = e
    phase_ms = {k: sum(v) / len(v) for k, v in phases.items() if v}

    peak, peak_src = measured_peaks()
    ab = algorithmic_bytes(cfg)
    dom = max(phase_ms, key=phase_ms.get) if phase_ms else None
    kernel_bytes = {"keys": ab["keys"], "scan": 0, "radix": 0, "reorder": ab["reorder"], "deposit": ab["deposit"],
                    "push": ab["push"]}
    roofline = None
    if dom:
        bpp = kernel_bytes.get(dom, 0)
        if B.FUSED_PHASE_IS_PUSH and dom == "push":
            bpp = B.fused_kernel_bytes(cfg.dim, 8 if cfg.dtype == "f64" else 4, sorts > 0)
        ach = bpp * cfg.N / (phase_ms[dom] * 1e-3) / 1e9
        traffic, traffic_source = ncu_traffic(cfg.name, dom)
        roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s",
                    "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_source,
                    "peak_source": peak_src, "algorithmic_bytes_per_particle": bpp,
                    "kernel_ms": phase_ms[dom]}
    # second roof of the dominant kernel: plain fp32/fp64 arithmetic.  Algorithmic flops
    # per particle of deposit + gather on the (p+1)^d stencil: products 1, deposit FMA 2, gather FMAs 2d.
    roofline_alu = None
    if dom == "push" and B.FUSED_PHASE_IS_PUSH:
        nodes = (cfg.order + 1) ** cfg.dim
        flop_pp = nodes * (1 + 2 + 2 * cfg.dim)
        sm_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        lanes = 128 if cfg.dtype == "f32" else 64
        peak_tf = 148 * lanes * 2 * sm_mhz * 1e6 / 1e12
        ach_tf = flop_pp * cfg.N / (phase_ms[dom] * 1e-3) / 1e12
        roofline_alu = {"bound": "alu", "kernel": dom, "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                        "frac": ach_tf / peak_tf, "flop_per_particle": flop_pp,
                        "peak_source": "148 SMs x %d lanes x 2 flop x SM clock (DESIGN.md section 6)" % lanes}
    bytes_step = ab["step"] if cfg.sort_every == 1 else (ab["step"] * sorts + ab["nosort_step"] * (K - sorts)) / K
    step_ach = bytes_step * cfg.N / (ms_step * 1e-3) / 1e9

    # ---- the same steady-state steps replayed from CUDA graphs (no host launches inside the timed region)
    graph_line = None
    if not args.graph and cfg.sort_every == 1:
        st.use_graph = True
        for _ in range(4):                                   # captures one graph per ping-pong direction
            st.step(cfg.dt, cfg.qm, do_sort=True)
        barrier()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for _ in range(K):
            st.step(cfg.dt, cfg.qm, do_sort=True)
        g1.record()
        barrier()
        st.use_graph = False
        gms = max_over_ranks(g0.elapsed_time(g1), dist if world > 1 else None, dev)
        graph_line = {"ms_per_step": gms / K, "value": replica_throughput(cfg.N, world, K, gms), "unit": UNIT, "steps": K,
                      "what": "the same steps replayed from two CUDA graphs (Stepper(graph=True)); the headline above is the plain launch path, whose per-phase events it needs"}

    # ---- the configuration as BASELINE.json words it: its own number of steps FROM THE SEEDED, UNSORTED state
    #      (the first step sorts every particle), one timed region, max over ranks
    cold = None
    if not args.no_cold:
        nsteps = cfg.steps
        st.reset(wl.x, wl.v, wl.w)
        barrier()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for k in range(nsteps):
            st.step(cfg.dt, cfg.qm, do_sort=(k % cfg.sort_every == 0))
        c1.record()
        barrier()
        cold_ms = max_over_ranks(c0.elapsed_time(c1), dist if world > 1 else None, dev)
        cold_bytes = ab["step"] if cfg.sort_every == 1 else None
        cold = {"steps": nsteps, "ms_total": cold_ms, "ms_per_step": cold_ms / nsteps,
                "value": replica_throughput(cfg.N, world, nsteps, cold_ms), "unit": UNIT,
                "what": "%d steps from the seeded random order (first step: every particle moves), as the config is stated" % nsteps}
        if cold_bytes:
            cold["frac_of_peak"] = cold_bytes * cfg.N / (cold_ms / nsteps * 1e-3) / 1e9 / peak

    # ---- end to end through the host-buffer entry point (pinned host memory, copies timed)
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(B, torch, cfg_rank, g, wl, dev, K, world, dist if world > 1 else None)

    # ---- the same with the particles resident on the device: per step E goes in, rho comes out
    e2e_resident = None
    if not args.no_e2e:
        e2e_resident = run_e2e_resident(B, torch, cfg_rank, g, wl, st, dev, K, world, dist if world > 1 else None)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # config 5 asks for the deposit with and without sorting (the paper's sorted vs unsorted columns,
    # PAPER.md:392-394): pic_deposit on the current sorted order, and on the never-sorted initial order
    deposit_compare = None
    if (args.config == "cfg5" or args.deposit_compare) and world == 1 and bucket is None:
        deposit_compare = run_deposit_compare(B, torch, cfg, g, wl, st, dev, nodes=args.deposit_compare)

    sort_compare = None
    if args.sort_compare and bucket is not None and world == 1:
        sort_compare = run_sort_compare(B, torch, cfg, g, st, bucket, dev)

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        cpu_baseline = run_cpu_baseline(cfg, args.cpu_particles)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg.dtype, "data": "synthetic", "config": workload_config(cfg, args),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "step_roofline": {"bytes_per_particle_step": bytes_step, "achieved": step_ach, "peak": peak,
                              "frac": step_ach / peak, "frac_of_8TBps_nominal": step_ach / 8000.0, "unit": "GB/s"},
            "phase_ms": phase_ms, "first_step_ms": first_ms, "cold": cold,
            "repeats": len(regions), "repeat_ms_per_step": repeat_ms,
            "repeat_protocol": "warm-up + K steps run %d time(s), each from the restored seeded state; the median region is the one reported" % len(regions)}
    if args.graph:
        line["config"]["cuda_graph"] = "sort steps replayed from CUDA graphs (one per ping-pong direction)"
    if args.closed_loop:
        line["config"]["workload"] += ", closed loop with the periodic Poisson solve (pic_step_selfconsistent)"
        line["config"]["closed_loop"] = True
    if bucket is not None:
        line["config"]["bucket"] = list(bucket)
        line["config"]["workload"] += ", buckets of %s cells (pic_step_buckets)" % "x".join(map(str, bucket))
    if sort_compare:
        line["sort_ms"] = sort_compare
    if graph_line:
        line["cuda_graph"] = graph_line
    if deposit_compare:
        line["deposit_ms"] = deposit_compare
    if e2e_resident:
        line["e2e_resident_particles"] = e2e_resident
    if roofline_alu:
        line["roofline_alu"] = roofline_alu
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_e2e(B, torch, cfg, g, wl, dev, K, world, dist):
    """Same metric through pic_step_host: every step copies the particles host->device from pinned
    memory, runs the step, and reads the advanced particles, perm, cell_offsets and rho back."""
    n, d = cfg.N, cfg.dim
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    A = dict(x=[pin(a) for a in wl.x], v=[pin(a) for a in wl.v], w=pin(wl.w))
    Bf = dict(x=[torch.empty_like(a).pin_memory() for a in A["x"]],
              v=[torch.empty_like(a).pin_memory() for a in A["v"]], w=torch.empty_like(A["w"]).pin_memory())
    E = [pin(a) for a in wl.E]
    perm = torch.empty(max(n, 4), dtype=torch.int32).pin_memory()
    off = torch.empty(g.cells + 1, dtype=torch.int32).pin_memory()
    rho = torch.empty(g.cells, dtype=g.torch_dtype).pin_memory()
    dws = torch.empty(B.pic_step_host_bytes(g, n), dtype=torch.uint8, device=dev)
    s = g.itemsize
    h2d = (2 * d + 1) * s * n + d * s * g.cells
    d2h = (2 * d + 1) * s * n + 4 * n + 4 * (g.cells + 1) + s * g.cells
    steps = max(1, min(K, 5))
    cur, nxt = A, Bf
    for k in range(2 + steps):
        if k == 2:
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
        B.pic_step_host(g, cur["x"], cur["v"], cur["w"], nxt["x"], nxt["v"], nxt["w"], perm, off, rho, E,
                        cfg.dt, cfg.qm, True, dws)
        cur, nxt = nxt, cur
    torch.cuda.synchronize()
    el = time.perf_counter() - t0
    el = max_over_ranks(el, dist, dev)
    return {"value": n * world * steps / el, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "steps": steps, "ms_per_step": 1e3 * el / steps,
            "api": "pic_step_host (pinned host buffers, sort every step)"}


def run_e2e_resident(B, torch, cfg, g, wl, st, dev, K, world, dist):
    """Same metric through pic_step_fields_host: the particles stay on the device (the paper's arrangement,
    PAPER.md:65, 447); every step copies the field E from pinned host memory to the device, runs the step and
    reads rho back.  Wall clock around K synchronous calls."""
    n = cfg.N
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    E = [pin(a) for a in wl.E]
    rho = torch.empty(g.cells, dtype=g.torch_dtype).pin_memory()
    ws = torch.empty(B.pic_step_fields_host_bytes(g, n), dtype=torch.uint8, device=dev)
    a, b = st.cur, st.nxt
    steps = max(1, K)
    for k in range(2 + steps):
        if k == 2:
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
        B.pic_step_fields_host(g, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], st.perm, st.cell_offsets, rho, E,
                               cfg.dt, cfg.qm, True, ws)
        a, b = b, a
    torch.cuda.synchronize()
    el = max_over_ranks(time.perf_counter() - t0, dist, dev)
    st.cur, st.nxt = a, b
    s = g.itemsize
    return {"value": n * world * steps / el, "unit": UNIT, "h2d_bytes_per_step": cfg.dim * s * g.cells,
            "d2h_bytes_per_step": s * g.cells, "steps": steps, "ms_per_step": 1e3 * el / steps,
            "api": "pic_step_fields_host (particles resident on the device; E in, rho out, pinned host buffers)"}


def run_deposit_compare(B, torch, cfg, g, wl, st, dev, reps=5, nodes=False):
    """ms per pic_deposit call: particles sorted by cell (per-cell kernel) against the same workload never
    sorted (threads on particles with global atomics, setrho 3.3.4)."""
    def timed(f):
        f()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    a = st.cur
    xs = [torch.empty_like(t) for t in a["x"]]
    vs = [torch.empty_like(t) for t in a["v"]]
    ws_ = torch.empty_like(a["w"])
    B.pic_sort(g, a["x"], a["v"], a["w"], xs, vs, ws_, st.perm, st.cell_offsets, st.ws)
    t_sorted = timed(lambda: B.pic_deposit(g, xs, ws_, st.rho, B.PIC_ORDER_SORTED, st.cell_offsets, st.ws))
    t_nodes = t_repl = None
    if nodes:      # the collision-free, bitwise reproducible alternative (threads on splines)
        reps, keep = 2, reps
        t_nodes = timed(lambda: B.pic_deposit_nodes(g, xs, ws_, st.rho, st.cell_offsets, st.ws))
        wsr = torch.empty(B.pic_deposit_replicated_bytes(g, cfg.N), dtype=torch.uint8, device=dev)
        t_repl = timed(lambda: B.pic_deposit_replicated(g, xs, ws_, st.rho, st.cell_offsets, wsr))
        del wsr
        reps = keep
    del vs
    x0 = [torch.from_numpy(np.ascontiguousarray(t)).to(dev) for t in wl.x]
    w0 = torch.from_numpy(np.ascontiguousarray(wl.w)).to(dev)
    t_unsorted = timed(lambda: B.pic_deposit(g, x0, w0, st.rho, B.PIC_ORDER_UNSORTED, None, st.ws))
    out = {"sorted": t_sorted, "never_sorted": t_unsorted, "unit": "ms per deposit of all particles"}
    if t_nodes is not None:
        out["nodes_deterministic"] = t_nodes
        out["replicated_deterministic"] = t_repl
    return out


def run_sort_compare(B, torch, cfg, g, st, bucket, dev, reps=3):
    """ms per sort of the run's pre-ordered particles (bucket order of the last step, advanced by one push): the stable
    out-of-place sort with the previous offsets as hint, against Alg. 2 in place (only misplaced particles move)."""
    a = st.cur
    n = cfg.N
    tmp = dict(x=[torch.empty_like(t) for t in a["x"]], v=[torch.empty_like(t) for t in a["v"]], w=torch.empty_like(a["w"]))
    nb = B.pic_bucket_count(g, bucket)
    off = torch.empty(nb + 4, dtype=torch.int32, device=dev)
    moved = torch.zeros(4, dtype=torch.int32, device=dev)
    ws2 = torch.empty(B.pic_sort_buckets_inplace_bytes(g, n), dtype=torch.uint8, device=dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_stable, t_inplace = [], []
    for r in range(reps + 1):
        off[: nb + 1].copy_(st.cell_offsets[: nb + 1])                 # the hint: offsets of the order the particles are in
        e0.record()
        B.pic_sort_buckets(g, bucket, a["x"], a["v"], a["w"], tmp["x"], tmp["v"], tmp["w"], st.perm, off, st.ws)
        e1.record()
        torch.cuda.synchronize()
        if r:
            t_stable.append(e0.elapsed_time(e1))
        for c in range(cfg.dim):
            tmp["x"][c].copy_(a["x"][c]); tmp["v"][c].copy_(a["v"][c])
        tmp["w"].copy_(a["w"])
        e0.record()
        B.pic_sort_buckets_inplace(g, bucket, tmp["x"], tmp["v"], tmp["w"], off, moved, ws2)
        e1.record()
        torch.cuda.synchronize()
        if r:
            t_inplace.append(e0.elapsed_time(e1))
    return {"stable_out_of_place": sum(t_stable) / reps, "alg2_in_place": sum(t_inplace) / reps,
            "misplaced_fraction": int(moved[0].item()) / max(n, 1), "unit": "ms per sort of the pre-ordered particles"}


def run_cpu_baseline(cfg, sample):
    """The oracle as it stands (single thread) on a bounded sample of the same workload, and the OpenMP build of
    the same loops on every host core this process may use (the paper's CPU reference is OpenMP on 8 cores,
    19.24 ns per particle and step).  Two legs each, like the GPU's `cold` and steady-state numbers:
    the first step from the seeded random order (`value`, as before) and a second step on that step's output, i.e. on
    particles that are already sorted (`steady_value`: what the GPU headline is measured on).  The OpenMP figures are
    also flat scalar keys (openmp_value, ...) so that they survive into the driver's record."""
    import oracle as O
    import pic_workloads as W
    sample = min(sample, cfg.N)
    c = cfg.scaled(sample)
    wl = W.make_workload(c)
    g = O.grid_of(c)
    t0 = time.perf_counter()
    r1 = O.step(g, wl.x, wl.v, wl.w, wl.E, c.dt, c.qm)
    el = time.perf_counter() - t0
    t0 = time.perf_counter()
    O.step(g, r1["x"], r1["v"], r1["w"], wl.E, c.dt, c.qm)
    el_s = time.perf_counter() - t0
    what = "first %d particles of %s on the full grid, 1 step (sort+deposit+push) from the seeded random order" % (sample, cfg.name)
    what_s = "the same particles one step later (already sorted, 1 step)"
    out = {"value": sample / el, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": "%s, %.1f s" % (what, el),
           "steady_value": sample / el_s, "steady_sample": "%s, %.1f s" % (what_s, el_s),
           "host_cores_available": len(os.sched_getaffinity(0))}
    del r1
    try:
        threads = len(os.sched_getaffinity(0))
        O.build_openmp()
        O.step_openmp(g, wl.x, wl.v, wl.w, wl.E, c.dt, c.qm, threads)          # thread pool start-up, page faults
        t0 = time.perf_counter()
        r1 = O.step_openmp(g, wl.x, wl.v, wl.w, wl.E, c.dt, c.qm, threads)
        el2 = time.perf_counter() - t0
        steady = []
        for _ in range(2):                                                      # steps 2 and 3: pre-ordered particles
            t0 = time.perf_counter()
            r1 = O.step_openmp(g, r1["x"], r1["v"], r1["w"], wl.E, c.dt, c.qm, threads)
            steady.append(time.perf_counter() - t0)
        el2_s = sum(steady) / len(steady)
        out["openmp"] = {"value": sample / el2, "unit": UNIT, "cores": threads, "kind": "oracle, OpenMP build of the same loops",
                         "ns_per_particle_step": 1e9 * el2 / sample, "sample": "%s, %.1f s" % (what, el2),
                         "steady_value": sample / el2_s, "steady_ns_per_particle_step": 1e9 * el2_s / sample,
                         "steady_sample": "steps 2-3 on the output of the step before (already sorted), %.1f s each" % el2_s,
                         "paper_reference": "19.24 ns per particle and step, OpenMP, 8 cores of a Xeon E5-2670, linear splines, 2-D (PAPER.md:388)"}
        out.update({"openmp_value": sample / el2, "openmp_cores": threads, "openmp_ns_per_particle_step": 1e9 * el2 / sample,
                    "openmp_steady_value": sample / el2_s, "openmp_steady_ns_per_particle_step": 1e9 * el2_s / sample})
    except Exception as e:                                    # no OpenMP runtime on the box
        out["openmp"] = {"unavailable": str(e)[:200]}
    return out


if __name__ == "__main__":
    main()
