"""paper_1603_02886_b200 -- thin Python binding of the C-ABI library declared in include/pic.h.

Argument marshalling only: every step of the hot path (cell keys, histogram, scan, stable
scatter, B-spline deposit, gather + accel + push) runs in the CUDA kernels of csrc/.  PyTorch is
used for device memory and streams, nothing else.  There is NO CPU fallback: if the library
cannot be loaded the import of any entry point raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpic_b200.so")

PIC_F32, PIC_F64 = 0, 1
PIC_OK = 0
PIC_ORDER_UNSORTED, PIC_ORDER_SORTED, PIC_ORDER_STALE = 0, 1, 2
PIC_SORT, PIC_SORT_CHAINED = 1, 3

EXPORTS = ("pic_workspace_bytes", "pic_sort", "pic_deposit", "pic_push", "pic_step",
           "pic_step_host_bytes", "pic_step_host", "pic_step_fields_host_bytes", "pic_step_fields_host",
           "pic_bucket_count", "pic_sort_buckets", "pic_step_buckets", "pic_sort_buckets_inplace_bytes", "pic_sort_buckets_inplace", "pic_deposit_nodes", "pic_deposit_replicated_bytes", "pic_deposit_replicated",
           "pic_deposit_static",
           "pic_field_solve_bytes", "pic_field_solve", "pic_step_selfconsistent_bytes", "pic_step_selfconsistent",
           "pic_last_launch_count", "pic_set_phase_events",
           "pic_strerror")
PHASES = ("begin", "keys", "scan", "radix", "reorder", "deposit", "push")

# True once pic_step runs deposit + gather + push as ONE kernel (recorded as phase "push")
FUSED_PHASE_IS_PUSH = True


def fused_kernel_bytes(dim: int, itemsize: int, with_sort: bool) -> int:
    """Algorithmic bytes per particle of the fused kernel: read x, v, w and write x, v (in place), or,
    with the sort's reorder fused in, read all A = 2d+1 attributes and write all of them to `out`.
    perm (an integer side array) is overhead and is not counted ("Byte model")."""
    a = 2 * dim + 1
    return (2 * a if with_sort else a + 2 * dim) * itemsize


class PicError(RuntimeError):
    pass


class pic_grid_t(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int32), ("n", ctypes.c_int32 * 3), ("h", ctypes.c_double * 3),
                ("order", ctypes.c_int32), ("dtype", ctypes.c_int32)]


class pic_particles_t(ctypes.Structure):
    _fields_ = [("x", ctypes.c_void_p * 3), ("v", ctypes.c_void_p * 3), ("w", ctypes.c_void_p),
                ("n", ctypes.c_int64)]


_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (python -m paper_1603_02886_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PicError("libpic_b200.so is missing: build it with `python -m paper_1603_02886_b200.build` "
                           "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, sz, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.c_double, ctypes.c_int
        G, P = ctypes.POINTER(pic_grid_t), ctypes.POINTER(pic_particles_t)
        E3 = ctypes.POINTER(ctypes.c_void_p)
        L.pic_workspace_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_sort.argtypes = [G, P, P, vp, vp, vp, sz, vp]
        L.pic_deposit.argtypes = [G, P, ci, vp, vp, vp, sz, vp]
        L.pic_push.argtypes = [G, P, ci, vp, E3, dbl, dbl, vp]
        L.pic_step.argtypes = [G, P, P, vp, vp, vp, E3, dbl, dbl, ci, vp, sz, vp]
        L.pic_step_host_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_step_host.argtypes = [G, P, P, vp, vp, vp, E3, dbl, dbl, ci, vp, sz, vp]
        L.pic_step_fields_host_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_step_fields_host.argtypes = [G, P, P, vp, vp, vp, E3, dbl, dbl, ci, vp, sz, vp]
        B3 = ctypes.POINTER(ctypes.c_int32)
        L.pic_bucket_count.argtypes = [G, B3, ctypes.POINTER(i64)]
        L.pic_sort_buckets.argtypes = [G, B3, P, P, vp, vp, vp, sz, vp]
        L.pic_sort_buckets_inplace_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_sort_buckets_inplace.argtypes = [G, B3, P, vp, vp, vp, sz, vp]
        L.pic_step_buckets.argtypes = [G, B3, P, P, vp, vp, vp, E3, dbl, dbl, vp, sz, vp]
        L.pic_deposit_nodes.argtypes = [G, P, vp, vp, vp, sz, vp]
        L.pic_deposit_static.argtypes = [G, P, vp, vp]
        L.pic_deposit_replicated_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_deposit_replicated.argtypes = [G, P, vp, vp, vp, sz, vp]
        L.pic_field_solve_bytes.argtypes = [G, ctypes.POINTER(sz)]
        L.pic_field_solve.argtypes = [G, vp, E3, vp, vp, sz, vp]
        L.pic_step_selfconsistent_bytes.argtypes = [G, i64, ctypes.POINTER(sz)]
        L.pic_step_selfconsistent.argtypes = [G, P, P, vp, vp, vp, E3, dbl, dbl, vp, sz, vp]
        L.pic_last_launch_count.argtypes = []
        L.pic_set_phase_events.argtypes = [ctypes.POINTER(ctypes.c_void_p), ci]
        L.pic_strerror.argtypes = [ci]
        L.pic_strerror.restype = ctypes.c_char_p
        for name in EXPORTS[:-1]:
            getattr(L, name).restype = ci
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != PIC_OK:
        raise PicError("%s failed: %s (%d)" % (what, lib().pic_strerror(rc).decode(), rc))


@dataclass(frozen=True)
class Grid:
    """pic_grid_t: periodic uniform grid, spline order and storage dtype."""
    dim: int
    n: Tuple[int, ...]
    h: Tuple[float, ...]
    order: int
    dtype: str  # "f32" | "f64"

    @property
    def cells(self) -> int:
        c = 1
        for k in self.n[: self.dim]:
            c *= k
        return c

    @property
    def itemsize(self) -> int:
        return 8 if self.dtype == "f64" else 4

    @property
    def torch_dtype(self):
        import torch
        return torch.float64 if self.dtype == "f64" else torch.float32

    def c(self) -> pic_grid_t:
        g = pic_grid_t()
        g.dim = self.dim
        for k in range(3):
            g.n[k] = self.n[k] if k < self.dim else 1
            g.h[k] = self.h[k] if k < self.dim else 1.0
        g.order = self.order
        g.dtype = PIC_F64 if self.dtype == "f64" else PIC_F32
        return g


def grid_of(cfg) -> Grid:
    """Grid of a pic_workloads.Config (duck-typed: dim, n, h, order, dtype)."""
    return Grid(cfg.dim, tuple(cfg.n), tuple([cfg.h] * cfg.dim), cfg.order, cfg.dtype)


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data          # numpy array (host entry point only)


def _particles(g: Grid, x: Sequence, v: Optional[Sequence], w, n: int) -> pic_particles_t:
    p = pic_particles_t()
    for c in range(3):
        p.x[c] = _ptr(x[c]) if c < g.dim else None
        p.v[c] = _ptr(v[c]) if (v is not None and c < g.dim) else None
    p.w = _ptr(w)
    p.n = n
    return p


def _field(g: Grid, E: Sequence):
    a = (ctypes.c_void_p * 3)()
    for c in range(3):
        a[c] = _ptr(E[c]) if c < g.dim else None
    return a


def _stream(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def _dev_check(g: Grid, tensors, n=None):
    import torch
    for t in tensors:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == g.torch_dtype):
            raise PicError("expected contiguous CUDA tensors of dtype %s" % g.dtype)
        if n is not None and t.numel() != n:
            raise PicError("tensor has %d elements, expected %d" % (t.numel(), n))


def pic_workspace_bytes(g: Grid, n: int) -> int:
    out = ctypes.c_size_t(0)
    cg = g.c()
    _check(lib().pic_workspace_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_workspace_bytes")
    return out.value


def pic_step_host_bytes(g: Grid, n: int) -> int:
    out = ctypes.c_size_t(0)
    cg = g.c()
    _check(lib().pic_step_host_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_step_host_bytes")
    return out.value


def pic_last_launch_count() -> int:
    return lib().pic_last_launch_count()


def pic_set_phase_events(events=None):
    """events: sequence of up to 7 torch.cuda.Event(enable_timing=True) (or None to switch off).
    The library records events[k] at the end of phase PHASES[k] of every following call."""
    if not events:
        _check(lib().pic_set_phase_events(None, 0), "pic_set_phase_events")
        return
    arr = (ctypes.c_void_p * len(events))()
    for k, e in enumerate(events):
        if e is not None:
            e.record()                # torch creates the cudaEvent_t lazily, on first record
            arr[k] = e.cuda_event
    _check(lib().pic_set_phase_events(arr, len(events)), "pic_set_phase_events")


def pic_sort(g: Grid, x_in, v_in, w_in, x_out, v_out, w_out, perm, cell_offsets, ws, stream=None):
    """Stable sort by cell key: out_a[j] = in_a[perm[j]]; cell_offsets[C+1].  All CUDA tensors."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_sort(ctypes.byref(cg), ctypes.byref(pi), ctypes.byref(po), _ptr(perm), _ptr(cell_offsets),
                          _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)), "pic_sort")


def _bucket3(g: Grid, bucket):
    b = [int(v) for v in bucket]
    if len(b) != g.dim:
        raise PicError("bucket must have one entry per dimension")
    return (ctypes.c_int32 * 3)(*(b + [1] * (3 - g.dim)))


def pic_bucket_count(g: Grid, bucket) -> int:
    """Number of buckets of bucket[c] cells per dimension on this grid (host computation)."""
    cg, out = g.c(), ctypes.c_int64(0)
    _check(lib().pic_bucket_count(ctypes.byref(cg), _bucket3(g, bucket), ctypes.byref(out)), "pic_bucket_count")
    return int(out.value)


def pic_sort_buckets(g: Grid, bucket, x_in, v_in, w_in, x_out, v_out, w_out, perm, bucket_offsets, ws, stream=None):
    """Stable sort by BUCKET key (boxes of bucket[c] cells): out_a[j] = in_a[perm[j]]; bucket_offsets[B+1]."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_sort_buckets(ctypes.byref(cg), _bucket3(g, bucket), ctypes.byref(pi), ctypes.byref(po), _ptr(perm),
                                  _ptr(bucket_offsets), _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)),
           "pic_sort_buckets")


def pic_sort_buckets_inplace_bytes(g: Grid, n: int) -> int:
    cg, out = g.c(), ctypes.c_size_t(0)
    _check(lib().pic_sort_buckets_inplace_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_sort_buckets_inplace_bytes")
    return int(out.value)


def pic_sort_buckets_inplace(g: Grid, bucket, x, v, w, bucket_offsets, moved, ws, stream=None):
    """Alg. 2: sort x, v, w IN PLACE by bucket key, moving only the misplaced particles; bucket_offsets[B+1] out;
    moved: int32 CUDA tensor of one element (or None)."""
    n = w.numel()
    _dev_check(g, list(x) + list(v) + [w], n)
    cg = g.c()
    p = _particles(g, x, v, w, n)
    _check(lib().pic_sort_buckets_inplace(ctypes.byref(cg), _bucket3(g, bucket), ctypes.byref(p), _ptr(bucket_offsets),
                                          _ptr(moved), _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)),
           "pic_sort_buckets_inplace")


def pic_step_buckets(g: Grid, bucket, x_in, v_in, w_in, x_out, v_out, w_out, perm, bucket_offsets, rho, E, dt: float,
                     qm: float, ws, stream=None):
    """sort by bucket -> deposit at x(t) -> accel -> push; out = particles in bucket order at t+1."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    _dev_check(g, list(E) + [rho], g.cells)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_step_buckets(ctypes.byref(cg), _bucket3(g, bucket), ctypes.byref(pi), ctypes.byref(po), _ptr(perm),
                                  _ptr(bucket_offsets), _ptr(rho), _field(g, E), dt, qm, _ptr(ws),
                                  ws.numel() * ws.element_size(), _stream(stream)), "pic_step_buckets")


def pic_deposit(g: Grid, x, w, rho, order_state=PIC_ORDER_UNSORTED, cell_offsets=None, ws=None, stream=None):
    """rho[C] (overwritten) = h^-d sum_i w_i prod_c W_p(x_ic/h_c - j_c)."""
    n = w.numel()
    _dev_check(g, list(x) + [w], n)
    _dev_check(g, [rho], g.cells)
    cg = g.c()
    p = _particles(g, x, None, w, n)
    wsb = ws.numel() * ws.element_size() if ws is not None else 0
    _check(lib().pic_deposit(ctypes.byref(cg), ctypes.byref(p), order_state, _ptr(cell_offsets), _ptr(rho),
                             _ptr(ws), wsb, _stream(stream)), "pic_deposit")


PIC_DEPOSIT_STATIC_MAX_NODES = 1 << 21


def pic_deposit_static(g: Grid, x, w, rho, stream=None):
    """rho[C] (overwritten) as pic_deposit(..., PIC_ORDER_UNSORTED) computes it, WITHOUT a workspace: for callers that
    may not allocate device memory (a plug-in that is only handed its buffers, code on a latency budget that rules out
    cudaMalloc, a process whose GPU memory is all in pools).  The double-precision sums of the fp32 deposit live in a
    16 MiB array inside the library.  fp32 grids of at most PIC_DEPOSIT_STATIC_MAX_NODES nodes; any particle order.
    Calls share that array: do not let two of them overlap on the GPU.  The first call on a device does a one-time
    address look-up and should be made before any stream capture (see include/pic.h)."""
    n = w.numel()
    _dev_check(g, list(x) + [w], n)
    _dev_check(g, [rho], g.cells)
    cg = g.c()
    p = _particles(g, x, None, w, n)
    _check(lib().pic_deposit_static(ctypes.byref(cg), ctypes.byref(p), _ptr(rho), _stream(stream)), "pic_deposit_static")


def pic_deposit_nodes(g: Grid, x, w, rho, cell_offsets, ws, stream=None):
    """rho[C] by the collision-free threads-on-nodes algorithm: fixed order of additions, bitwise reproducible.
    x, w sorted by cell; cell_offsets from pic_sort."""
    n = w.numel()
    _dev_check(g, list(x) + [w], n)
    _dev_check(g, [rho], g.cells)
    cg = g.c()
    p = _particles(g, x, None, w, n)
    _check(lib().pic_deposit_nodes(ctypes.byref(cg), ctypes.byref(p), _ptr(cell_offsets), _ptr(rho), _ptr(ws),
                                   ws.numel() * ws.element_size(), _stream(stream)), "pic_deposit_nodes")


def pic_deposit_replicated_bytes(g: Grid, n: int) -> int:
    cg, out = g.c(), ctypes.c_size_t(0)
    _check(lib().pic_deposit_replicated_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_deposit_replicated_bytes")
    return int(out.value)


def pic_deposit_replicated(g: Grid, x, w, rho, cell_offsets, ws, stream=None):
    """rho[C] by per-cell local grids and a per-node assembly (setrho 3.3.3): no atomics, bitwise reproducible.
    x, w sorted by cell; cell_offsets from pic_sort; ws of pic_deposit_replicated_bytes()."""
    n = w.numel()
    _dev_check(g, list(x) + [w], n)
    _dev_check(g, [rho], g.cells)
    cg = g.c()
    p = _particles(g, x, None, w, n)
    _check(lib().pic_deposit_replicated(ctypes.byref(cg), ctypes.byref(p), _ptr(cell_offsets), _ptr(rho), _ptr(ws),
                                        ws.numel() * ws.element_size(), _stream(stream)), "pic_deposit_replicated")


def pic_field_solve_bytes(g: Grid) -> int:
    cg, out = g.c(), ctypes.c_size_t(0)
    _check(lib().pic_field_solve_bytes(ctypes.byref(cg), ctypes.byref(out)), "pic_field_solve_bytes")
    return int(out.value)


def pic_field_solve(g: Grid, rho, E, phi, ws, stream=None):
    """Periodic Poisson solve: rho[C] -> E[c][C] (and phi[C] unless None); -Laplace(phi) = rho - mean, E = -grad(phi)."""
    _dev_check(g, [rho] + list(E) + ([phi] if phi is not None else []), g.cells)
    cg = g.c()
    _check(lib().pic_field_solve(ctypes.byref(cg), _ptr(rho), _field(g, E), _ptr(phi), _ptr(ws),
                                 ws.numel() * ws.element_size(), _stream(stream)), "pic_field_solve")


def pic_step_selfconsistent_bytes(g: Grid, n: int) -> int:
    cg, out = g.c(), ctypes.c_size_t(0)
    _check(lib().pic_step_selfconsistent_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_step_selfconsistent_bytes")
    return int(out.value)


def pic_step_selfconsistent(g: Grid, x_in, v_in, w_in, x_out, v_out, w_out, perm, cell_offsets, rho, E, dt: float,
                            qm: float, ws, stream=None):
    """One step of the closed loop: sort -> deposit -> field solve (E is WRITTEN) -> accel -> push."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    _dev_check(g, list(E) + [rho], g.cells)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_step_selfconsistent(ctypes.byref(cg), ctypes.byref(pi), ctypes.byref(po), _ptr(perm),
                                         _ptr(cell_offsets), _ptr(rho), _field(g, E), dt, qm, _ptr(ws),
                                         ws.numel() * ws.element_size(), _stream(stream)), "pic_step_selfconsistent")


def pic_push(g: Grid, x, v, E, dt: float, qm: float, order_state=PIC_ORDER_UNSORTED, cell_offsets=None,
             stream=None):
    """In place: v += qm*dt*E(x); x += dt*v; periodic wrap."""
    n = x[0].numel()
    _dev_check(g, list(x) + list(v), n)
    _dev_check(g, list(E), g.cells)
    cg = g.c()
    p = _particles(g, x, v, None, n)
    _check(lib().pic_push(ctypes.byref(cg), ctypes.byref(p), order_state, _ptr(cell_offsets), _field(g, E),
                          dt, qm, _stream(stream)), "pic_push")


def pic_step(g: Grid, x_in, v_in, w_in, x_out, v_out, w_out, perm, cell_offsets, rho, E, dt: float, qm: float,
             do_sort=True, ws=None, stream=None):
    """sort (if do_sort) -> deposit at x(t) -> accel -> push.  out = particles in sorted order at t+1.
    do_sort: False / 0, True / PIC_SORT, or PIC_SORT_CHAINED (in = unmodified out of the previous step, see pic.h)."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    _dev_check(g, list(E) + [rho], g.cells)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    wsb = ws.numel() * ws.element_size() if ws is not None else 0
    _check(lib().pic_step(ctypes.byref(cg), ctypes.byref(pi), ctypes.byref(po), _ptr(perm), _ptr(cell_offsets),
                          _ptr(rho), _field(g, E), dt, qm, int(do_sort), _ptr(ws), wsb, _stream(stream)),
           "pic_step")


def pic_step_host(g: Grid, x_in, v_in, w_in, x_out, v_out, w_out, perm, cell_offsets, rho, E, dt: float,
                  qm: float, do_sort: bool, dev_ws, stream=None):
    """pic_step on HOST buffers (numpy arrays or pinned CPU tensors); copies in, runs, copies out, syncs."""
    n = w_in.numel() if hasattr(w_in, "numel") else w_in.size
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_step_host(ctypes.byref(cg), ctypes.byref(pi), ctypes.byref(po), _ptr(perm), _ptr(cell_offsets),
                               _ptr(rho), _field(g, E), dt, qm, 1 if do_sort else 0, _ptr(dev_ws),
                               dev_ws.numel() * dev_ws.element_size(), _stream(stream)), "pic_step_host")


def pic_step_fields_host_bytes(g: Grid, n: int) -> int:
    out = ctypes.c_size_t(0)
    cg = g.c()
    _check(lib().pic_step_fields_host_bytes(ctypes.byref(cg), n, ctypes.byref(out)), "pic_step_fields_host_bytes")
    return out.value


def pic_step_fields_host(g: Grid, x_in, v_in, w_in, x_out, v_out, w_out, perm, cell_offsets, rho_host, E_host,
                         dt: float, qm: float, do_sort: bool, ws, stream=None):
    """pic_step with the particles on the device (CUDA tensors) and E, rho on the host (numpy / pinned tensors)."""
    n = w_in.numel()
    _dev_check(g, list(x_in) + list(v_in) + [w_in] + list(x_out) + list(v_out) + [w_out], n)
    cg = g.c()
    pi, po = _particles(g, x_in, v_in, w_in, n), _particles(g, x_out, v_out, w_out, n)
    _check(lib().pic_step_fields_host(ctypes.byref(cg), ctypes.byref(pi), ctypes.byref(po), _ptr(perm),
                                      _ptr(cell_offsets), _ptr(rho_host), _field(g, E_host), dt, qm,
                                      1 if do_sort else 0, _ptr(ws), ws.numel() * ws.element_size(), _stream(stream)),
           "pic_step_fields_host")


class Stepper:
    """Device-resident particle state with ping-pong buffers: the usual way to run many steps."""

    def __init__(self, g: Grid, x, v, w, E, device="cuda", bucket=None, closed_loop=False, graph=False):
        """bucket: cells per bucket and dimension -> the sort steps are pic_step_buckets (cell_offsets then holds the
        BUCKET offsets); None: pic_step.  closed_loop: the sort steps are pic_step_selfconsistent (E is recomputed from
        rho every step; the E given here only sizes the arrays).  graph: the sort steps are replayed from CUDA graphs
        (one per direction of the ping-pong), which takes the 20-odd launches of a step off the host: for problems so
        small that the step is launch bound.  Every choice inside a step (first or pre-ordered sort, chained or not)
        is made on the device, so one captured step serves all of them."""
        import torch
        self.g, self.n = g, int(w.shape[0])
        self.bucket = None if bucket is None else tuple(int(b) for b in bucket)
        dev = torch.device(device)
        up = lambda a: torch.as_tensor(a).to(dev).contiguous()
        self.cur = dict(x=[up(a) for a in x], v=[up(a) for a in v], w=up(w))
        self.nxt = dict(x=[torch.empty_like(a) for a in self.cur["x"]],
                        v=[torch.empty_like(a) for a in self.cur["v"]], w=torch.empty_like(self.cur["w"]))
        self.E = [up(a) for a in E]
        self.perm = torch.empty(max(self.n, 4), dtype=torch.int32, device=dev)
        self.cell_offsets = torch.zeros(g.cells + 4, dtype=torch.int32, device=dev)
        self.rho = torch.empty(g.cells, dtype=g.torch_dtype, device=dev)
        self.closed_loop = bool(closed_loop)
        self.use_graph = bool(graph)
        self._graphs = {}
        self.last_launches = 0
        nbytes = pic_step_selfconsistent_bytes(g, self.n) if self.closed_loop else pic_workspace_bytes(g, self.n)
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        self.sorted_once = False
        self._chain_ok = False

    def reset(self, x, v, w):
        """Start again from host arrays x, v, w (as if no step had been taken: no order hint)."""
        import torch
        for c in range(self.g.dim):
            self.cur["x"][c].copy_(torch.as_tensor(x[c]))
            self.cur["v"][c].copy_(torch.as_tensor(v[c]))
        self.cur["w"].copy_(torch.as_tensor(w))
        self.cell_offsets.zero_()
        self.sorted_once = False
        self._chain_ok = False       # the arrays were written from outside: the next sort reads the positions

    def step(self, dt: float, qm: float, do_sort: bool = True, stream=None, chained: bool = True):
        """One pic_step on the resident particles.  chained: sort steps are PIC_SORT_CHAINED -- this object owns the
        particle arrays and nothing else writes them between steps, which is what that flag states (the library
        checks the rest, so the first step and a step after reset() or an unsorted step fall back by themselves)."""
        a, b = self.cur, self.nxt
        if do_sort and self.use_graph and stream is None:
            self._graph_step(dt, qm, chained)
            return
        self._enqueue(a, b, dt, qm, do_sort, stream, chained)

    def _graph_step(self, dt, qm, chained):
        """replay (capture on first use) the sort step from the current buffers into the other set"""
        import torch
        a, b = self.cur, self.nxt
        self.last_launches = 0
        if not self.sorted_once:                # the first step runs as it is (it also loads the kernels)
            self._enqueue(a, b, dt, qm, True, None, chained)
            return
        key = (a["w"].data_ptr(), float(dt), float(qm), bool(chained and self._chain_ok))
        if key not in self._graphs:
            gr = torch.cuda.CUDAGraph()
            state = (self.cur, self.nxt, self._chain_ok, self.sorted_once)
            torch.cuda.synchronize()
            with torch.cuda.graph(gr):
                self._enqueue(a, b, dt, qm, True, None, chained)
            self.cur, self.nxt, self._chain_ok, self.sorted_once = state      # capturing runs nothing
            self._graphs[key] = (gr, pic_last_launch_count())
        gr, self.last_launches = self._graphs[key]
        gr.replay()
        self.cur, self.nxt = b, a
        self._chain_ok = not (self.closed_loop or self.bucket is not None)

    def _enqueue(self, a, b, dt, qm, do_sort, stream, chained):
        if do_sort and self.closed_loop:
            pic_step_selfconsistent(self.g, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], self.perm, self.cell_offsets,
                                    self.rho, self.E, dt, qm, self.ws, stream)
            self.cur, self.nxt = b, a
            self.sorted_once = True
        elif do_sort and self.bucket is not None:
            pic_step_buckets(self.g, self.bucket, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], self.perm,
                             self.cell_offsets, self.rho, self.E, dt, qm, self.ws, stream)
            self.cur, self.nxt = b, a
            self.sorted_once = True
        elif do_sort:
            pic_step(self.g, a["x"], a["v"], a["w"], b["x"], b["v"], b["w"], self.perm, self.cell_offsets,
                     self.rho, self.E, dt, qm, PIC_SORT_CHAINED if (chained and self._chain_ok) else PIC_SORT,
                     self.ws, stream)
            self._chain_ok = True
            self.cur, self.nxt = b, a
            self.sorted_once = True
        else:   # in place, current order
            pic_step(self.g, a["x"], a["v"], a["w"], a["x"], a["v"], a["w"], None,
                     self.cell_offsets if self.sorted_once else None, self.rho, self.E, dt, qm, False, self.ws,
                     stream)
