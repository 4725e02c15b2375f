"""numpy front end of the CPU oracle (oracle/pic_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It does
not import, and is not imported by, paper_1603_02886_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic_ref.c")
_LIB = os.path.join(_HERE, "libpicref.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2, IEEE semantics: no fast-math, no FMA contraction."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_LIB_OMP = os.path.join(_HERE, "libpicref_omp.so")


def build_openmp(force: bool = False) -> str:
    """The TIMED-ONLY OpenMP build of the same source (bench.py's cpu_baseline; never used for parity)."""
    if force or not os.path.exists(_LIB_OMP) or os.path.getmtime(_LIB_OMP) < os.path.getmtime(_SRC):
        tmp = _LIB_OMP + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB_OMP)
    return _LIB_OMP


def step_openmp(g: "Grid", x, v, w, E, dt: float, qm: float, threads: int):
    """pic_ref_step of the OpenMP build on `threads` host threads -> dict like step()."""
    lib = ctypes.CDLL(build_openmp())
    lib.pic_ref_step.restype = ctypes.c_int
    omp = ctypes.CDLL("libgomp.so.1")
    omp.omp_set_num_threads(int(threads))
    n = w.shape[0]
    xo = [np.empty_like(a) for a in x]
    vo = [np.empty_like(a) for a in v]
    wo = np.empty_like(w)
    perm = np.empty(n, np.int32)
    off = np.empty(g.cells + 1, np.int32)
    rho = np.empty(g.cells, np.float64)
    cg = g.c()
    _rc(lib.pic_ref_step(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x), _ptrs(v), ctypes.c_void_p(w.ctypes.data),
                         _ptrs(xo), _ptrs(vo), ctypes.c_void_p(wo.ctypes.data), ctypes.c_void_p(perm.ctypes.data),
                         ctypes.c_void_p(off.ctypes.data), ctypes.c_void_p(rho.ctypes.data), _ptrs(E),
                         ctypes.c_double(dt), ctypes.c_double(qm), ctypes.c_int(1)))
    return dict(x=xo, v=vo, w=wo, perm=perm, cell_offsets=off, rho=rho)


class _Grid(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int32), ("n", ctypes.c_int32 * 3), ("h", ctypes.c_double * 3),
                ("order", ctypes.c_int32), ("dtype", ctypes.c_int32)]


@dataclass(frozen=True)
class Grid:
    dim: int
    n: Tuple[int, ...]
    h: Tuple[float, ...]
    order: int
    dtype: str  # "f32" | "f64"

    @property
    def cells(self) -> int:
        return int(np.prod(self.n[: self.dim]))

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32

    def c(self) -> _Grid:
        g = _Grid()
        g.dim = self.dim
        for k in range(3):
            g.n[k] = self.n[k] if k < self.dim else 1
            g.h[k] = self.h[k] if k < self.dim else 1.0
        g.order = self.order
        g.dtype = 1 if self.dtype == "f64" else 0
        return g


def grid_of(cfg) -> Grid:
    """Grid of a pic_workloads.Config."""
    return Grid(cfg.dim, tuple(cfg.n), tuple([cfg.h] * cfg.dim), cfg.order, cfg.dtype)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.pic_ref_bspline.argtypes = [ctypes.c_int, ctypes.c_double]
        lib.pic_ref_bspline.restype = ctypes.c_double
        for name in ("pic_ref_stencil_1d", "pic_ref_keys", "pic_ref_sort", "pic_ref_deposit",
                     "pic_ref_deposit_allpairs", "pic_ref_gather", "pic_ref_gather_allnodes",
                     "pic_ref_push", "pic_ref_step"):
            getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def _ptrs(arrs: Sequence[np.ndarray]):
    p = (ctypes.c_void_p * 3)()
    for k in range(3):
        p[k] = arrs[k].ctypes.data if k < len(arrs) else None
    return p


def _chk(g: Grid, arrs, n=None, dtype=None):
    dt = dtype or g.np_dtype
    for a in arrs:
        assert isinstance(a, np.ndarray) and a.dtype == dt and a.flags.c_contiguous, (a.dtype, dt)
        if n is not None:
            assert a.shape == (n,), (a.shape, n)


def _rc(rc):
    if rc != 0:
        raise ValueError("oracle: bad argument (rc=%d)" % rc)


def bspline(p: int, t: float) -> float:
    return _load().pic_ref_bspline(int(p), float(t))


def stencil_1d(g: Grid, c: int, x: np.ndarray, i: int = 0):
    """(node indices, weights) of particle i in dimension c."""
    _chk(g, [x])
    idx = np.zeros(4, np.int32)
    wt = np.zeros(4, np.float64)
    cg = g.c()
    m = _load().pic_ref_stencil_1d(ctypes.byref(cg), c, ctypes.c_void_p(x.ctypes.data),
                                   ctypes.c_int64(i), ctypes.c_void_p(idx.ctypes.data),
                                   ctypes.c_void_p(wt.ctypes.data))
    if m < 0:
        _rc(m)
    return idx[:m].copy(), wt[:m].copy()


def keys(g: Grid, x) -> np.ndarray:
    n = x[0].shape[0]
    _chk(g, x, n)
    key = np.empty(n, np.int32)
    cg = g.c()
    _rc(_load().pic_ref_keys(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x),
                             ctypes.c_void_p(key.ctypes.data)))
    return key


def sort(g: Grid, x, v, w):
    """-> (x_out, v_out, w_out, perm[n] int32, cell_offsets[C+1] int32)."""
    n = w.shape[0]
    _chk(g, list(x) + list(v) + [w], n)
    xo = [np.empty_like(a) for a in x]
    vo = [np.empty_like(a) for a in v]
    wo = np.empty_like(w)
    perm = np.empty(n, np.int32)
    off = np.empty(g.cells + 1, np.int32)
    cg = g.c()
    _rc(_load().pic_ref_sort(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x), _ptrs(v),
                             ctypes.c_void_p(w.ctypes.data), _ptrs(xo), _ptrs(vo),
                             ctypes.c_void_p(wo.ctypes.data), ctypes.c_void_p(perm.ctypes.data),
                             ctypes.c_void_p(off.ctypes.data)))
    return xo, vo, wo, perm, off


def _bucket3(g: Grid, bucket):
    b = (ctypes.c_int32 * 3)(1, 1, 1)
    for c in range(g.dim):
        b[c] = int(bucket[c])
    return b


def bucket_count(g: Grid, bucket) -> int:
    """Number of buckets of `bucket[c]` cells per dimension (NEXT-2)."""
    cg = g.c()
    lib = _load()
    lib.pic_ref_bucket_count.restype = ctypes.c_int64
    B = lib.pic_ref_bucket_count(ctypes.byref(cg), _bucket3(g, bucket))
    if B < 0:
        _rc(-1)
    return int(B)


def bucket_keys(g: Grid, x, bucket) -> np.ndarray:
    n = x[0].shape[0]
    _chk(g, x, n)
    key = np.empty(n, np.int32)
    cg = g.c()
    _rc(_load().pic_ref_bucket_keys(ctypes.byref(cg), _bucket3(g, bucket), ctypes.c_int64(n), _ptrs(x),
                                    ctypes.c_void_p(key.ctypes.data)))
    return key


def sort_buckets(g: Grid, x, v, w, bucket):
    """Stable sort by bucket key -> (x_out, v_out, w_out, perm[n] int32, bucket_offsets[B+1] int32)."""
    n = w.shape[0]
    _chk(g, list(x) + list(v) + [w], n)
    xo = [np.empty_like(a) for a in x]
    vo = [np.empty_like(a) for a in v]
    wo = np.empty_like(w)
    perm = np.empty(n, np.int32)
    off = np.empty(bucket_count(g, bucket) + 1, np.int32)
    cg = g.c()
    _rc(_load().pic_ref_sort_buckets(ctypes.byref(cg), _bucket3(g, bucket), ctypes.c_int64(n), _ptrs(x), _ptrs(v),
                                     ctypes.c_void_p(w.ctypes.data), _ptrs(xo), _ptrs(vo),
                                     ctypes.c_void_p(wo.ctypes.data), ctypes.c_void_p(perm.ctypes.data),
                                     ctypes.c_void_p(off.ctypes.data)))
    return xo, vo, wo, perm, off


def sort_buckets_inplace(g: Grid, x, v, w, bucket):
    """Alg. 2 (sort for pre-ordered particles, in place, only misplaced particles move)
    -> (x, v, w copies after the sort, bucket_offsets[B+1] int32, number of particles moved)."""
    n = w.shape[0]
    _chk(g, list(x) + list(v) + [w], n)
    xo = [a.copy() for a in x]
    vo = [a.copy() for a in v]
    wo = w.copy()
    off = np.empty(bucket_count(g, bucket) + 1, np.int32)
    moved = ctypes.c_int64(0)
    cg = g.c()
    _rc(_load().pic_ref_sort_buckets_inplace(ctypes.byref(cg), _bucket3(g, bucket), ctypes.c_int64(n), _ptrs(xo), _ptrs(vo),
                                             ctypes.c_void_p(wo.ctypes.data), ctypes.c_void_p(off.ctypes.data),
                                             ctypes.byref(moved)))
    return xo, vo, wo, off, int(moved.value)


def deposit(g: Grid, x, w, allpairs: bool = False) -> np.ndarray:
    """rho[C] in float64, x fastest."""
    n = w.shape[0]
    _chk(g, list(x) + [w], n)
    rho = np.empty(g.cells, np.float64)
    cg = g.c()
    f = _load().pic_ref_deposit_allpairs if allpairs else _load().pic_ref_deposit
    _rc(f(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x), ctypes.c_void_p(w.ctypes.data),
          ctypes.c_void_p(rho.ctypes.data)))
    return rho


def gather(g: Grid, x, E, allnodes: bool = False):
    """Field at the particles, float64, one array per dimension."""
    n = x[0].shape[0]
    _chk(g, x, n)
    _chk(g, E, g.cells)
    Ep = [np.empty(n, np.float64) for _ in range(g.dim)]
    cg = g.c()
    f = _load().pic_ref_gather_allnodes if allnodes else _load().pic_ref_gather
    _rc(f(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x), _ptrs(E), _ptrs(Ep)))
    return Ep


def push(g: Grid, x, v, E, dt: float, qm: float):
    """accel + push; returns new (x, v) (inputs are not modified)."""
    n = x[0].shape[0]
    _chk(g, list(x) + list(v), n)
    _chk(g, E, g.cells)
    xo = [a.copy() for a in x]
    vo = [a.copy() for a in v]
    cg = g.c()
    _rc(_load().pic_ref_push(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(xo), _ptrs(vo), _ptrs(E),
                             ctypes.c_double(dt), ctypes.c_double(qm)))
    return xo, vo


def step(g: Grid, x, v, w, E, dt: float, qm: float, do_sort: bool = True, cell_offsets=None):
    """sort -> deposit(x^t) -> accel -> push.  -> dict(x, v, w, perm, cell_offsets, rho)."""
    n = w.shape[0]
    _chk(g, list(x) + list(v) + [w], n)
    _chk(g, E, g.cells)
    xo = [np.empty_like(a) for a in x]
    vo = [np.empty_like(a) for a in v]
    wo = np.empty_like(w)
    perm = np.empty(n, np.int32)
    off = np.empty(g.cells + 1, np.int32) if cell_offsets is None else cell_offsets.copy()
    rho = np.empty(g.cells, np.float64)
    cg = g.c()
    _rc(_load().pic_ref_step(ctypes.byref(cg), ctypes.c_int64(n), _ptrs(x), _ptrs(v),
                             ctypes.c_void_p(w.ctypes.data), _ptrs(xo), _ptrs(vo),
                             ctypes.c_void_p(wo.ctypes.data), ctypes.c_void_p(perm.ctypes.data),
                             ctypes.c_void_p(off.ctypes.data), ctypes.c_void_p(rho.ctypes.data),
                             _ptrs(E), ctypes.c_double(dt), ctypes.c_double(qm),
                             ctypes.c_int(1 if do_sort else 0)))
    return dict(x=xo, v=vo, w=wo, perm=perm, cell_offsets=off, rho=rho)


# ---------------------------------------------------------------------------------------------
# NEXT-4: the field solve, step ii of the loop -- "field_solver(): -Laplace(phi) = rho"
# (section 3; "we solve Poisson's equation for computing the field potential phi"),
# periodic boundary conditions.  The paper leaves the step out ("Step ii involving field_solver is
# not considered"), so everything beyond the equation is a reading (R21-R23):
#   R21  E = -grad(phi) (electrostatics; "the forces on each particle from the electric potential")
#   R22  the mean of rho is dropped (a periodic box is solvable only for zero net charge: uniform neutralising
#        background); phi has zero mean
#   R23  spectral discretisation on the node grid: with rho^ = DFT(rho) and wave numbers
#        kappa_c(m) = 2 pi mt / L_c, mt = m for m <= n/2, m - n above,
#        phi^ = rho^ / sum_c kappa_c^2,   E_c^ = -i kappa'_c phi^,
#        kappa' = kappa except kappa' = 0 at the Nyquist index m = n/2 of an even n (the derivative of that
#        mode of a real grid function is not a real grid function).
# Plain numpy, float64; np.fft.fftn / ifftn are the library primitive that serves as the step.  Pinned in
# tests/test_oracle_field.py against the analytic single-mode solution, a brute-force O(C^2) Fourier sum on
# tiny grids, the finite-difference Gauss law on smooth fields and the cold-plasma oscillation frequency.
def field_solve(g: Grid, rho):
    """(phi, [E_c]) on the node grid, x fastest, float64."""
    shape = tuple(reversed(g.n[: g.dim]))                        # C order: z, y, x
    r = np.asarray(rho, np.float64).reshape(shape)
    rh = np.fft.fftn(r)
    kap, kapd = [], []
    for c in range(g.dim):
        n, L = g.n[c], g.n[c] * g.h[c]
        m = np.arange(n)
        mt = np.where(m <= n // 2, m, m - n).astype(np.float64)
        k = 2.0 * np.pi * mt / L
        kd = k.copy()
        if n % 2 == 0:
            kd[n // 2] = 0.0
        ax = [1] * g.dim
        ax[g.dim - 1 - c] = n
        kap.append(k.reshape(ax))
        kapd.append(kd.reshape(ax))
    k2 = sum(k * k for k in kap)
    k2[(0,) * g.dim] = 1.0
    ph = rh / k2
    ph[(0,) * g.dim] = 0.0
    phi = np.real(np.fft.ifftn(ph)).reshape(-1)
    E = [np.real(np.fft.ifftn(-1j * kapd[c] * ph)).reshape(-1) for c in range(g.dim)]
    return phi, E


def step_selfconsistent(g: Grid, x, v, w, dt: float, qm: float):
    """One step of the closed loop i-iv: sort -> setrho -> field_solver -> accel -> push.
    E is stored in the grid's dtype before the push, as the CUDA path stores it.  -> dict like step() plus E, phi."""
    xs, vs, ws, perm, off = sort(g, x, v, w)
    rho = deposit(g, xs, ws)
    phi, E = field_solve(g, rho)
    Es = [e.astype(g.np_dtype) for e in E]
    xo, vo = push(g, xs, vs, Es, dt, qm)
    return dict(x=xo, v=vo, w=ws, perm=perm, cell_offsets=off, rho=rho, E=Es, phi=phi)
