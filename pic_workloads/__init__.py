"""Seeded synthetic workloads shaped like the paper's benchmark.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_1603_02886_b200/`).  It holds none of the method's arithmetic: it
draws counter-based random numbers (gen.c) and evaluates the prescribed, frozen
field.  The five configurations are those of BASELINE.json; the recipe is
restated in DESIGN.md ("Input recipe").
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, replace
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libpicw.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gen.c into libpicw.so (gcc, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC",
                               "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, i64, dbl, vp, ci = (ctypes.c_uint64, ctypes.c_int64, ctypes.c_double,
                                 ctypes.c_void_p, ctypes.c_int)
        lib.picw_uniform01.argtypes = [u64, u64, i64, i64, vp]
        lib.picw_fill_uniform.argtypes = [u64, u64, i64, dbl, dbl, dbl, ci, vp]
        lib.picw_fill_normal.argtypes = [u64, u64, u64, i64, dbl, dbl, ci, vp]
        lib.picw_fill_clustered.argtypes = [u64, u64, u64, u64, u64, i64, dbl, dbl, dbl, dbl, ci, vp]
        lib.picw_field_modes.argtypes = [ci, vp, ci, vp, vp, vp, vp, ci, ci, vp]
        for f in (lib.picw_uniform01, lib.picw_fill_uniform, lib.picw_fill_normal,
                  lib.picw_fill_clustered, lib.picw_field_modes):
            f.restype = None
        _lib = lib
    return _lib


# stream ids (fixed; part of the recipe)
S_X = (0, 1, 2)
S_V = ((10, 11), (12, 13), (14, 15))
S_W = 20
S_SEL = 30
S_BLOB = ((40, 41), (42, 43), (44, 45))
S_MODE_K = (50, 51, 52)
S_MODE_AMP = 53
S_MODE_PHASE = 54


@dataclass(frozen=True)
class Config:
    """One BASELINE.json configuration."""
    name: str
    dim: int
    n: Tuple[int, ...]          # cells (= nodes) per dimension
    N: int                      # particles
    dtype: str                  # "f32" | "f64"
    order: int                  # B-spline degree p
    weights: str                # "inv_n" (w=1/N) | "uniform" (w=0.5+u) | "one"
    modes: int                  # 0 -> the single mode sin(2 pi x/Lx) of config 1; else M seeded low-k modes
    steps: int
    sort_every: int = 1
    clustered: bool = False
    h: float = 1.0
    dt: float = 0.1
    qm: float = 1.0
    sigma_v: float = 1.0
    seed: int = 0

    @property
    def cells(self) -> int:
        return int(np.prod(self.n))

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32

    @property
    def L(self) -> Tuple[float, ...]:
        return tuple(k * self.h for k in self.n)

    def scaled(self, N: int, **kw) -> "Config":
        return replace(self, N=int(N), **kw)


CONFIGS = {
    # BASELINE.json configs[0..4]
    "cfg1": Config("cfg1", 2, (64, 64), 100_000, "f64", 1, "inv_n", 0, 1),
    "cfg2": Config("cfg2", 2, (256, 256), 10_000_000, "f64", 2, "uniform", 4, 10),
    "cfg3": Config("cfg3", 3, (128, 128, 128), 100_000_000, "f32", 3, "one", 8, 10),
    "cfg4": Config("cfg4", 3, (128, 128, 128), 100_000_000, "f32", 3, "one", 8, 10, clustered=True),
    # config 5 is a sweep: ppc in {8,32,128,512} on 64^3, sort every {1,4,16}; base entry = ppc 8
    "cfg5": Config("cfg5", 3, (64, 64, 64), 8 * 64 ** 3, "f64", 2, "one", 8, 100),
}
CFG5_PPC = (8, 32, 128, 512)
CFG5_SORT_EVERY = (1, 4, 16)


def cfg5(ppc: int, sort_every: int = 1) -> Config:
    return replace(CONFIGS["cfg5"], name="cfg5_ppc%d_k%d" % (ppc, sort_every),
                   N=ppc * 64 ** 3, sort_every=sort_every)


@dataclass
class Workload:
    cfg: Config
    x: list          # dim arrays [N], storage dtype, 0 <= x < L
    v: list          # dim arrays [N]
    w: np.ndarray    # [N]
    E: list          # dim arrays [C], storage dtype, x fastest
    modes: dict      # k, dir, amp, phase of the prescribed field


def uniform01(seed: int, stream: int, i0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().picw_uniform01(seed, stream, i0, n, out.ctypes.data)
    return out


def field_modes(cfg: Config):
    """Wave vectors, directions, amplitudes and phases of the prescribed field."""
    d = cfg.dim
    if cfg.modes == 0:  # config 1: E_x = sin(2 pi j_x / n_x), E_y = 0
        k = np.zeros((1, 3), np.int32); k[0, 0] = 1
        dirs = np.zeros((1, 3)); dirs[0, 0] = 1.0
        return dict(k=k, dir=dirs, amp=np.ones(1), phase=np.zeros(1))
    M = cfg.modes
    k = np.zeros((M, 3), np.int32)
    for c in range(d):
        k[:, c] = np.floor(5.0 * uniform01(cfg.seed, S_MODE_K[c], 0, M)).astype(np.int32) - 2
    zero = ~np.any(k != 0, axis=1)
    k[zero, 0] = 1
    norm = np.sqrt((k.astype(np.float64) ** 2).sum(axis=1))
    dirs = k.astype(np.float64) / norm[:, None]
    amp = (0.5 + 0.5 * uniform01(cfg.seed, S_MODE_AMP, 0, M)) / M
    phase = 2.0 * math.pi * uniform01(cfg.seed, S_MODE_PHASE, 0, M)
    return dict(k=k, dir=dirs, amp=amp, phase=phase)


def make_field(cfg: Config):
    lib = _load()
    m = field_modes(cfg)
    n3 = np.array(list(cfg.n) + [1] * (3 - cfg.dim), np.int32)
    k = np.ascontiguousarray(m["k"], np.int32)
    dirs = np.ascontiguousarray(m["dir"], np.float64)
    amp = np.ascontiguousarray(m["amp"], np.float64)
    ph = np.ascontiguousarray(m["phase"], np.float64)
    E = []
    for c in range(cfg.dim):
        out = np.empty(cfg.cells, cfg.np_dtype)
        lib.picw_field_modes(cfg.dim, n3.ctypes.data, len(amp), k.ctypes.data, dirs.ctypes.data,
                             amp.ctypes.data, ph.ctypes.data, c, int(cfg.dtype == "f64"),
                             out.ctypes.data)
        E.append(out)
    return E, m


def make_workload(cfg: Config) -> Workload:
    """Particles (random initial order) and field of one configuration, host numpy arrays."""
    lib = _load()
    N, f64, dt = cfg.N, int(cfg.dtype == "f64"), cfg.np_dtype
    x, v = [], []
    for c in range(cfg.dim):
        xc = np.empty(N, dt)
        L = cfg.L[c]
        if cfg.clustered:   # config 4: 70 % Gaussian blob (sigma = 4 cells) at the box centre
            lib.picw_fill_clustered(cfg.seed, S_SEL, S_X[c], S_BLOB[c][0], S_BLOB[c][1], N,
                                    0.7, 0.5 * L, 4.0 * cfg.h, L, f64, xc.ctypes.data)
        else:
            lib.picw_fill_uniform(cfg.seed, S_X[c], N, 0.0, L, L, f64, xc.ctypes.data)
        x.append(xc)
        vc = np.empty(N, dt)
        lib.picw_fill_normal(cfg.seed, S_V[c][0], S_V[c][1], N, 0.0, cfg.sigma_v, f64, vc.ctypes.data)
        v.append(vc)
    if cfg.weights == "inv_n":
        w = np.full(N, 1.0 / N, dt)
    elif cfg.weights == "uniform":
        w = np.empty(N, dt)
        lib.picw_fill_uniform(cfg.seed, S_W, N, 0.5, 1.5, 0.0, f64, w.ctypes.data)
    else:
        w = np.ones(N, dt)
    E, m = make_field(cfg)
    return Workload(cfg, x, v, w, E, m)
