"""Pins of the oracle's field solve (oracle.field_solve; "-Laplace(phi) = rho", 86, 88)
against things that are not the oracle: the analytic solution for one Fourier mode, a brute-force O(C^2) Fourier sum
written out with explicit loops over wave numbers (no FFT), the finite-difference Gauss law on smooth fields, and --
for the closed loop -- the cold-plasma oscillation frequency omega_p^2 = (q/m) rho_0."""
import itertools

import numpy as np
import pytest

import oracle as O


def _nodes(g):
    """coordinates of all nodes, x fastest: list over dimensions of arrays [C]"""
    idx = np.indices(tuple(reversed(g.n[: g.dim])))              # z, y, x order
    return [idx[g.dim - 1 - c].reshape(-1) * g.h[c] for c in range(g.dim)]


@pytest.mark.parametrize("n,h,m", [((16, 12), (1.0, 1.0), (1, 0)), ((16, 12), (0.5, 2.0), (2, -3)), ((9, 7), (1.0, 0.3), (-4, 3)),
                                   ((8, 6, 10), (1.0, 1.0, 1.0), (1, 1, 1)), ((8, 6, 10), (0.25, 1.5, 0.7), (3, -2, 4)),
                                   ((5, 4, 3), (1.0, 2.0, 3.0), (2, 1, -1))])
def test_single_mode_is_the_analytic_solution(n, h, m):
    """rho = A cos(k.x + th)  =>  phi = rho / |k|^2,  E = -grad phi = A k / |k|^2 sin(k.x + th)   (continuous PDE)."""
    d = len(n)
    g = O.Grid(d, n, h, 1, "f64")
    X = _nodes(g)
    k = [2.0 * np.pi * m[c] / (n[c] * h[c]) for c in range(d)]
    assert all(abs(m[c]) < n[c] / 2 for c in range(d))            # below Nyquist: representable
    ph = sum(k[c] * X[c] for c in range(d)) + 0.37
    A = 1.7
    rho = A * np.cos(ph) + 0.9                                    # the mean is dropped (R22)
    phi, E = O.field_solve(g, rho)
    k2 = sum(kc * kc for kc in k)
    assert np.allclose(phi, A * np.cos(ph) / k2, rtol=0, atol=1e-12 * A / k2)
    for c in range(d):
        assert np.allclose(E[c], A * k[c] / k2 * np.sin(ph), rtol=0, atol=1e-12 * A / np.sqrt(k2))


@pytest.mark.parametrize("n,h", [((4, 6), (1.0, 0.5)), ((5, 3), (1.0, 1.0)), ((3, 4, 5), (1.0, 2.0, 0.5)), ((4, 4, 2), (1.0, 1.0, 1.0))])
def test_brute_force_fourier_sum(n, h):
    """phi[j] = (1/C) sum_m rho^_m e^{+i k_m.x_j} / |k_m|^2 with rho^_m = sum_j rho_j e^{-i k_m.x_j}: explicit loops over
    every wave number and node, signed wave numbers, Nyquist derivative zero."""
    d = len(n)
    g = O.Grid(d, n, h, 1, "f64")
    rng = np.random.default_rng(11)
    C = int(np.prod(n))
    rho = rng.normal(size=C)
    X = _nodes(g)
    phi = np.zeros(C, complex)
    E = [np.zeros(C, complex) for _ in range(d)]
    for m in itertools.product(*[range(k) for k in n]):
        if all(v == 0 for v in m):
            continue
        ms = [m[c] if m[c] <= n[c] // 2 else m[c] - n[c] for c in range(d)]
        k = [2.0 * np.pi * ms[c] / (n[c] * h[c]) for c in range(d)]
        kd = [0.0 if (n[c] % 2 == 0 and m[c] == n[c] // 2) else k[c] for c in range(d)]
        phase = sum(k[c] * X[c] for c in range(d))
        rh = np.sum(rho * np.exp(-1j * phase))
        ph = rh / sum(kc * kc for kc in k)
        phi += ph * np.exp(1j * phase) / C
        for c in range(d):
            E[c] += -1j * kd[c] * ph * np.exp(1j * phase) / C
    p, Eo = O.field_solve(g, rho)
    assert np.allclose(p, phi.real, rtol=0, atol=1e-12 * np.max(np.abs(phi)))
    for c in range(d):
        assert np.allclose(Eo[c], E[c].real, rtol=0, atol=1e-12 * np.max(np.abs(E[c])))
    assert abs(np.sum(p)) < 1e-12 * C * np.max(np.abs(p))


def test_gauss_law_by_finite_differences():
    """div E = rho - mean(rho) and E = -grad phi, checked with central differences on a smooth charge density:
    the error falls four-fold per grid doubling (a wrong sign, factor 2 pi or transposed axis does not)."""
    errs = []
    for n in (32, 64):
        g = O.Grid(3, (n, n, n), (1.0 / n, 2.0 / n, 0.5 / n), 1, "f64")
        X = _nodes(g)
        L = [g.n[c] * g.h[c] for c in range(3)]
        rho = (np.sin(2 * np.pi * X[0] / L[0]) * np.cos(4 * np.pi * X[1] / L[1]) + 0.5 * np.cos(2 * np.pi * (X[2] / L[2] + X[0] / L[0])) + 3.0)
        phi, E = O.field_solve(g, rho)
        shape = (n, n, n)
        div = np.zeros(shape)
        for c in range(3):
            ax = 2 - c
            Ec, pc = E[c].reshape(shape), phi.reshape(shape)
            div += (np.roll(Ec, -1, ax) - np.roll(Ec, 1, ax)) / (2 * g.h[c])
            grad = (np.roll(pc, -1, ax) - np.roll(pc, 1, ax)) / (2 * g.h[c])
            assert np.max(np.abs(grad + Ec)) < 0.04 * np.max(np.abs(Ec)) * (32 / n) ** 2 + 1e-12   # (kh)^2/6 of the m = 2 mode
        errs.append(np.max(np.abs(div.reshape(-1) - (rho - rho.mean()))) / np.max(np.abs(rho - rho.mean())))
    assert errs[0] < 0.05 and 3.5 < errs[0] / errs[1] < 4.5


def test_solution_is_linear_and_mean_free():
    g = O.Grid(2, (12, 10), (1.0, 1.0), 1, "f64")
    rng = np.random.default_rng(2)
    a, b = rng.normal(size=120), rng.normal(size=120)
    pa, Ea = O.field_solve(g, a)
    pb, Eb = O.field_solve(g, b)
    pc, Ec = O.field_solve(g, 2.0 * a - 3.0 * b + 7.0)
    assert np.allclose(pc, 2 * pa - 3 * pb, atol=1e-12)
    for c in range(2):
        assert np.allclose(Ec[c], 2 * Ea[c] - 3 * Eb[c], atol=1e-12)
        assert abs(Ec[c].mean()) < 1e-13
    pz, Ez = O.field_solve(g, np.full(120, 4.2))
    assert np.max(np.abs(pz)) < 1e-13 and all(np.max(np.abs(e)) < 1e-13 for e in Ez)      # a uniform charge: no field


@pytest.mark.parametrize("order", [1, 3])
def test_cold_plasma_oscillation_frequency(order):
    """Closed loop (PAPER.md:79-84 steps i-iv): cold particles on a lattice, displaced by a small sine wave, oscillate at
    omega_p^2 = (q/m) rho_0 (div E = rho, dv/dt = (q/m) E).  The amplitude of the fundamental of rho follows
    cos(omega t) with omega = omega_p * [sinc(k h / 2)]^(p+1) (the spline shape enters twice: deposit and gather)
    within the leapfrog's O((omega dt)^2)."""
    n = (32, 4)
    ppc = 16
    g = O.Grid(2, n, (1.0, 1.0), order, "f64")
    N = n[0] * n[1] * ppc
    ix = (np.arange(N) % (n[0] * 4) + 0.5) / 4.0                  # 4 x 4 particles per cell, regular lattice
    iy = (np.arange(N) // (n[0] * 4) + 0.5) / 4.0
    k = 2 * np.pi / n[0]
    amp = 1e-3
    x = [np.mod(ix + amp * np.sin(k * ix), n[0]), iy.copy()]
    v = [np.zeros(N), np.zeros(N)]
    rho0, qm = 0.25, 1.0                                           # omega_p = 0.5
    w = np.full(N, rho0 / ppc)
    dt = 0.2
    omega = np.sqrt(qm * rho0) * np.sinc(k / 2 / np.pi) ** (order + 1)
    a = []
    for s in range(64):
        r = O.step_selfconsistent(g, x, v, w, dt, qm)
        rr = r["rho"].reshape(n[1], n[0]).mean(axis=0)
        a.append(2.0 * np.mean(rr * np.cos(k * np.arange(n[0]))))
        x, v, w = r["x"], r["v"], r["w"]
    a = np.array(a)
    t = dt * np.arange(64)
    # x(t+dt) uses v(t+dt): the density at step s is at time t_s, started from rest half a step "late" in v
    model = a[0] * np.cos(omega * t)
    assert abs(a[0]) > 0.5 * amp * k * rho0
    assert np.max(np.abs(a - model)) < 0.08 * abs(a[0])
    # and it really oscillates: sign change near a quarter period
    q = int(round(np.pi / 2 / omega / dt))
    assert abs(a[q]) < 0.15 * abs(a[0]) and a[2 * q] * np.sign(a[0]) < -0.8 * abs(a[0])
