"""Pins of the oracle's B-spline basis and 1-D stencil (oracle/pic_ref.c, O1).

Independent of the oracle: the textbook truncated-power formula of the cardinal
B-spline, exact rational worked values (tests/golden), and the paper's own hat
function / trilinear products.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
from conftest import read_golden


def cardinal_bspline(p, t):
    """Centred cardinal B-spline of degree p by the truncated-power (Schoenberg) formula:
    B_p(t) = 1/p! * sum_k (-1)^k C(p+1,k) (t + (p+1)/2 - k)_+^p.  Textbook; shares nothing
    with the piecewise form in the oracle."""
    s = 0.0
    for k in range(p + 2):
        u = t + 0.5 * (p + 1) - k
        if u > 0:
            s += (-1) ** k * math.comb(p + 1, k) * u ** p
    return s / math.factorial(p)


@pytest.mark.parametrize("p", [1, 2, 3])
def test_closed_form_vs_truncated_power(p):
    for t in np.linspace(-2.6, 2.6, 1041):
        assert abs(O.bspline(p, float(t)) - cardinal_bspline(p, float(t))) < 2e-14  # cancellation in the truncated powers


def test_p1_is_the_papers_hat_function():
    # IF ABS(w) <= 1: MIN(1-w, 1+w)
    for w in np.linspace(-1.5, 1.5, 301):
        want = min(1.0 - w, 1.0 + w) if abs(w) <= 1.0 else 0.0
        assert O.bspline(1, float(w)) == pytest.approx(want, abs=1e-16)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("p", [1, 2, 3])
def test_stencil_matches_closed_form_and_moments(p, dtype):
    n = 16
    g = O.Grid(2, (n, n), (1.0, 1.0), p, dtype)
    rng = np.random.default_rng(p)
    ts = np.concatenate([rng.uniform(0, n, 400), [0.0, 0.5, 1.0, 7.5, n - 1.0, n - 0.5, n - 1e-7]])
    for t in ts:
        x = np.array([t], g.np_dtype)
        tt = float(x[0])
        idx, wt = O.stencil_1d(g, 0, x)
        assert len(idx) == p + 1
        # closed form at the unfolded node positions
        i0 = min(max(math.floor(tt), 0), n - 1)
        first = {1: i0, 2: i0 + (1 if tt - i0 >= 0.5 else 0) - 1, 3: i0 - 1}[p]
        for a in range(p + 1):
            j = first + a
            assert idx[a] == j % n
            assert wt[a] == pytest.approx(cardinal_bspline(p, tt - j), abs=2e-14)
        # partition of unity, first moment, second central moment
        js = np.arange(first, first + p + 1, dtype=np.float64)
        assert math.fsum(wt) == pytest.approx(1.0, abs=4e-16)
        assert math.fsum(wt * js) == pytest.approx(tt, abs=1e-14)
        m2 = math.fsum(wt * (tt - js) ** 2)
        xi = tt - i0
        want = xi * (1 - xi) if p == 1 else (p + 1) / 12.0
        assert m2 == pytest.approx(want, abs=1e-14)
        # nothing outside the stencil carries weight
        assert cardinal_bspline(p, tt - (first - 1)) == pytest.approx(0.0, abs=2e-14)
        assert cardinal_bspline(p, tt - (first + p + 1)) == pytest.approx(0.0, abs=2e-14)


def test_worked_values_golden():
    rows = read_golden("bspline_worked_values.txt")
    seen = 0
    for p, t, node, frac in rows:
        p, t, node = int(p), float(t), int(node)
        want = float(Fraction(frac))
        g = O.Grid(2, (16, 16), (1.0, 1.0), p, "f64")
        idx, wt = O.stencil_1d(g, 0, np.array([t]))
        assert node in idx, (p, t, node, idx)
        assert wt[list(idx).index(node)] == pytest.approx(want, abs=1e-16)
        assert O.bspline(p, t - node) == pytest.approx(want, abs=1e-16)
        seen += 1
    assert seen == 27


def test_periodic_fold_of_the_stencil():
    n = 8
    g3 = O.Grid(2, (n, n), (1.0, 1.0), 3, "f64")
    idx, _ = O.stencil_1d(g3, 0, np.array([0.25]))
    assert list(idx) == [n - 1, 0, 1, 2]
    idx, _ = O.stencil_1d(g3, 0, np.array([n - 0.75]))
    assert list(idx) == [n - 2, n - 1, 0, 1]
    g2 = O.Grid(2, (n, n), (1.0, 1.0), 2, "f64")
    idx, _ = O.stencil_1d(g2, 0, np.array([0.25]))
    assert list(idx) == [n - 1, 0, 1]
    idx, _ = O.stencil_1d(g2, 0, np.array([n - 0.25]))
    assert list(idx) == [n - 1, 0, 1]
    g1 = O.Grid(2, (n, n), (1.0, 1.0), 1, "f64")
    idx, _ = O.stencil_1d(g1, 0, np.array([n - 0.25]))
    assert list(idx) == [n - 1, 0]


def test_x_equal_L_behaves_as_x_equal_0():
    # reading R5: key and stencil clamp to the last cell, xi reaches 1, polynomials are continuous
    n = 8
    for p in (1, 2, 3):
        g = O.Grid(2, (n, n), (1.0, 1.0), p, "f64")
        xa = [np.array([float(n)]), np.array([3.3])]
        xb = [np.array([0.0]), np.array([3.3])]
        w = np.array([1.0])
        assert np.allclose(O.deposit(g, xa, w), O.deposit(g, xb, w), atol=1e-16)
        assert O.keys(g, xa)[0] == n - 1 + n * 3


def test_non_unit_spacing_uses_x_over_h():
    g = O.Grid(2, (8, 8), (0.5, 2.0), 1, "f64")
    idx, wt = O.stencil_1d(g, 0, np.array([1.375]))     # t = 2.75
    assert list(idx) == [2, 3] and wt == pytest.approx([0.25, 0.75])
    idx, wt = O.stencil_1d(g, 1, np.array([5.0]))       # t = 2.5
    assert list(idx) == [2, 3] and wt == pytest.approx([0.5, 0.5])


def test_paper_trilinear_products_golden():
    # one particle at (ix+wx, iy+wy, iz+wz), linear splines, 3-D
    rows = read_golden("paper_trilinear_products.txt")
    n = 8
    g = O.Grid(3, (n, n, n), (1.0, 1.0, 1.0), 1, "f64")
    ix, iy, iz = 2, 5, 3
    x = [np.array([ix + 0.25]), np.array([iy + 0.375]), np.array([iz + 0.125])]
    rho = O.deposit(g, x, np.array([1.0])).reshape(n, n, n)   # [z][y][x]
    total = 0.0
    for dx, dy, dz, val in rows:
        got = rho[iz + int(dz), iy + int(dy), ix + int(dx)]
        assert got == float(val), (dx, dy, dz, got, val)
        total += got
    assert total == 1.0
    assert np.count_nonzero(rho) == 8
