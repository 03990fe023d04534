"""Pins for the 2-D heat oracle (oracle/heat2d.inc).  Expected values come from closed forms and
invariants, not from a second typing of the update formula."""
from math import comb

import numpy as np
import pytest

import oracle


def _grid(n):
    return 1.0 / n, 0.25 / (n * n)       # dx, dt with alpha = 1: Fo = 1/4 exactly


def test_delta_response_at_Fo_quarter_is_the_lattice_walk_distribution_exactly():
    """Fo = 1/4 makes 1 - 4 Fo = 0: every step replaces a value by the mean of its four neighbours, so a unit delta becomes the
    distribution of the simple random walk on Z^2 -- P_n(i, j) = C(n, (n+i+j)/2) C(n, (n+i-j)/2) / 4^n (rotate by 45 degrees: two
    independent 1-D walks) -- all dyadic rationals, exact in binary floating point.  Pins Fo, the four neighbours and c0."""
    n, steps = 32, 7
    dx, dt = _grid(n)
    u = np.zeros((n, n))
    u[n // 2, n // 2] = 4.0 ** steps
    got = oracle.heat2d(u, steps, 1.0, dx, dt)
    want = np.zeros((n, n))
    for j in range(-steps, steps + 1):
        for i in range(-steps, steps + 1):
            if (steps + i + j) % 2 == 0 and abs(i + j) <= steps and abs(i - j) <= steps:
                want[n // 2 + j, n // 2 + i] = comb(steps, (steps + i + j) // 2) * comb(steps, (steps + i - j) // 2)
    assert np.array_equal(got, want)


def test_asymmetric_one_step_response_pins_the_index_order():
    """One step of a delta at Fo = 0.2 with distinct extents nx != ny: centre 1 - 4 Fo, the four neighbours Fo, and nothing
    else; a transposed index (i * ny + j) or a swapped extent shows up at once."""
    nx, ny = 12, 20
    dx = 1.0 / 16
    dt = 0.2 * dx * dx
    u = np.zeros((ny, nx))
    u[3, 10] = 1.0
    got = oracle.heat2d(u, 1, 1.0, dx, dt)
    want = np.zeros((ny, nx))
    want[3, 10] = 1 - 4 * 0.2
    for dj, di in ((0, 1), (0, -1), (1, 0), (-1, 0)):
        want[(3 + dj) % ny, (10 + di) % nx] = 0.2
    assert np.allclose(got, want, rtol=0, atol=1e-16)
    assert np.count_nonzero(got) == 5
    # periodic wrap in both directions, independently
    u = np.zeros((ny, nx))
    u[0, nx - 1] = 1.0
    got = oracle.heat2d(u, 1, 1.0, dx, dt)
    assert got[0, 0] == pytest.approx(0.2) and got[ny - 1, nx - 1] == pytest.approx(0.2) and got[1, nx - 1] == pytest.approx(0.2)


@pytest.mark.parametrize("kx,ky,Fo", [(1, 0, 0.25), (0, 3, 0.2), (2, 5, 0.1), (7, 7, 0.25)])
def test_separable_amplification_factor(kx, ky, Fo):
    """A product mode sin(2 pi kx x) cos(2 pi ky y) is an eigenvector of the periodic 5-point scheme:
    G = 1 - 4 Fo (sin^2(pi kx / nx) + sin^2(pi ky / ny))   (the 2-D form of north_star's 1 - 4 r sin^2(k dx / 2))."""
    nx, ny, steps = 64, 48, 25
    dx = 1.0 / nx
    dt = Fo * dx * dx
    x, y = np.arange(nx) / nx, np.arange(ny) / ny
    u0 = np.sin(2 * np.pi * kx * x + 0.3)[None, :] * np.cos(2 * np.pi * ky * y - 0.2)[:, None]
    G = 1 - 4 * Fo * (np.sin(np.pi * kx / nx) ** 2 + np.sin(np.pi * ky / ny) ** 2)
    got = oracle.heat2d(u0, steps, 1.0, dx, dt)
    assert np.max(np.abs(got - G ** steps * u0)) < 1e-13


def test_sum_is_conserved_uniform_is_fixed_and_max_principle():
    rng = np.random.default_rng(5)
    nx, ny = 40, 24
    dx = 1.0 / nx
    dt = 0.23 * dx * dx
    u0 = rng.uniform(-1, 1, (ny, nx))
    u = oracle.heat2d(u0, 50, 1.0, dx, dt)
    assert abs(u.sum() - u0.sum()) < 1e-12 * np.abs(u0).sum()
    assert u.max() <= u0.max() and u.min() >= u0.min() and np.ptp(u) < 0.5 * np.ptp(u0)
    c = np.full((ny, nx), 0.7)
    assert np.max(np.abs(oracle.heat2d(c, 9, 1.0, dx, dt) - 0.7)) < 1e-15


def test_transposition_commutes_with_stepping_bitwise_and_fp32_runs_in_fp32():
    """(uE + uW) + (uN + uS): exchanging the roles of x and y only commutes the outer addition."""
    rng = np.random.default_rng(6)
    u0 = rng.uniform(-1, 1, (24, 56)).astype(np.float32)
    dx = 1.0 / 64
    dt = 0.2 * dx * dx
    a = oracle.heat2d(u0, 17, 1.0, dx, dt)
    b = oracle.heat2d(np.ascontiguousarray(u0.T), 17, 1.0, dx, dt).T
    assert a.dtype == np.float32 and np.array_equal(a, b)
    d = oracle.heat2d(u0.astype(np.float64), 17, 1.0, dx, dt)
    assert 0 < np.max(np.abs(d - a)) < 1e-5


def test_field_uniform_in_y_follows_the_pinned_1d_oracle():
    """With no y dependence the scheme is (1 - 2 Fo) u + Fo (uE + uW): the 1-D FTCS of oracle.heat (pinned on its own)."""
    rng = np.random.default_rng(7)
    nx, ny = 64, 10
    dx = 1.0 / nx
    dt = 0.2 * dx * dx
    row = rng.uniform(-1, 1, nx)
    got = oracle.heat2d(np.tile(row, (ny, 1)), 30, 1.0, dx, dt)
    ref = oracle.heat(row[None, :], 30, 1.0, dx, dt)[0]
    assert np.max(np.abs(got - ref[None, :])) < 1e-14
    assert np.max(np.abs(got - got[0:1, :])) == 0.0


def test_shift_equivariance_bitwise():
    rng = np.random.default_rng(8)
    u0 = rng.uniform(-1, 1, (32, 32))
    dx = 1.0 / 32
    dt = 0.25 * dx * dx
    a = oracle.heat2d(np.roll(u0, (5, -9), axis=(0, 1)), 12, 1.0, dx, dt)
    assert np.array_equal(a, np.roll(oracle.heat2d(u0, 12, 1.0, dx, dt), (5, -9), axis=(0, 1)))
