"""Pins for the heat oracle (Eq. 2) -- closed forms and exact small cases, no GPU."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _heat(u, n, nx, r=0.25):
    dx = 1.0 / nx
    return oracle.heat(u, n, 1.0, dx, r * dx * dx)


def test_delta_response_is_pascal_row_exact():
    """nx=8, r=1/4, delta at i=1, 3 steps => 64 u = binomial row 6, wrapped (exact in binary)."""
    gold = np.loadtxt(os.path.join(GOLD, "heat_delta_nx8.txt"))
    for dt in (np.float64, np.float32):
        u0 = np.zeros((1, 8), dtype=dt)
        u0[0, 1] = 1
        u = _heat(u0, 3, 8)
        assert u.dtype == dt
        assert np.array_equal(64 * u[0], gold.astype(dt))


def test_delta_response_asymmetric_start_catches_transposed_neighbours():
    """One step from e_2 at r=0.3: (Fo, 1-2Fo, Fo) lands on i=1,2,3 only; wrap at the ends."""
    nx = 8
    u0 = np.zeros((1, nx))
    u0[0, 0] = 1.0
    u = _heat(u0, 1, nx, r=0.3)[0]
    Fo = 1.0 * (0.3 / 64) / (1 / 64)
    assert u[0] == pytest.approx(1 - 2 * Fo, rel=1e-15)
    assert u[1] == pytest.approx(Fo, rel=1e-15) and u[7] == pytest.approx(Fo, rel=1e-15)
    assert np.all(u[2:7] == 0)


@pytest.mark.parametrize("mode,n", [(1, 10_000), (3, 10_000), (17, 1_000)])
def test_single_mode_decays_by_amplification_factor(mode, n):
    """sin(k x) is an eigenvector of periodic FTCS with G = 1 - 4 r sin^2(k dx/2) (north_star)."""
    nx, r = 1024, 0.25
    x = np.arange(nx) / nx
    k = 2 * np.pi * mode
    u0 = np.sin(k * x)[None, :]
    G = 1.0 - 4.0 * r * np.sin(k * (1.0 / nx) / 2.0) ** 2
    u = _heat(u0, n, nx, r)
    assert 0.05 < G ** n < 0.95                       # a real decay, not yet in the rounding floor
    err = np.max(np.abs(u - G ** n * u0)) / np.max(np.abs(G ** n * u0))
    assert err < 1e-11


def test_amplification_factor_other_r_and_cosine_phase():
    nx, n, r = 256, 500, 0.4
    x = np.arange(nx) / nx
    u0 = np.cos(2 * np.pi * 5 * x + 0.3)[None, :]
    G = 1.0 - 4.0 * r * np.sin(2 * np.pi * 5 / nx / 2.0) ** 2
    u = _heat(u0, n, nx, r)
    assert np.max(np.abs(u - G ** n * u0)) < 1e-12


def test_nyquist_mode_annihilated_at_quarter():
    """(-1)^i has G = 1 - 4r = 0 at r = 1/4: exactly zero after one step."""
    for dt in (np.float64, np.float32):
        u0 = ((-1.0) ** np.arange(64)).astype(dt)[None, :]
        assert np.all(_heat(u0, 1, 64) == 0)


def test_uniform_fixed_and_sum_conserved_and_max_principle():
    nx = 512
    assert np.all(_heat(np.full((1, nx), 3.25), 100, nx) == 3.25)
    w = wl.heat_noise(nx, seed=7)
    u0 = w.initial(np.float64)
    u = oracle.heat(u0, 200, w.alpha, w.dx, w.dt)
    assert abs(u.sum() - u0.sum()) < 1e-11
    assert u.max() <= u0.max() and u.min() >= u0.min()
    assert np.max(np.abs(u)) < 0.5 * np.max(np.abs(u0))      # grid-scale noise really decays


def test_shift_equivariance_bitwise():
    w = wl.heat_noise(256, seed=3)
    u0 = w.initial(np.float32)
    a = oracle.heat(np.roll(u0, 37, axis=1), 50, w.alpha, w.dx, w.dt)
    b = np.roll(oracle.heat(u0, 50, w.alpha, w.dx, w.dt), 37, axis=1)
    assert np.array_equal(a, b)


def test_config1_scale_closed_form():
    """Config 1 without its noise: the mode-1 amplitude after 10 000 steps is G^n (probe value 0.9101698669...)."""
    w = wl.heat_config1()
    x = np.arange(w.nx) / w.nx
    u0 = np.sin(2 * np.pi * x)[None, :]
    G = 1.0 - np.sin(np.pi / w.nx) ** 2
    u = oracle.heat(u0, w.nsteps, w.alpha, w.dx, w.dt)
    assert G ** w.nsteps == pytest.approx(0.910169866907783, rel=1e-12)
    assert np.max(np.abs(u - G ** w.nsteps * u0)) < 1e-11


def test_zero_steps_identity_and_input_untouched():
    w = wl.heat_noise(64)
    u0 = w.initial(np.float64)
    keep = u0.copy()
    assert np.array_equal(oracle.heat(u0, 0, 1.0, w.dx, w.dt), keep)
    oracle.heat(u0, 5, 1.0, w.dx, w.dt)
    assert np.array_equal(u0, keep)
