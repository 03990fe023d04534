"""Pins for the Kuramoto-Sivashinsky oracle (Eq. 4, 15, 16 PAPER.md:64, 291, 295; sign reading G1)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import workloads as wl


def test_uniform_field_is_fixed_point():
    """With the -2u_i reading (G1) every difference of a constant vanishes."""
    u0 = np.full((1, 64), 1.375)
    assert np.array_equal(oracle.ks(u0, 25, wl.KS_DX, wl.KS_DT), u0)


def test_sum_conserved():
    """Every term of Eq. 4 telescopes on a periodic grid."""
    w = wl.ks_config3(1 << 12)
    u0 = w.initial(np.float64)
    u = oracle.ks(u0, 2000, w.dx, w.dt)
    assert np.isfinite(u).all()
    assert abs(u.mean() - u0.mean()) < 1e-14
    assert 1.0 < np.max(np.abs(u)) < 10.0            # stable and O(1) (reading K1)


@pytest.mark.parametrize("A,mode", [(0.0, 9), (0.7, 5), (-1.3, 20)])
def test_linearised_growth_factor(A, mode):
    """u = A + eps sin(kx): per step the perturbation is multiplied by 1 + z + z^2/2 (midpoint RK2),
    z = dt * ( -i A sin(k dx)/dx + s/dx^2 - s^2/dx^4 ),  s = 4 sin^2(k dx/2).
    Pins c1 (incl. the 1/4 and the sign of the nonlinear term through the phase speed A),
    c2, c4, the stencil weights (1,-2,1), (1,-4,6,-4,1), and both RK2 stages."""
    nx, n, eps = 128, 200, 1e-7
    dx, dt = wl.KS_DX, wl.KS_DT
    x = np.arange(nx) * dx
    k = 2 * np.pi * mode / (nx * dx)
    s = 4 * np.sin(k * dx / 2) ** 2
    z = dt * (-1j * A * np.sin(k * dx) / dx + s / dx ** 2 - s ** 2 / dx ** 4)
    G = 1 + z + z * z / 2
    u0 = (A + eps * np.sin(k * x))[None, :]
    u = oracle.ks(u0, n, dx, dt)
    expect = eps * np.imag(G ** n * np.exp(1j * k * x))
    got = u[0] - A
    assert np.max(np.abs(got - expect)) < 2e-6 * np.max(np.abs(expect))
    assert abs(abs(G) - 1) > 1e-4 or A != 0       # the test is not vacuous


def test_shift_equivariance_bitwise():
    w = wl.ks_noise(256, seed=11)
    u0 = w.initial(np.float64)
    a = oracle.ks(np.roll(u0, 101, axis=1), 40, w.dx, w.dt)
    b = np.roll(oracle.ks(u0, 40, w.dx, w.dt), 101, axis=1)
    assert np.array_equal(a, b)


def test_reflection_symmetry_to_rounding():
    """x -> -x, u -> -u maps solutions to solutions (odd nonlinear term)."""
    w = wl.ks_noise(128, seed=5)
    u0 = w.initial(np.float64)
    a = oracle.ks(u0, 200, w.dx, w.dt)
    b = -oracle.ks(-u0[:, ::-1].copy(), 200, w.dx, w.dt)[:, ::-1]
    assert np.max(np.abs(a - b)) < 1e-12 * np.max(np.abs(a))


def _ks_exact_rational(u, dx, dt, nsteps):
    """Eq. 4 + 15 + 16 evaluated literally (with divisions, no stored reciprocals) in exact rationals."""
    n = len(u)

    def f(v):
        out = []
        for i in range(n):
            vm2, vm1, v0, vp1, vp2 = v[(i - 2) % n], v[(i - 1) % n], v[i], v[(i + 1) % n], v[(i + 2) % n]
            adv = (vp1 ** 2 - vm1 ** 2) / (4 * dx)
            d2 = (vp1 + vm1 - 2 * v0) / dx ** 2
            d4 = (vp2 - 4 * vp1 + 6 * v0 - 4 * vm1 + vm2) / dx ** 4
            out.append(-(adv + d2 + d4))
        return out

    for _ in range(nsteps):
        fu = f(u)
        half = [u[i] + dt / 2 * fu[i] for i in range(n)]
        fh = f(half)
        u = [u[i] + dt * fh[i] for i in range(n)]
    return u


def test_tiny_grid_against_exact_rational_hand_stepping():
    """nx=8, 3 steps (north_star 'brute-force hand-stepped tiny grids'), dyadic dx, dt so inputs are exact."""
    rng = np.random.default_rng(8)
    u0 = np.round(rng.uniform(-1, 1, 8) * 64) / 64
    dx, dt = 0.75, 1.0 / 128
    exact = _ks_exact_rational([Fraction(float(v)) for v in u0], Fraction(dx), Fraction(dt), 3)
    exact = np.array([float(v) for v in exact])
    u = oracle.ks(u0[None, :], 3, dx, dt)[0]
    assert np.max(np.abs(u - exact)) < 8 * np.finfo(np.float64).eps * np.max(np.abs(exact))
    u32 = oracle.ks(u0[None, :].astype(np.float32), 3, dx, dt)[0]
    assert u32.dtype == np.float32
    assert np.max(np.abs(u32 - exact)) < 16 * np.finfo(np.float32).eps * np.max(np.abs(exact))


def test_literal_config3_spacing_is_unstable_reading_K1():
    """Documents reading K1: [0,32pi) at nx=2^14 with dt=0.005 blows up within a handful of steps."""
    nx = 1 << 14
    dx = 32 * np.pi / nx
    x = np.arange(nx) * dx
    u0 = (np.cos(x / 16) * (1 + np.sin(x / 16)) + 1e-3 * np.random.default_rng(1612).standard_normal(nx))[None, :]
    with np.errstate(all="ignore"):
        u = oracle.ks(u0, 6, dx, 0.005)
    assert not np.isfinite(u).all()
