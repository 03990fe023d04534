"""Pins of the insulated-ends heat oracle (the paper's own heat problem; Eq. 9 PAPER.md:266-269 with reading G7 of
DESIGN.md: the ghost value beyond an end is the adjacent interior value).  None of these re-types the oracle's loop."""
from fractions import Fraction

import numpy as np
import pytest

import oracle


def _grid(nx, r=0.25):
    dx = 1.0 / nx
    return dx, r * dx * dx


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("nx,nsteps,r", [(8, 5, 0.25), (64, 200, 0.25), (257, 333, 0.3), (1024, 100, 0.125)])
def test_equals_the_periodic_oracle_on_the_mirrored_rod_bitwise(dtype, nx, nsteps, r):
    """A rod with insulated ends is one half of a periodic ring of 2 nx points holding the rod and its mirror image: the ring's
    symmetry is preserved bit for bit (uR + uL is commutative), so the already-pinned periodic oracle decides every value."""
    rng = np.random.default_rng(1612)
    u = rng.uniform(-1, 1, nx).astype(dtype)
    dx, dt = _grid(nx, r)
    ring = np.concatenate([u, u[::-1]])
    ref = oracle.heat(ring, nsteps, 1.0, dx, dt)
    got = oracle.heat_insulated(u, nsteps, 1.0, dx, dt)
    assert np.array_equal(ref[:nx].view(np.uint8), got.view(np.uint8))
    assert np.array_equal(np.ascontiguousarray(ref[nx:][::-1]).view(np.uint8), got.view(np.uint8))


@pytest.mark.parametrize("k", [0, 1, 3, 17, 63])
def test_cosine_modes_decay_by_the_neumann_amplification_factor(k):
    """cos(k pi (i + 1/2) / n) are the eigenvectors of the FTCS operator with mirrored ghosts (DCT-II modes); the factor per step
    is G = 1 - 4 r sin^2(k pi / 2n) -- the Neumann counterpart of north_star's 1 - 4 r sin^2(k dx / 2)."""
    nx, r, nsteps = 64, 0.25, 300
    dx, dt = _grid(nx, r)
    i = np.arange(nx)
    u0 = np.cos(k * np.pi * (i + 0.5) / nx)
    G = 1.0 - 4.0 * r * np.sin(k * np.pi / (2 * nx)) ** 2
    got = oracle.heat_insulated(u0, nsteps, 1.0, dx, dt)
    assert np.max(np.abs(got - G ** nsteps * u0)) <= 1e-12


def test_hand_stepped_four_point_rod_is_exact():
    """nx = 4, r = 1/4, u0 = delta at the left end, three steps, by exact rational arithmetic with explicit ghost cells
    (every value is dyadic, so float equality is exact).  A transposed or missing ghost changes the end values."""
    r = Fraction(1, 4)
    u = [Fraction(1), Fraction(0), Fraction(0), Fraction(0)]
    for _ in range(3):
        g = [u[0]] + u + [u[-1]]                               # ghost = adjacent interior value at both ends
        u = [r * (g[j + 2] + g[j]) + (1 - 2 * r) * g[j + 1] for j in range(4)]
    dx, dt = _grid(4)
    got = oracle.heat_insulated(np.array([1.0, 0, 0, 0]), 3, 1.0, dx, dt)
    assert [Fraction(float(v)) for v in got] == u
    assert sum(u) == 1                                          # and the hand-stepped rod conserves the heat


def test_sum_is_conserved_uniform_is_fixed_and_the_ends_differ_from_periodic():
    nx = 128
    dx, dt = _grid(nx)
    rng = np.random.default_rng(2495)
    u0 = rng.uniform(0, 1, nx)
    u0[:8] += 5.0                                               # heat piled at the left end must not leak to the right end
    got = oracle.heat_insulated(u0, 500, 1.0, dx, dt)
    assert abs(got.sum() - u0.sum()) <= 1e-11 * u0.sum()
    assert got.min() >= u0.min() - 1e-15 and got.max() <= u0.max() + 1e-15
    assert np.array_equal(oracle.heat_insulated(np.full(nx, 0.75), 50, 1.0, dx, dt), np.full(nx, 0.75))
    per = oracle.heat(u0, 500, 1.0, dx, dt)
    assert abs(per[-1] - got[-1]) > 1e-3                        # the periodic ring leaks across the seam, the rod does not
