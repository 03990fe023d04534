"""Seeded synthetic workloads for the swept-rule hot path (inputs only).

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_1612_02495_b200/`).  It holds no arithmetic of the method: it only
builds initial arrays and the (nx, dx, dt, params) tuples that BASELINE.json's
five configs name, following the readings in SURVEY.md §8(c) S2, S8-S10, K1,
E3-E4 (restated in DESIGN.md "Input recipe").  Arrays are generated once on the
host in float64 with numpy `default_rng(seed)` and then cast to the run dtype;
the very same array is handed to the oracle and to the GPU, so the RNG can
never influence parity.

The paper itself never states its initial data ("initial
temperature gradient"; "periodic initial and boundary
conditions"); these inputs stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

HEAT, KS, EULER = 0, 1, 2
PROBLEM_NAMES = {HEAT: "heat", KS: "ks", EULER: "euler"}
PROBLEM_IDS = {v: k for k, v in PROBLEM_NAMES.items()}
# stencil radius per sub-step, sub-steps per timestep, fields per point (SURVEY §8 notation)
RADIUS = {HEAT: 1, KS: 2, EULER: 2}
STAGES = {HEAT: 1, KS: 2, EULER: 2}
NCOMP = {HEAT: 1, KS: 1, EULER: 3}

SEED_NOISE = 1612
SEED_MODES = 2495
KS_DX = math.pi / 4.0          # reading K1: dx = 32*pi/128 for every nx
KS_DT = 0.005
EULER_GAMMA = 1.4


@dataclass
class Workload:
    """One problem instance: everything `swept_create` and the oracle need."""
    problem: int
    nx: int
    dx: float
    dt: float
    u0: np.ndarray                 # float64, shape [ncomp, nx] (C-contiguous)
    alpha: float = 1.0             # heat only
    gamma: float = EULER_GAMMA     # Euler only
    nsteps: int = 0                # the config's step count (tests may run fewer)
    tile_width: int = 0            # the config's W if it names one
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def ncomp(self) -> int:
        return NCOMP[self.problem]

    def initial(self, dtype) -> np.ndarray:
        """Initial field cast to the run dtype, fresh copy, shape [ncomp, nx]."""
        return np.ascontiguousarray(self.u0.astype(dtype, copy=True))


def _is_pow2(n: int) -> bool:
    return n > 0 and (n & (n - 1)) == 0


# ----------------------------------------------------------------------------------------------
# heat (configs 1, 2, 5): x_i = i/nx, dx = 1/nx, alpha = 1, dt = r*dx*dx  (reading S2)
# ----------------------------------------------------------------------------------------------
def heat_grid(nx: int, r: float = 0.25, alpha: float = 1.0):
    dx = 1.0 / nx
    dt = r * dx * dx / alpha
    return dx, dt


def heat_config1(nx: int = 1024, seed: int = SEED_NOISE) -> Workload:
    """Config 1: u = sin(2 pi x) + 0.01 * U[-1,1] noise, 10 000 steps, W = 64."""
    dx, dt = heat_grid(nx)
    x = np.arange(nx, dtype=np.float64) / nx
    eta = np.random.default_rng(seed).uniform(-1.0, 1.0, nx)
    u0 = np.sin(2.0 * np.pi * x) + 0.01 * eta
    return Workload(HEAT, nx, dx, dt, u0[None, :], nsteps=10_000, tile_width=64, name="heat-config1")


def heat_config2(nx: int, seed: int = SEED_MODES) -> Workload:
    """Config 2: u = sum_{m=1..4} a_m sin(2 pi m x), a_m ~ U[0,1] (reading S9), 50 000 steps."""
    dx, dt = heat_grid(nx)
    x = np.arange(nx, dtype=np.float64) / nx
    a = np.random.default_rng(seed).uniform(0.0, 1.0, 4)
    u0 = np.zeros(nx)
    for m in range(1, 5):
        u0 += a[m - 1] * np.sin(2.0 * np.pi * m * x)
    return Workload(HEAT, nx, dx, dt, u0[None, :], nsteps=50_000, name="heat-config2")


def heat_noise(nx: int, seed: int = SEED_NOISE, r: float = 0.25, alpha: float = 1.0) -> Workload:
    """Grid-scale U[-1,1] noise: every step changes every value at O(1) (SURVEY §8(c) 'sensitive').  r = alpha dt / dx^2: with the
    configs' r = 1/4 every product of the update is exact in binary; any other r (and alpha != 1) makes rounding order matter."""
    dx, dt = heat_grid(nx, r, alpha)
    u0 = np.random.default_rng(seed).uniform(-1.0, 1.0, nx)
    return Workload(HEAT, nx, dx, dt, u0[None, :], alpha=alpha, name="heat-noise")


def heat_rod(nx: int, seed: int = SEED_NOISE, r: float = 0.25, alpha: float = 1.0) -> Workload:
    """The paper's heat problem: a rod with an initial temperature gradient and insulated ends -- a linear ramp
    3 -> 0 from the left end to the right end plus grid-scale U[-1,1] noise, so that every step changes every value and the
    two ends differ (a periodic ring would leak across the seam).  Used with boundary = insulated."""
    dx, dt = heat_grid(nx, r, alpha)
    u0 = 3.0 * (1.0 - (np.arange(nx) + 0.5) / nx) + np.random.default_rng(seed).uniform(-1.0, 1.0, nx)
    return Workload(HEAT, nx, dx, dt, u0[None, :], alpha=alpha, name="heat-rod")


# ----------------------------------------------------------------------------------------------
# Kuramoto-Sivashinsky (configs 3, 5): dx = pi/4 for every nx (reading K1), dt = 0.005
# ----------------------------------------------------------------------------------------------
def ks_config3(nx: int, seed: int = SEED_NOISE) -> Workload:
    """Config 3: u = cos(x/16)(1 + sin(x/16)) + 1e-3 N(0,1), x_i = i*dx, 20 000 steps."""
    x = np.arange(nx, dtype=np.float64) * KS_DX
    noise = np.random.default_rng(seed).standard_normal(nx)
    u0 = np.cos(x / 16.0) * (1.0 + np.sin(x / 16.0)) + 1e-3 * noise
    return Workload(KS, nx, KS_DX, KS_DT, u0[None, :], nsteps=20_000, name="ks-config3")


def ks_noise(nx: int, seed: int = SEED_NOISE, amp: float = 1.0) -> Workload:
    u0 = amp * np.random.default_rng(seed).uniform(-1.0, 1.0, nx)
    return Workload(KS, nx, KS_DX, KS_DT, u0[None, :], name="ks-noise")


# ----------------------------------------------------------------------------------------------
# Euler (configs 4, 5): [0,1), cell centres x_i = (i+1/2)/nx (reading E3), dt from CFL 0.5 at t=0 (E4)
# ----------------------------------------------------------------------------------------------
def euler_conserved(rho, vel, p, gamma: float = EULER_GAMMA) -> np.ndarray:
    """Primitive -> conserved (rho, m = rho u, E = p/(gamma-1) + rho u^2/2); an input conversion only."""
    rho = np.asarray(rho, dtype=np.float64)
    vel = np.asarray(vel, dtype=np.float64)
    p = np.asarray(p, dtype=np.float64)
    return np.stack([rho, rho * vel, p / (gamma - 1.0) + 0.5 * rho * vel * vel])


def euler_dt_cfl(rho, vel, p, dx: float, cfl: float = 0.5, gamma: float = EULER_GAMMA) -> float:
    smax = float(np.max(np.abs(vel) + np.sqrt(gamma * np.asarray(p) / np.asarray(rho))))
    return cfl * dx / smax


def euler_config4(nx: int) -> Workload:
    """Config 4: Sod states (1,0,1) on 0.25 <= x < 0.75, (0.125,0,0.1) elsewhere (mirrored => periodic)."""
    dx = 1.0 / nx
    x = (np.arange(nx, dtype=np.float64) + 0.5) / nx
    hi = (x >= 0.25) & (x < 0.75)
    rho = np.where(hi, 1.0, 0.125)
    vel = np.zeros(nx)
    p = np.where(hi, 1.0, 0.1)
    dt = euler_dt_cfl(rho, vel, p, dx)
    return Workload(EULER, nx, dx, dt, euler_conserved(rho, vel, p), nsteps=10_000, name="euler-config4")


# ----------------------------------------------------------------------------------------------
# config 5: smooth random Fourier series, 16 modes, amplitudes ~ k^-2 (reading S10)
# ----------------------------------------------------------------------------------------------
def fourier_series(nx: int, seed: int, nmodes: int = 16) -> np.ndarray:
    rng = np.random.default_rng(seed)
    A = rng.standard_normal(nmodes)
    B = rng.standard_normal(nmodes)
    xi = np.arange(nx, dtype=np.float64) / nx        # x / domain length
    s = np.zeros(nx)
    for k in range(1, nmodes + 1):
        s += (A[k - 1] * np.cos(2.0 * np.pi * k * xi) + B[k - 1] * np.sin(2.0 * np.pi * k * xi)) / (k * k)
    return s / np.max(np.abs(s))


def config5(problem: int, nx: int = 1 << 22) -> Workload:
    """Config 5 (stress/tuning): heat, KS or Euler on the 16-mode series, 100 000 steps."""
    if problem == HEAT:
        dx, dt = heat_grid(nx)
        return Workload(HEAT, nx, dx, dt, fourier_series(nx, SEED_MODES)[None, :], nsteps=100_000, name="heat-config5")
    if problem == KS:
        return Workload(KS, nx, KS_DX, KS_DT, fourier_series(nx, SEED_MODES)[None, :], nsteps=100_000, name="ks-config5")
    if problem == EULER:
        dx = 1.0 / nx
        rho = 1.0 + 0.2 * fourier_series(nx, SEED_MODES + 0)
        vel = 0.2 * fourier_series(nx, SEED_MODES + 1)
        p = 1.0 + 0.2 * fourier_series(nx, SEED_MODES + 2)
        dt = euler_dt_cfl(rho, vel, p, dx)
        return Workload(EULER, nx, dx, dt, euler_conserved(rho, vel, p), nsteps=100_000, name="euler-config5")
    raise ValueError(f"unknown problem {problem}")


def euler_noise(nx: int, seed: int = SEED_NOISE) -> Workload:
    """Positive grid-scale noise state for sensitive Euler parity runs (short runs only)."""
    rng = np.random.default_rng(seed)
    dx = 1.0 / nx
    rho = 1.0 + 0.3 * rng.uniform(-1.0, 1.0, nx)
    vel = 0.3 * rng.uniform(-1.0, 1.0, nx)
    p = 1.0 + 0.3 * rng.uniform(-1.0, 1.0, nx)
    dt = euler_dt_cfl(rho, vel, p, dx, cfl=0.25)
    return Workload(EULER, nx, dx, dt, euler_conserved(rho, vel, p), name="euler-noise")


def make(problem, nx: int, kind: str = "config") -> Workload:
    """Dispatch helper used by tests and bench: kind in {'config', 'noise', 'config5'}."""
    if isinstance(problem, str):
        problem = PROBLEM_IDS[problem]
    if not _is_pow2(nx):
        raise ValueError("nx must be a power of two (periodic index is `& (nx-1)`, PAPER.md:171)")
    if kind == "noise":
        return {HEAT: heat_noise, KS: ks_noise, EULER: euler_noise}[problem](nx)
    if kind == "config5":
        return config5(problem, nx)
    return {HEAT: heat_config2, KS: ks_config3, EULER: euler_config4}[problem](nx)


def steps_per_half_cycle(problem: int, tile_width: int) -> int:
    """L/S: full timesteps one swept half-cycle advances (SURVEY §8 notation)."""
    return tile_width // (2 * RADIUS[problem] * STAGES[problem])


# ----------------------------------------------------------------------------------------------
# 2-D heat: inputs only -- a seeded smooth field plus grid-scale noise on [0,1)^2
# ----------------------------------------------------------------------------------------------
def heat2d_grid(n: int, fo: float = 0.25):
    """dx = dy = 1/n, alpha = 1, dt = fo dx^2 (fo = 1/4 is the stability limit of the 5-point FTCS scheme)."""
    dx = 1.0 / n
    return dx, fo * dx * dx


def heat2d_field(nx: int, ny: int, seed: int = SEED_NOISE, noise: float = 1.0) -> np.ndarray:
    """sin(2 pi x) cos(4 pi y) + noise * U[-1,1] grid-scale noise, float64 [ny, nx]."""
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    smooth = np.sin(2 * np.pi * x)[None, :] * np.cos(4 * np.pi * y)[:, None]
    return np.ascontiguousarray(smooth + noise * np.random.default_rng(seed).uniform(-1.0, 1.0, (ny, nx)))
