"""Pins for the Euler oracle (BASELINE.json config 4; MUSCL/minmod/Rusanov midpoint, readings E1-E5)."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
G = wl.EULER_GAMMA


def _prim(U, gamma=G):
    rho, m, E = U
    u = m / rho
    return rho, u, (gamma - 1) * (E - 0.5 * m * u)


def test_uniform_state_is_fixed_point_exactly():
    U0 = wl.euler_conserved(np.full(32, 0.9), np.full(32, 0.4), np.full(32, 1.7))
    U = oracle.euler(U0, 20, G, 1 / 32, 0.2 / 32)
    assert np.array_equal(U, U0)


def test_conservation_and_positivity_sod():
    w = wl.euler_config4(1024)
    U0 = w.initial(np.float64)
    U = oracle.euler(U0, 2000, w.gamma, w.dx, w.dt)          # raises if rho or p go non-positive
    s0, s1 = U0.sum(axis=1), U.sum(axis=1)
    assert abs(s1[0] - s0[0]) < 1e-13 * abs(s0[0])
    assert abs(s1[2] - s0[2]) < 1e-13 * abs(s0[2])
    assert abs(s1[1]) < 1e-11                                   # total momentum stays 0 (mirror symmetry)
    rho, u, p = _prim(U)
    assert rho.min() > 0 and p.min() > 0
    assert np.abs(u).max() > 0.5                                # waves really moved


def test_conservation_noise_state():
    w = wl.euler_noise(512, seed=2)
    U0 = w.initial(np.float64)
    U = oracle.euler(U0, 300, w.gamma, w.dx, w.dt)
    for k in range(3):
        assert abs(U[k].sum() - U0[k].sum()) < 1e-12 * np.abs(U0[k]).sum()
    assert np.max(np.abs(U - U0)) > 0.05


def test_mirror_symmetry():
    """Cell-centred grid, high state on [1/4, 3/4): rho, E even and m odd about x = 1/2 (reading E3)."""
    w = wl.euler_config4(512)
    U = oracle.euler(w.initial(np.float64), 600, w.gamma, w.dx, w.dt)
    assert np.max(np.abs(U[0] - U[0][::-1])) < 1e-12
    assert np.max(np.abs(U[2] - U[2][::-1])) < 1e-12
    assert np.max(np.abs(U[1] + U[1][::-1])) < 1e-12


def _sod_star(gamma=G, L=(1.0, 0.0, 1.0), R=(0.125, 0.0, 0.1)):
    """Exact Riemann solver for the star region: Newton iteration on the pressure function."""
    rl, ul, pl = L
    rr, ur, pr = R
    cl, cr = np.sqrt(gamma * pl / rl), np.sqrt(gamma * pr / rr)

    def fk(p, rk, pk, ck):
        if p > pk:      # shock
            A, B = 2 / ((gamma + 1) * rk), (gamma - 1) / (gamma + 1) * pk
            f = (p - pk) * np.sqrt(A / (p + B))
            df = np.sqrt(A / (p + B)) * (1 - (p - pk) / (2 * (B + p)))
        else:           # rarefaction
            f = 2 * ck / (gamma - 1) * ((p / pk) ** ((gamma - 1) / (2 * gamma)) - 1)
            df = 1 / (rk * ck) * (p / pk) ** (-(gamma + 1) / (2 * gamma))
        return f, df

    p = 0.5 * (pl + pr)
    for _ in range(50):
        fl, dfl = fk(p, rl, pl, cl)
        fr, dfr = fk(p, rr, pr, cr)
        p_new = p - (fl + fr + ur - ul) / (dfl + dfr)
        if abs(p_new - p) < 1e-14:
            p = p_new
            break
        p = p_new
    u = 0.5 * (ul + ur) + 0.5 * (fk(p, rr, pr, cr)[0] - fk(p, rl, pl, cl)[0])
    rsl = rl * (p / pl) ** (1 / gamma)                                             # behind the rarefaction
    rsr = rr * ((p / pr + (gamma - 1) / (gamma + 1)) / ((gamma - 1) / (gamma + 1) * p / pr + 1))  # behind the shock
    return p, u, rsl, rsr


def test_exact_riemann_solver_reproduces_textbook_sod_values():
    gold = dict(line.split()[:2] for line in open(os.path.join(GOLD, "sod_star_state.txt")) if not line.startswith("#"))
    p, u, rsl, rsr = _sod_star()
    assert p == pytest.approx(float(gold["p_star"]), abs=1e-5)
    assert u == pytest.approx(float(gold["u_star"]), abs=1e-5)
    assert rsl == pytest.approx(float(gold["rho_star_L"]), abs=1e-5)
    assert rsr == pytest.approx(float(gold["rho_star_R"]), abs=1e-5)


def test_sod_star_states_before_the_mirrored_waves_meet():
    """At t = 0.1 (< 0.14) each half of the mirrored tube is the textbook Sod solution."""
    nx = 4096
    w = wl.euler_config4(nx)
    n = int(round(0.1 / w.dt))
    t = n * w.dt
    U = oracle.euler(w.initial(np.float64), n, w.gamma, w.dx, w.dt)
    rho, u, p = _prim(U)
    ps, us, rsl, rsr = _sod_star()
    x = (np.arange(nx) + 0.5) / nx
    cs = np.sqrt(G * ps / rsl)
    tail, contact = 0.75 + (us - cs) * t, 0.75 + us * t
    shock = 0.75 + t * np.sqrt(G * 0.1 / 0.125) * np.sqrt((G + 1) / (2 * G) * ps / 0.1 + (G - 1) / (2 * G))
    i1 = np.argmin(np.abs(x - 0.5 * (tail + contact)))
    i2 = np.argmin(np.abs(x - 0.5 * (contact + shock)))
    assert rho[i1] == pytest.approx(rsl, abs=1e-3) and u[i1] == pytest.approx(us, abs=1e-3) and p[i1] == pytest.approx(ps, abs=1e-3)
    assert rho[i2] == pytest.approx(rsr, abs=1e-3) and u[i2] == pytest.approx(us, abs=1e-3) and p[i2] == pytest.approx(ps, abs=1e-3)
    # mirrored copy at x = 0.25 moves the other way
    j1 = nx - 1 - i1
    assert rho[j1] == pytest.approx(rsl, abs=1e-3) and u[j1] == pytest.approx(-us, abs=1e-3)
    # undisturbed states away from the waves
    assert rho[nx // 2] == 1.0 and rho[0] == 0.125


def _euler_numpy_step(U, gamma, lam):
    """Independent second evaluation: vectorised np.roll form of the textbook formulas (no fma order)."""

    def minmod(a, b):
        return np.where(a * b > 0, np.where(np.abs(a) < np.abs(b), a, b), 0.0)

    def flux(W):
        rho, m, E = W
        u = m / rho
        p = (gamma - 1) * (E - 0.5 * m * u)
        return np.stack([m, m * u + p, (E + p) * u]), np.abs(u) + np.sqrt(gamma * p / rho)

    def rhs(W):
        sig = minmod(W - np.roll(W, 1, axis=1), np.roll(W, -1, axis=1) - W)
        WL = W + 0.5 * sig
        WR = np.roll(W - 0.5 * sig, -1, axis=1)
        fL, sL = flux(WL)
        fR, sR = flux(WR)
        F = 0.5 * (fL + fR) - 0.5 * np.maximum(sL, sR) * (WR - WL)      # F_{i+1/2}
        return F - np.roll(F, 1, axis=1)

    Us = U - 0.5 * lam * rhs(U)
    return U - lam * rhs(Us)


@pytest.mark.parametrize("nx,n", [(8, 3), (64, 40)])
def test_tiny_grid_against_independent_evaluation(nx, n):
    rng = np.random.default_rng(nx)
    U0 = wl.euler_conserved(1 + 0.4 * rng.uniform(-1, 1, nx), 0.5 * rng.uniform(-1, 1, nx), 1 + 0.4 * rng.uniform(-1, 1, nx))
    dx = 1.0 / nx
    dt = 0.2 * dx
    V = U0.copy()
    for _ in range(n):
        V = _euler_numpy_step(V, G, dt / dx)
    U = oracle.euler(U0, n, G, dx, dt)
    assert np.max(np.abs(U - V)) < 1e-13 * np.max(np.abs(V)) * n
    assert np.max(np.abs(U - U0)) > 1e-3


def test_shift_equivariance_bitwise_and_fp32_runs_in_fp32():
    w = wl.euler_noise(128, seed=9)
    U0 = w.initial(np.float32)
    a = oracle.euler(np.roll(U0, 45, axis=1), 30, w.gamma, w.dx, w.dt)
    b = np.roll(oracle.euler(U0, 30, w.gamma, w.dx, w.dt), 45, axis=1)
    assert a.dtype == np.float32 and np.array_equal(a, b)
    d = oracle.euler(w.initial(np.float64), 30, w.gamma, w.dx, w.dt)
    assert 0 < np.max(np.abs(np.roll(d, 45, axis=1) - b)) < 1e-4


def test_positivity_flag_raises():
    w = wl.euler_config4(256)
    with pytest.raises(FloatingPointError):
        oracle.euler(w.initial(np.float64), 200, w.gamma, w.dx, 4.0 * w.dt)   # CFL 2: must break


# ------------------------------------------------------------------------------------------------------------------
# Pins for the SECOND-ORDER parts of the scheme (BASELINE.json config 4: "second-order finite volume with MUSCL
# reconstruction, minmod limiter ... predictor-corrector in time"): expected values come from the exact solution of the
# PDE and from the total-variation-diminishing property of a minmod-limited scheme, not from a second typing of the
# formulas.  `euler` is the stepping routine under test, so that test_mutants_of_the_oracle_fail_the_second_order_pins
# can run the same checks on deliberately broken builds of oracle/schemes.inc.
# ------------------------------------------------------------------------------------------------------------------
def _l1_errors_smooth_density_wave(euler, sizes=(64, 128, 256, 512), T=0.25, cfl=0.4):
    """A density wave carried at constant velocity and pressure is an exact solution of the Euler equations:
    rho(x, t) = rho0(x - u t), u = p = 1.  Returns the L1 error of the cell values at time T for each grid size."""
    errs = []
    for nx in sizes:
        dx = 1.0 / nx
        x = (np.arange(nx) + 0.5) * dx
        smax = 1.0 + np.sqrt(G * 1.0 / 0.8)                       # |u| + c at the density minimum
        n = int(np.ceil(T / (cfl * dx / smax)))
        dt = T / n
        U0 = wl.euler_conserved(1 + 0.2 * np.sin(2 * np.pi * x), np.ones(nx), np.ones(nx))
        rho = euler(U0, n, G, dx, dt)[0]
        errs.append(float(np.mean(np.abs(rho - (1 + 0.2 * np.sin(2 * np.pi * (x - T)))))))
    return errs


def _check_second_order(euler):
    errs = _l1_errors_smooth_density_wave(euler)
    ratios = [a / b for a, b in zip(errs, errs[1:])]
    assert errs[-1] < 1e-4, errs
    # second order in space AND time: the error falls by ~4 per halving of dx with dt ~ dx (minmod clips the two
    # extrema of the sine, which costs a little: 3.5-3.8 observed); a first-order reconstruction or a predictor that
    # is not a half step gives ~2
    assert all(r >= 3.4 for r in ratios), (errs, ratios)


def _check_tvd_contact(euler, nx=256, nsteps=400):
    """A square density pulse carried at constant u = p = 1 is a pure contact: the scheme reduces to scalar advection
    of rho, for which minmod-limited MUSCL creates no new extrema and does not increase the total variation."""
    dx = 1.0 / nx
    x = (np.arange(nx) + 0.5) * dx
    rho0 = np.where((x >= 0.25) & (x < 0.5), 2.0, 1.0)
    dt = 0.5 * dx / (1.0 + np.sqrt(G * 1.0 / 1.0))                 # the config's CFL 0.5 at the initial state
    U = wl.euler_conserved(rho0, np.ones(nx), np.ones(nx))
    tv = lambda r: float(np.sum(np.abs(np.roll(r, -1) - r)))
    tv_prev, eps = tv(rho0), 1e-12
    for _ in range(nsteps // 20):
        U = euler(U, 20, G, dx, dt)
        rho = U[0]
        assert rho.min() >= 1.0 - eps and rho.max() <= 2.0 + eps, (rho.min(), rho.max())
        assert tv(rho) <= tv_prev + eps, (tv(rho), tv_prev)
        tv_prev = tv(rho)
    # u and p stay constant across a contact
    _, u, p = _prim(U)
    assert np.max(np.abs(u - 1)) < 1e-12 and np.max(np.abs(p - 1)) < 1e-12
    # and the pulse is still a pulse (the limiter did not flatten it into first-order mush): second-order MUSCL keeps
    # the plateau value at the pulse centre after 400 steps, a first-order scheme has already eroded it
    assert rho.max() > 1.999


def _oracle_euler(U0, n, gamma, dx, dt):
    return oracle.euler(U0, n, gamma, dx, dt)


def test_second_order_accuracy_on_a_smooth_density_wave():
    _check_second_order(_oracle_euler)


def test_minmod_limiter_is_tvd_on_a_square_contact():
    _check_tvd_contact(_oracle_euler)


def _check_rusanov_speed(euler):
    """Which side's signal speed the Rusanov dissipation takes.  Semi-discrete limit: for dt -> 0 the predictor state tends to U^m, so
    one step changes cell i by -lambda (F_{i+1/2}(U^m) - F_{i-1/2}(U^m)) + O(lambda^2).  Datum: two constant states at rest on 8 cells
    (every minmod slope is zero: a cell next to the jump has one zero difference), gamma = 2 so that c^2 = 2 p / rho is 1 on one side
    and 4 on the other: |u| + c = 1 and 2 exactly, a = max = 2.  At the jump face f = (0, p, 0) on both sides, so by the definition
    of the flux, F = (f_L + f_R)/2 - (a/2)(U_R - U_L) = (-(a/2) [rho], (p_L + p_R)/2, -(a/2) [E]) with E = p / (gamma - 1) = p; the
    faces inside a state carry (0, p, 0).  Expected change of the cells beside the jump, in units of lambda, with a = 2:
    rho +-1, m -+(9/4 - p_own), E +-7/2.  With a = min = 1 the density and energy changes halve.  Both orientations of the jump are on
    the periodic grid (faces 3|4 and 7|0), so taking one fixed side's speed fails as well."""
    gamma, lam = 2.0, 1e-6
    rho = np.array([1.0] * 4 + [2.0] * 4)
    p = np.array([0.5] * 4 + [4.0] * 4)                      # c = sqrt(2 p / rho) = 1 | 2
    U0 = np.stack([rho, np.zeros(8), p / (gamma - 1.0)])
    U1 = euler(U0, 1, gamma, 1.0, lam)
    d = (U1 - U0) / lam
    a = 2.0
    drho, dE, pm = 0.5 * a * (2.0 - 1.0), 0.5 * a * (4.0 - 0.5), 0.5 * (0.5 + 4.0)
    want = np.zeros((3, 8))
    #            cell 0 (face 7|0)   cell 3 (face 3|4)   cell 4 (face 3|4)   cell 7 (face 7|0)
    want[0, [0, 3, 4, 7]] = [+drho, +drho, -drho, -drho]
    want[1, [0, 3, 4, 7]] = [-(0.5 - pm), -(pm - 0.5), -(4.0 - pm), -(pm - 4.0)]
    want[2, [0, 3, 4, 7]] = [+dE, +dE, -dE, -dE]
    assert np.max(np.abs(d - want)) < 1e-4, (d, want)


def test_rusanov_takes_the_larger_signal_speed():
    _check_rusanov_speed(_oracle_euler)


# name -> (text in oracle/schemes.inc, replacement, the pin that must catch it)
MUTANTS = {
    "first-order (sigma = 0)": ("if (p > (REAL)0.0) return (R_FABS(a) < R_FABS(b)) ? a : b;", "if (p > (REAL)0.0) return (REAL)0.0;", "order"),
    "maxmod (|a| > |b|)": ("(R_FABS(a) < R_FABS(b)) ? a : b", "(R_FABS(a) > R_FABS(b)) ? a : b", "tvd"),
    "unlimited central slope": ("if (p > (REAL)0.0) return (R_FABS(a) < R_FABS(b)) ? a : b;\n    return (REAL)0.0;",
                                "return (REAL)0.5 * (a + b);", "tvd"),
    "full-step predictor (lambda for lambda/2)": ("FN(euler_stage)(U, U, Us, nx, lamh, gamma, gm1)", "FN(euler_stage)(U, U, Us, nx, lam, gamma, gm1)", "order"),
    "forward Euler (corrector from U^m)": ("FN(euler_stage)(Us, U, Un, nx, lam, gamma, gm1)", "FN(euler_stage)(U, U, Un, nx, lam, gamma, gm1)", "order"),
    "face states of the wrong sign": ("R_FMA((REAL)-0.5, sp, w[ip])", "R_FMA((REAL)0.5, sp, w[ip])", "order"),
    "Rusanov speed: the smaller side": ("const REAL a = R_FMAX(sL, sR);", "const REAL a = (sL < sR) ? sL : sR;", "speed"),
    "Rusanov speed: the left side only": ("const REAL a = R_FMAX(sL, sR);", "const REAL a = sL;", "speed"),
    "Rusanov speed: the mean of the sides": ("const REAL a = R_FMAX(sL, sR);", "const REAL a = (REAL)0.5 * (sL + sR);", "speed"),
}
PINS = {"order": lambda f: _check_second_order(f), "tvd": lambda f: _check_tvd_contact(f), "speed": lambda f: _check_rusanov_speed(f)}


@pytest.mark.parametrize("name", list(MUTANTS))
def test_mutants_of_the_oracle_fail_the_second_order_pins(name, tmp_path):
    """The pins above must FAIL for the plausible mistakes they exist to catch: each mutant is oracle/schemes.inc with
    one line changed, built into a scratch library (oracle/ itself is untouched)."""
    import ctypes
    import shutil
    import subprocess
    from oracle import build as obuild
    old, new, pin = MUTANTS[name]
    src = open(os.path.join(obuild.HERE, "schemes.inc")).read()
    assert src.count(old) == 1, f"mutation site not found exactly once: {old!r}"
    (tmp_path / "schemes.inc").write_text(src.replace(old, new))
    for f in os.listdir(obuild.HERE):          # every other source of the oracle library, unchanged
        if f.endswith((".c", ".inc", ".h")) and f != "schemes.inc":
            shutil.copy(os.path.join(obuild.HERE, f), tmp_path / f)
    so = tmp_path / "libmutant.so"
    subprocess.run(["gcc", *obuild.CFLAGS, "-o", str(so), "swept_oracle.c", "-lm"], check=True, cwd=tmp_path)
    L = ctypes.CDLL(str(so))
    L.oracle_euler_f64.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.c_long, ctypes.c_long, ctypes.c_double, ctypes.c_double, ctypes.c_double]
    L.oracle_euler_f64.restype = ctypes.c_int

    def mutant(U0, n, gamma, dx, dt):
        a = np.array(U0, dtype=np.float64, copy=True, order="C")
        rc = L.oracle_euler_f64(a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), a.shape[1], int(n), float(gamma), float(dx), float(dt))
        assert rc >= 0
        return a

    with pytest.raises(AssertionError):
        PINS[pin](mutant)
