"""-m "not gpu": the swept geometry and the host driver's launch plan, pinned to the
numbers the paper prints (tests/golden/paper_geometry.txt) and to a plain-Python model of the swept rule.

The model below restates PAPER.md:82-98, 102, 114 in the in-place staircase form of row A4: two flat rows R0 (even
tiers) and R1 (odd tiers); a kernel of mode up / diamond / down loads R0 on [0,W) and R1 on [-h, W+h) of its tile,
advances the tiers its mode prescribes with a plain periodic stencil, and stores R0 on [0,W), R1 on [h, W-h).  It is
executed on the launch list `swept_plan` returns -- the very list `swept_run` enqueues -- and must reproduce naive
stepping exactly (integer-valued stencils, so equality is exact), with every (point, tier) updated exactly once.
"""
import os

import numpy as np
import pytest

import paper_1612_02495_b200 as sw

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_geometry.txt")


def _golden():
    out = {}
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = int(line[1])
    return out


# ---- closed forms -----------------------------------------------------------------------
def up_updates(W, h):
    L = W // (2 * h)
    return (L - 1) * W // 2


def down_updates(W, h):
    L = W // (2 * h)
    return (L + 1) * W // 2


def diamond_updates(W, h):
    return (W // (2 * h)) * W


def test_paper_geometry_numbers():
    g = _golden()
    n, h = 512, 1
    # a full triangle (tier 0 included) for n = 512 holds 65 792 values = 514 kB in double
    tri = sum(n - 2 * h * t for t in range(n // (2 * h)))
    assert tri == g["triangle_values_n512"] == n + up_updates(n, h)
    assert 8 * tri == g["triangle_bytes_n512_fp64"]
    # the two-row matrix holds 2(n+2) values
    assert 2 * (n + 2 * h) == g["two_row_values_n512"]
    # a full cycle (two half-cycles) advances n timesteps for the heat scheme
    assert 2 * sw.steps_per_half_cycle(sw.HEAT, n) == n      # PAPER.md:98 "advance by n timesteps with two ... global memory accesses": n/2 per half-cycle
    # a 32-point node gives four KS timesteps per (half-)cycle, "which only reduces instances of communication
    # by 1/8": one global exchange per L = 8 sub-timesteps = 4 two-stage timesteps
    assert sw.steps_per_half_cycle(sw.KS, 32) == g["ks_steps_per_cycle_n32"]
    assert 32 // (2 * sw.problem_info(sw.KS)["radius"]) == 8


def test_triangle_counts_sum_to_whole_tiers():
    for h in (1, 2):
        for W in (8, 32, 64, 512, 1024):
            L = W // (2 * h)
            assert up_updates(W, h) + down_updates(W, h) == diamond_updates(W, h) == L * W
            assert up_updates(W, h) == sum(W - 2 * h * t for t in range(1, L))
            assert down_updates(W, h) == sum(2 * h * t for t in range(1, L + 1))


# ---- plain-Python model of the swept rule on the staircase rows ---------------------------------------------------
class Model:
    """Integer stencil `new[x] = sum_k c_k * prev[x+k]` (radius h); S = 2 makes even tiers accumulate onto the value two
    tiers below (the paper's RK2 structure, Fig. 5 `+=`), odd tiers overwrite."""

    def __init__(self, nx, h, S, u0):
        self.nx, self.h, self.S = nx, h, S
        self.R = [np.array(u0, dtype=object), np.zeros(nx, dtype=object)]
        self.coef = {1: (1, 2, 1), 2: (1, -3, 5, 2, -1)}[h]
        self.count = np.zeros(nx, dtype=np.int64)      # tier of the newest value held for every point (checked at the end)
        self.updates = 0

    def point(self, win, base, odd):
        v = sum(c * x for c, x in zip(self.coef, win))
        if self.S == 2 and not odd:
            return base + 3 * v
        return v

    def naive(self, nsteps):
        a = self.R[0].copy()
        nx, h = self.nx, self.h
        for _ in range(nsteps):
            if self.S == 1:
                a = np.array([self.point([a[(i + k) % nx] for k in range(-h, h + 1)], None, True) for i in range(nx)], dtype=object)
            else:
                p = np.array([self.point([a[(i + k) % nx] for k in range(-h, h + 1)], None, True) for i in range(nx)], dtype=object)
                a = np.array([self.point([p[(i + k) % nx] for k in range(-h, h + 1)], a[i], False) for i in range(nx)], dtype=object)
        return a

    def tile(self, mode, W, g0):
        nx, h = self.nx, self.h
        L, c = W // (2 * h), W // 2
        row = [{x: self.R[0][(g0 + x) % nx] for x in range(W)}, {}]
        if mode != "up":
            row[1] = {x: self.R[1][(g0 + x) % nx] for x in range(-h, W + h)}
        spans = []
        if mode != "up":
            spans += [(t, c - h * t, c + h * t) for t in range(1, L + 1)]
        if mode != "down":
            spans += [(t, h * t, W - h * t) for t in range(1, L)]
        for t, lo, hi in spans:
            src, dst = row[(t - 1) & 1], row[t & 1]
            new = {x: self.point([src[x + k] for k in range(-h, h + 1)], row[0].get(x), bool(t & 1)) for x in range(lo, hi)}
            dst.update(new)
            self.updates += hi - lo
        return row

    def tile_window(self, W, g0, lo, hi):
        """One diamond tile restricted to the tiers lo < t <= hi of its 2L - 1 (t <= L: the expanding part; the ring kernel's
        per-phase window, swept_ring.cuh).  (0, L] is "down", (L, 2L - 1] is "up", (0, 2L - 1] the whole diamond."""
        nx, h = self.nx, self.h
        L, c = W // (2 * h), W // 2
        row = [{x: self.R[0][(g0 + x) % nx] for x in range(W)}, {x: self.R[1][(g0 + x) % nx] for x in range(-h, W + h)}]
        spans = [(t, c - h * t, c + h * t) for t in range(1, L + 1)] + [(L + t, h * t, W - h * t) for t in range(1, L)]
        for t, a, b in spans:
            if not (lo < t <= hi):
                continue
            src, dst = row[(t - 1) & 1], row[t & 1]
            new = {x: self.point([src[x + k] for k in range(-h, h + 1)], row[0].get(x), bool(t & 1)) for x in range(a, b)}
            dst.update(new)
            self.updates += b - a
        return row

    def ring(self, W, q, r):
        """SWEPT_LAUNCH_RING: q half-cycles and r remainder timesteps in one sweep.  Phase p runs the tiers (lo, hi] of every
        diamond of its alignment: lo = L in phase 0 (the flat field is tier L of the first diamonds), hi = L + rt in phase q and
        rt in the extra phase q + 1, rt = S r (the truncated closing cycle).  The flat result is tier rt of the phase-(q+1) tiles
        where they reach it and tier L + rt of the phase-q tiles elsewhere: both have the parity of rt."""
        nx, h = self.nx, self.h
        L, rt = W // (2 * h), self.S * r
        assert 0 <= rt < L
        nph = q + 1 + (1 if rt else 0)
        for p in range(nph):
            lo = L if p == 0 else 0
            hi = 2 * L - 1 if p < q else (L + rt if p == q else rt)
            offset = W // 2 if p & 1 else 0
            rows = [self.tile_window(W, t * W + offset, lo, hi) for t in range(nx // W)]
            for t, row in enumerate(rows):
                g0 = t * W + offset
                for x in range(W):
                    self.R[0][(g0 + x) % nx] = row[0][x]
                for x in range(h, W - h):
                    self.R[1][(g0 + x) % nx] = row[1][x]
        self.R[0] = self.R[rt & 1].copy()

    def launch(self, mode, W, offset):
        nx, h = self.nx, self.h
        rows = [self.tile(mode, W, t * W + offset) for t in range(nx // W)]     # all tiles read before any writes ...
        for t, row in enumerate(rows):                                           # ... (snapshot semantics; A4 shows in-place is equal)
            g0 = t * W + offset
            for x in range(W):
                self.R[0][(g0 + x) % nx] = row[0][x]
            if mode != "down":
                for x in range(h, W - h):
                    self.R[1][(g0 + x) % nx] = row[1][x]

    def classic(self, nsteps):
        self.R[0] = self.naive(nsteps)
        self.updates += nsteps * self.S * self.nx

    def run_plan(self, plan):
        for kind, W, offset, count in plan:
            if kind == sw.LAUNCH_CLASSIC:
                self.classic(count)
            elif kind == sw.LAUNCH_UP:
                self.launch("up", W, offset)
            elif kind == sw.LAUNCH_DOWN:
                self.launch("down", W, offset)
            elif kind == sw.LAUNCH_DIAMOND:
                for k in range(count):
                    self.launch("diamond", W, offset if k % 2 == 0 else (0 if offset else W // 2))
            elif kind == sw.LAUNCH_RING or (kind == sw.LAUNCH_BAND and (offset or not count)):
                self.ring(W, count, offset)                      # the whole run in one launch, remainder as a truncated closing cycle
            elif kind in (sw.LAUNCH_CHAIN, sw.LAUNCH_BAND):      # the same phases in one launch (tile flags / streaming bands)
                for p in range(count + 1):
                    self.launch("up" if p == 0 else ("down" if p == count else "diamond"), W, W // 2 if p & 1 else 0)
            else:
                raise AssertionError(kind)


CASES = [
    # problem, nx, W, nsteps
    (sw.HEAT, 64, 16, 8 * 3),            # 3 half-cycles, no remainder: closes on the shifted alignment
    (sw.HEAT, 64, 16, 8 * 4 + 7),        # remainder 7 = 4 + 2 + 1 classic
    (sw.HEAT, 32, 32, 16 * 2 + 5),       # single tile wrapping onto itself
    (sw.HEAT, 64, 8, 3),                 # fewer steps than one half-cycle: q = 0
    (sw.KS, 64, 16, 2 * 3 + 1),          # h = 2, S = 2: 2 timesteps per half-cycle of 16 points
    (sw.KS, 64, 32, 4 * 2 + 3),
    (sw.EULER, 32, 8, 5),
]


@pytest.mark.parametrize("chain", [0, 1, 2], ids=["per-launch", "chain", "band"])
@pytest.mark.parametrize("problem,nx,W,nsteps", CASES)
def test_plan_executed_on_the_model_equals_naive_stepping(problem, nx, W, nsteps, chain):
    h, S = sw.problem_info(problem)["radius"], sw.problem_info(problem)["stages"]
    rng = np.random.default_rng(1612)
    u0 = [int(v) for v in rng.integers(-5, 6, nx)]
    plan = sw.plan(problem, nx, nsteps, W, kernel=sw.KERNEL_SMEM, chain=chain)
    m = Model(nx, h, S, u0)
    m.run_plan(plan)
    ref = Model(nx, h, S, u0).naive(nsteps)
    assert list(m.R[0]) == list(ref)
    # every (point, tier) exactly once: the update count is nx * S * nsteps, whatever the decomposition
    assert m.updates == nx * S * nsteps


def test_plan_structure_and_launch_counts():
    # config 1: 10 000 = 312 * 32 + 16
    plan = sw.plan(sw.HEAT, 1024, 10000, 64, kernel=sw.KERNEL_SMEM, chain=False)
    assert plan == [(sw.LAUNCH_UP, 32, 0, 1), (sw.LAUNCH_DOWN, 32, 16, 1), (sw.LAUNCH_UP, 64, 0, 1), (sw.LAUNCH_DIAMOND, 64, 32, 311),
                    (sw.LAUNCH_DOWN, 64, 0, 1)]
    # the WAVE kernels offer W >= 64 for heat: the 16 remainder steps run on the classic kernel, the sweep is one chained launch
    plan = sw.plan(sw.HEAT, 1024, 10000, 64, kernel=sw.KERNEL_WAVE, chain=True)
    assert plan == [(sw.LAUNCH_CLASSIC, 0, 0, 16), (sw.LAUNCH_CHAIN, 64, 0, 312)]
    # config 2 remainders: 50 000 steps, W = 1024: r = 336 = 256 + 64 + 16
    plan = sw.plan(sw.HEAT, 1 << 22, 50000, 1024, kernel=sw.KERNEL_WAVE, chain=True)
    assert [(k, W) for k, W, _, _ in plan] == [(sw.LAUNCH_UP, 512), (sw.LAUNCH_DOWN, 512), (sw.LAUNCH_UP, 128), (sw.LAUNCH_DOWN, 128),
                                               (sw.LAUNCH_CLASSIC, 0), (sw.LAUNCH_CHAIN, 1024)]
    assert plan[-1][3] == 97 and plan[-2][3] == 16
    # SWEPT_OPT_CHAIN = 2 (streaming bands) and the default 3 (ring kernel): ONE launch, the 336 remainder timesteps as a
    # truncated closing cycle inside it
    assert sw.plan(sw.HEAT, 1 << 22, 50000, 1024, kernel=sw.KERNEL_WAVE, chain=sw.CHAIN_BANDS) == [(sw.LAUNCH_BAND, 1024, 336, 97)]
    assert sw.plan(sw.HEAT, 1 << 22, 50000, 1024, kernel=sw.KERNEL_WAVE) == [(sw.LAUNCH_RING, 1024, 336, 97)]
    assert sw.plan(sw.KS, 4096, 3, 256, kernel=sw.KERNEL_WAVE) == [(sw.LAUNCH_RING, 256, 3, 0)]           # q = 0: only the truncated cycle
    # widths the ring kernel does not take (a tile shorter than 64 iterations; a single tile): the plan of option 2
    assert sw.plan(sw.HEAT, 1024, 10000, 64, kernel=sw.KERNEL_WAVE) == [(sw.LAUNCH_CLASSIC, 0, 0, 16), (sw.LAUNCH_BAND, 64, 0, 312)]
    assert [k for k, *_ in sw.plan(sw.HEAT, 256, 300, 256, kernel=sw.KERNEL_WAVE)][-1] == sw.LAUNCH_BAND
    # q = 0 without the ring kernel: everything classic or narrower tiles
    assert sw.plan(sw.KS, 4096, 3, 128, kernel=sw.KERNEL_WAVE) == [(sw.LAUNCH_CLASSIC, 0, 0, 3)]
    assert sw.plan(sw.KS, 4096, 0, 128) == []


RING_CASES = [
    # problem, nx, W, nsteps: the truncated closing cycle on the plain-Python model (any W: the model has no 64-iteration limit)
    (sw.HEAT, 64, 16, 8 * 3),            # no remainder: phase q closes at tier L
    (sw.HEAT, 64, 16, 8 * 4 + 7),        # odd remainder: the flat result sits on the odd staircase row
    (sw.HEAT, 64, 16, 8 * 3 + 2),
    (sw.HEAT, 32, 16, 5),                # q = 0: the upright triangle truncated at tier L + 5, then tiers 1..5 of the shifted tiles
    (sw.HEAT, 64, 32, 16 * 2 + 15),      # remainder L - 1
    (sw.KS, 64, 16, 2 * 3 + 1),
    (sw.KS, 64, 32, 4 * 2 + 3),
    (sw.KS, 64, 32, 1),
    (sw.EULER, 64, 32, 4 * 3 + 2),
]


@pytest.mark.parametrize("problem,nx,W,nsteps", RING_CASES)
def test_ring_plan_with_truncated_closing_cycle_equals_naive_stepping(problem, nx, W, nsteps):
    """The remainder inside the launch: q half-cycles + r timesteps as phases with tier windows."""
    info = sw.problem_info(problem)
    h, S = info["radius"], info["stages"]
    rng = np.random.default_rng(2495)
    u0 = [int(v) for v in rng.integers(-5, 6, nx)]
    sph = W // (2 * h * S)
    m = Model(nx, h, S, u0)
    m.run_plan([(sw.LAUNCH_RING, W, nsteps % sph, nsteps // sph)])
    ref = Model(nx, h, S, u0).naive(nsteps)
    assert list(m.R[0]) == list(ref)
    assert m.updates == nx * S * nsteps          # every (point, tier) exactly once


def test_plan_rejects_illegal_widths():
    for bad in (0, 3, 48, 4, 1 << 13):
        with pytest.raises(sw.SweptError):
            sw.plan(sw.KS, 4096, 100, bad, kernel=sw.KERNEL_SMEM)
    with pytest.raises(sw.SweptError):
        sw.plan(sw.HEAT, 4096, 100, 32, kernel=sw.KERNEL_WAVE)      # WAVE heat starts at W = 64
    with pytest.raises(sw.SweptError):
        sw.plan(sw.HEAT, 1000, 100, 64)


# ---------------------------------------------------------------------------------------------------------------
# streaming-band schedule (SWEPT_OPT_CHAIN = 2): host logic of swept_band.cuh through the C ABI, no device needed
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ntiles,sms,wpb", [(2, 148, 1), (64, 148, 1), (1024, 148, 8), (4096, 148, 16), (16384, 148, 8), (8192, 148, 28),
                                            (4096, 132, 12), (1000, 7, 3), (5, 148, 4)])
def test_band_assignment_covers_every_band_once_and_balances_the_sub_partitions(ntiles, sms, wpb):
    lay = sw.band_layout(ntiles, sms, wpb)
    assert lay["blocks"] <= sms and lay["blocks"] * wpb >= min(ntiles, sms * wpb)          # at most one block per SM
    assert lay["slots"] == lay["blocks"] * lay["slots_per_block"] and lay["slots_per_block"] * lay["warps_per_slot"] == wpb
    owners = {}
    per_slot = {}
    for band in range(ntiles):
        b, w, i = sw.band_owner(lay, band)
        assert 0 <= b < lay["blocks"] and 0 <= w < wpb and 0 <= i < lay["max_bands_per_warp"]
        assert (b, w, i) not in owners                                                      # one owner position per band
        owners[(b, w, i)] = band
        slot = (b, w % lay["slots_per_block"])                                              # warps w, w+SL, ... share a sub-partition
        per_slot[slot] = per_slot.get(slot, 0) + 1
    # every warp's list is gap-free (indices 0..k-1) and in band order with a constant stride (the kernel relies on both)
    by_warp = {}
    for (b, w, i), band in owners.items():
        by_warp.setdefault((b, w), {})[i] = band
    for lst in by_warp.values():
        assert sorted(lst) == list(range(len(lst)))
        bands = [lst[i] for i in range(len(lst))]
        assert all(y - x == lay["slots"] * lay["warps_per_slot"] for x, y in zip(bands, bands[1:]))
    # neighbouring bands never share a warp (a warp would wait on its own unfinished tile), and the load per sub-partition
    # slot differs by at most one band
    if lay["slots"] >= 2:
        for band in range(ntiles):
            assert sw.band_owner(lay, band)[:2] != sw.band_owner(lay, (band + 1) % ntiles)[:2] or ntiles < 2
    loads = list(per_slot.values()) + [0] * (lay["slots"] - len(per_slot))
    assert max(loads) - min(loads) <= 1
    assert max(len(l) for l in by_warp.values()) == lay["max_bands_per_warp"]


def test_band_layout_rejects_bad_arguments():
    for args in ((0, 148, 4), (10, 0, 4), (10, 148, 0), (10, 148, 6), (10, 148, 33)):
        with pytest.raises(sw.SweptError):
            sw.band_layout(*args)
    with pytest.raises(sw.SweptError):
        sw.band_owner(sw.band_layout(8, 4, 2), 8)


# ---------------------------------------------------------------------------------------------------------------
# insulated ends (SWEPT_BC_INSULATED): the split boundary node as two mirrored tiles, in the model
# ---------------------------------------------------------------------------------------------------------------
class RodModel(Model):
    """The same tile model on a rod whose ghost values are the adjacent interior values: index map g -> -1-g / 2nx-1-g at every
    load, stores only inside the rod, and one extra tile on every shifted launch (tiles on [jW - W/2, jW + W/2), j = 0..nx/W)."""

    def idx(self, g):
        return -1 - g if g < 0 else (2 * self.nx - 1 - g if g >= self.nx else g)

    def naive(self, nsteps):
        a = self.R[0].copy()
        nx, h = self.nx, self.h
        for _ in range(nsteps):
            a = np.array([self.point([a[self.idx(i + k)] for k in range(-h, h + 1)], None, True) for i in range(nx)], dtype=object)
        return a

    def tile(self, mode, W, g0):
        h = self.h
        L, c = W // (2 * h), W // 2
        row = [{x: self.R[0][self.idx(g0 + x)] for x in range(W)}, {}]
        if mode != "up":
            row[1] = {x: self.R[1][self.idx(g0 + x)] for x in range(-h, W + h)}
        spans = []
        if mode != "up":
            spans += [(t, c - h * t, c + h * t) for t in range(1, L + 1)]
        if mode != "down":
            spans += [(t, h * t, W - h * t) for t in range(1, L)]
        for t, lo, hi in spans:
            src, dst = row[(t - 1) & 1], row[t & 1]
            dst.update({x: self.point([src[x + k] for k in range(-h, h + 1)], row[0].get(x), bool(t & 1)) for x in range(lo, hi)})
        return row

    def launch(self, mode, W, offset):
        nx, h = self.nx, self.h
        starts = [t * W for t in range(nx // W)] if offset == 0 else [j * W - W // 2 for j in range(nx // W + 1)]
        rows = [self.tile(mode, W, g0) for g0 in starts]
        for g0, row in zip(starts, rows):
            for x in range(W):
                if 0 <= g0 + x < nx:
                    self.R[0][g0 + x] = row[0][x]
            if mode != "down":
                for x in range(h, W - h):
                    if 0 <= g0 + x < nx:
                        self.R[1][g0 + x] = row[1][x]

    def classic(self, nsteps):
        self.R[0] = self.naive(nsteps)


@pytest.mark.parametrize("chain", [0, 1], ids=["per-launch", "chain"])
@pytest.mark.parametrize("nx,W,nsteps", [(64, 16, 8 * 3), (64, 16, 8 * 4 + 7), (32, 32, 16 * 3 + 5), (64, 8, 3), (48 * 0 + 128, 32, 16 * 5 + 9)])
def test_plan_on_the_rod_model_equals_naive_stepping_with_mirrored_ghosts(nx, W, nsteps, chain):
    """Heat-like symmetric 3-point integer stencil: the launch plan executed with two mirrored boundary tiles per shifted launch
    reproduces naive stepping of the rod exactly (odd and even half-cycle counts, remainders, a single tile)."""
    rng = np.random.default_rng(2495)
    u0 = [int(v) for v in rng.integers(-5, 6, nx)]
    plan = sw.plan(sw.HEAT, nx, nsteps, W, kernel=sw.KERNEL_SMEM, chain=chain)
    m = RodModel(nx, 1, 1, u0)
    m.run_plan(plan)
    ref = RodModel(nx, 1, 1, u0).naive(nsteps)
    assert list(m.R[0]) == list(ref)
    assert list(ref) != list(Model(nx, 1, 1, u0).naive(nsteps))        # and the rod is not the ring


# ---------------------------------------------------------------------------------------------------------------
# streaming-band schedule: a model of the chunk / counter protocol of swept_band.cuh on the C ABI's band assignment
# ---------------------------------------------------------------------------------------------------------------
def _simulate_band_schedule(ntiles, sms, wpb, q, NJI):
    """Every warp runs its tiles phase-major; local time advances in chunks of 32 iterations.  At a chunk boundary K0 a warp
    (1) flushes the output chunk of local times [K0-64, K0-32) -- prog[band] = p NCH + c + 1 -- and (2) may enter the chunk only
    if the left band has flushed chunk c of phase p-1.  Returns (finished, rounds): finished is False on a cycle of waits."""
    NCH = NJI // 32
    lay = sw.band_layout(ntiles, sms, wpb)
    lists = {}
    for band in range(ntiles):
        b, w, i = sw.band_owner(lay, band)
        lists.setdefault((b, w), {})[i] = band
    warps = [[l[i] for i in range(len(l))] for l in lists.values()]
    prog = [0] * ntiles
    K0 = [0] * len(warps)                       # boundary each warp stands at
    end = [len(bands) * (q + 1) * NJI + 31 for bands in warps]
    flushed = [-1] * len(warps)                 # last boundary whose flush ran
    rounds = 0
    while any(k0 < e for k0, e in zip(K0, end)):
        moved = False
        rounds += 1
        for wi, bands in enumerate(warps):
            k = len(bands)
            while K0[wi] < end[wi]:
                kb = K0[wi]
                if flushed[wi] < kb:                                   # (1) flush, once per boundary, before any waiting
                    lt0 = kb - 64
                    if 0 <= lt0 < k * (q + 1) * NJI:
                        s = lt0 // NJI
                        p, m = divmod(s, k)
                        if p < q:
                            prog[bands[m]] = p * NCH + (lt0 % NJI) // 32 + 1
                    flushed[wi] = kb
                    moved = True
                if kb < k * (q + 1) * NJI:                             # (2) fetch: may block
                    s = kb // NJI
                    p, m = divmod(s, k)
                    if p > 0:
                        left = (bands[m] - 1) % ntiles
                        if prog[left] < (p - 1) * NCH + (kb % NJI) // 32 + 1:
                            break
                K0[wi] = kb + 32
                moved = True
        if not moved:
            return False, rounds
    # every band flushed all q phases' output chunks
    assert all(pr == q * NCH for pr in prog), prog[:8]
    return True, rounds


@pytest.mark.parametrize("ntiles,sms,wpb", [(2, 148, 1), (8, 148, 1), (64, 4, 4), (256, 16, 8), (1024, 148, 8), (500, 7, 12), (96, 2, 16)])
@pytest.mark.parametrize("NJI", [64, 128, 512])
def test_band_schedule_never_deadlocks_with_two_or_more_chunks_per_tile(ntiles, sms, wpb, NJI):
    done, _ = _simulate_band_schedule(ntiles, sms, wpb, q=5, NJI=NJI)
    assert done


def test_band_schedule_with_one_chunk_per_tile_is_a_cycle_of_waits():
    """NJI = 32 (heat W = 64, KS / Euler W = 128): at the start of phase p lane 0 needs the chunk its left neighbour flushes only
    32 iterations after ITS phase-p start; with every band in lockstep nobody can move -- the hang observed on the GPU, and the
    reason those widths run on the tile-flag kernel (band_grid refuses NCH < 2)."""
    done, _ = _simulate_band_schedule(64, 148, 1, q=3, NJI=32)
    assert not done


def test_multiply_high_division_by_the_band_count_is_exact():
    """DivK (csrc/swept_band.cuh): floor(s / k) = (s * ceil(2^32 / k)) >> 32 for every s with s k < 2^32 -- the range the kernels
    use it in (s = local tile number < 2^30 / NJI, k = bands per warp).  Checked exhaustively for small s, at the range's edges
    and on a seeded sample, for every k the band layouts can produce."""
    rng = np.random.default_rng(1612)
    for k in list(range(2, 130)) + [255, 256, 1000, 4095, 4096, 65535]:
        m = ((1 << 32) + k - 1) // k
        assert m < (1 << 32)
        top = ((1 << 32) - 1) // k                      # largest s with s k < 2^32
        samples = np.concatenate([np.arange(0, min(top, 5000)), top - np.arange(0, min(top, 5000)), rng.integers(0, top + 1, 20000),
                                  (np.arange(1, min(top // k, 3000) + 1) * k - 1), (np.arange(1, min(top // k, 3000) + 1) * k)])
        samples = samples[(samples >= 0) & (samples <= top)].astype(object)
        for s in samples[:: max(1, len(samples) // 4000)]:
            assert (int(s) * m) >> 32 == int(s) // k, (k, s)
