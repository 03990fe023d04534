"""Host logic of the 2-D swept rule, checked on a plain-Python integer model before any kernel.

Decomposition: in each direction the 1-D swept rule partitions the axis, at local tier s = 1..L of a
half-cycle (L = W/2), into the shrinking intervals U(s) = [s, W - s) of the tiles of one alignment and the expanding intervals
D(s) = [c - s, c + s), c = W/2, of the tiles shifted by W/2 (Fig. 1).  The 2-D rule is the product: every point is,
at tier s, in exactly one of U x U (pyramid), D x U / U x D (the two bridges), D x D (inverted pyramid), and the 5-point stencil makes
U x U self-contained, the bridges depend on U x U, and D x D on all three.  D x D of one half-cycle and U x U of the next sit on the
same (shifted) tiles and fuse into an octahedron, so a half-cycle is TWO launches: bridges, octahedra.  Values live in two
arrays, P0 (newest even tier at every point) and P1 (newest odd tier) -- the 2-D form of the in-place staircase rows R0 / R1.
"""
import numpy as np
import pytest


class Model2D:
    """Integer 5-point stencil new = c0 u + (E + W + N + S) on a periodic [ny][nx] grid; P[0] / P[1] hold even / odd tiers."""

    def __init__(self, nx, ny, u0):
        self.nx, self.ny = nx, ny
        self.P = [np.array(u0, dtype=object).reshape(ny, nx), np.zeros((ny, nx), dtype=object)]
        self.updates = 0

    @staticmethod
    def point(u, e, w, n, s):
        return 3 * u + ((e + w) + (n + s))

    def naive(self, nsteps):
        a = self.P[0].copy()
        for _ in range(nsteps):
            a = 3 * a + ((np.roll(a, -1, 1) + np.roll(a, 1, 1)) + (np.roll(a, -1, 0) + np.roll(a, 1, 0)))
        return a

    def region(self, W, ox, oy, mx, my, tiers):
        """One launch: every tile of the grid shifted by (ox, oy) runs the local tiers `tiers` (1..2L-1; s > L continues as the
        next half-cycle's U x U) on the rectangle rect_x(s) x rect_y(s), mx / my in 'U', 'D'.  Snapshot semantics: all tiles load
        before any stores; a tile stores only the points it updated (both planes where it wrote both)."""
        nx, ny, L, c = self.nx, self.ny, W // 2, W // 2

        def rect(mode, s):
            if s > L:                       # the shrinking half of an octahedron: local tier s - L of U
                return (s - L, W - (s - L))
            return (s, W - s) if mode == "U" else (c - s, c + s)

        stores = []
        for ty in range(ny // W):
            for tx in range(nx // W):
                gx0, gy0 = tx * W + ox, ty * W + oy
                pl = [{(x, y): self.P[p][(gy0 + y) % ny, (gx0 + x) % nx] for x in range(-1, W + 1) for y in range(-1, W + 1)} for p in (0, 1)]
                wrote = {}
                for s in tiers:
                    (xa, xb), (ya, yb) = rect(mx, s), rect(my, s)
                    src, dst = pl[(s - 1) & 1], pl[s & 1]
                    new = {(x, y): self.point(src[x, y], src[x + 1, y], src[x - 1, y], src[x, y + 1], src[x, y - 1])
                           for x in range(xa, xb) for y in range(ya, yb)}
                    dst.update(new)
                    self.updates += len(new)
                    for k in new:
                        wrote.setdefault(k, set()).add(s & 1)
                stores.append((gx0, gy0, pl, wrote))
        for gx0, gy0, pl, wrote in stores:
            for (x, y), planes in wrote.items():
                for p in planes:
                    self.P[p][(gy0 + y) % ny, (gx0 + x) % nx] = pl[p][x, y]

    def swept(self, W, K):
        """K half-cycles of L = W/2 timesteps: pyramids, then per half-cycle bridges + octahedra (the last one only its lower half)."""
        L, h = W // 2, W // 2
        self.region(W, 0, 0, "U", "U", range(1, L))                                  # upright pyramids from the flat field
        for k in range(K):
            a = (k % 2) * h                                                          # alignment that shrinks in this half-cycle
            b = h - a
            self.region(W, b, a, "D", "U", range(1, L + 1))                          # bridges: expanding in x, shrinking in y
            self.region(W, a, b, "U", "D", range(1, L + 1))                          # ... and the other way round (same launch)
            self.region(W, b, b, "D", "D", range(1, L + 1) if k == K - 1 else range(1, 2 * L))   # inverted pyramids / octahedra


@pytest.mark.parametrize("nx,ny,W,K", [(16, 16, 8, 1), (16, 16, 8, 2), (16, 8, 8, 3), (8, 8, 8, 2), (24, 16, 8, 4), (16, 16, 16, 2), (32, 16, 16, 3)])
def test_2d_swept_plan_on_the_model_equals_naive_stepping(nx, ny, W, K):
    rng = np.random.default_rng(1612)
    u0 = [int(v) for v in rng.integers(-5, 6, nx * ny)]
    m = Model2D(nx, ny, u0)
    m.swept(W, K)
    ref = Model2D(nx, ny, u0).naive(K * (W // 2))
    assert np.array_equal(m.P[0], ref)
    assert m.updates == nx * ny * K * (W // 2)          # every (point, tier) exactly once


def test_region_volumes():
    """Per tile and half-cycle: pyramid + two bridges + inverted pyramid = L W^2 point updates (the four products of the 1-D
    triangles' row lengths sum to W x W at every tier)."""
    for W in (8, 16, 32, 64):
        L, c = W // 2, W // 2
        uu = sum((W - 2 * s) ** 2 for s in range(1, L + 1))
        du = sum(2 * s * (W - 2 * s) for s in range(1, L + 1))
        dd = sum((2 * s) ** 2 for s in range(1, L + 1))
        assert uu + 2 * du + dd == L * W * W


# ---- the register kernels' closed forms (csrc/heat2d.cu: tile32, tile32f) -------------------------------------------------------
def _rect(region, ybridge, s, W=32):
    """The rectangle [xa, xb) x [ya, yb) a tile updates at local tier s, as the kernels compute it."""
    L = C = W // 2
    if region == "pyramid":
        return s, W - s, s, W - s
    if region == "bridges":
        ea, eb, sa, sb = C - s, C + s, s, W - s
        return (sa, sb, ea, eb) if ybridge else (ea, eb, sa, sb)
    if s <= L:
        return C - s, C + s, C - s, C + s
    return s - L, W - (s - L), s - L, W - (s - L)


REGIONS = [("pyramid", False, 15), ("bridges", False, 15), ("bridges", True, 15), ("inverted", False, 16), ("octahedron", False, 31)]


@pytest.mark.parametrize("region,ybridge,S1", REGIONS)
def test_register_kernel_store_rule_matches_the_rectangles(region, ybridge, S1):
    """The register kernels do not record which tiers touched a point; they store by closed form: point (x, y) was updated at the
    tiers [s_lo, s_hi] (none if s_hi < s_lo).  Brute force over the rectangles: the set of tiers is exactly that interval."""
    W, L, C = 32, 16, 16
    for y in range(W):
        for x in range(W):
            tiers = [s for s in range(1, S1 + 1) if (lambda r: r[0] <= x < r[1] and r[2] <= y < r[3])(_rect(region, ybridge, s))]
            ux, uy = min(x, W - 1 - x), min(y, W - 1 - y)
            dx, dy = max(C - x, x - C + 1), max(C - y, y - C + 1)
            if region == "pyramid":
                s_lo, s_hi = 1, min(ux, uy)
            elif region == "bridges":
                s_lo, s_hi = (dy, ux) if ybridge else (dx, uy)
            elif region == "inverted":
                s_lo, s_hi = max(dx, dy), L
            else:
                s_lo, s_hi = max(dx, dy), L + min(ux, uy)
            want = list(range(s_lo, s_hi + 1)) if s_hi >= s_lo and s_hi >= 1 else []
            assert tiers == want, (region, ybridge, x, y, tiers, want)


@pytest.mark.parametrize("region,ybridge,S1", REGIONS)
def test_folded_layout_of_the_register_kernel(region, ybridge, S1):
    """tile32f folds rows 16..31 onto lanes 16..31 (register row r holds row r in the lower half, row 31 - r in the upper) and
    runs register rows ya..15 of both halves together.  That needs (1) every rectangle symmetric about the centre row, yb = 32 - ya
    with ya <= 15; (2) the row terms of the store rule equal in both halves: min(y, 31 - y) = r and max(16 - y, y - 15) = 16 - r;
    (3) only the full-tile tier (s = L of an inverted pyramid) touching rows 0 / 31 and columns 0 / 31, the only places where the
    fold's halo values are used."""
    W, L = 32, 16
    for s in range(1, S1 + 1):
        xa, xb, ya, yb = _rect(region, ybridge, s)
        if xa >= xb or ya >= yb:
            assert region == "bridges" and s == L        # (a bridge's tier L would be empty; the kernels stop at L - 1)
            continue
        assert ya + yb == W and 0 <= ya <= 15
        full = region in ("inverted", "octahedron") and s == L
        assert (ya == 0) == full and (xa == 0 or xb == W) == full
    for r in range(16):
        for y in (r, 31 - r):
            assert min(y, W - 1 - y) == r and max(16 - y, y - 15) == 16 - r
