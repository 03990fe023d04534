// heat2d.cu -- the 2-D swept rule for the heat equation (include/swept2d.h): kernels and C ABI.
//
// Block = tile of W x W points, thread = point, two shared-memory planes of (W + 2)^2 values: plane 0 holds the newest even
// tier of every point of the tile and its one-point halo, plane 1 the newest odd tier -- the 2-D form of the paper's two-row
// shared matrix.  A launch runs one REGION kind on every tile of its alignment: at local tier s the points
// of rect_x(s) x rect_y(s) are updated from plane (s-1)&1 into plane s&1 (one block barrier per tier), where per direction
//     U (shrinking, the upright triangle of PAPER.md:82):   [s, W - s)
//     D (expanding, the inverted triangle of PAPER.md:98):  [W/2 - s, W/2 + s)
// and tiers s > L of an octahedron continue as U with s - L.  Afterwards every thread stores what it updated: plane p of its point
// if it wrote plane p -- nothing else, so tiles of one launch never write what another reads (tests/test_geometry2d.py runs the same
// plan on a plain-Python model).  The point update is Heat2D<T>::point of stencils.cuh, shared with the classic kernel.
#include <math.h>
#include <string.h>

#include <new>

#include "../../include/swept2d.h"
#include "internal.h"
#include "stencils.cuh"

using namespace swept;

struct swept2d_ctx {
    int dtype, device, kernel;
    int64_t nx, ny;
    double dx, dt, alpha;
    ConstBlock cb;
    void *work;
    void *host_stage;      // device buffer of swept2d_run_host (allocated on first use)
    size_t field_bytes;
    int64_t launches_last, launches_total;
};

namespace {

enum { R_PYRAMID = 0, R_BRIDGES = 1, R_INVERTED = 2, R_OCTAHEDRON = 3 };

// Classic path: a thread updates 16 bytes of consecutive x points (2 doubles / 4 floats): one aligned vector load each for its own
// row and the rows above and below, two scalar loads for the E / W ends (L1 hits), one vector store -- the 1-D classic kernel's
// layout (naive.cu).  With one point per thread the kernel was bound by instruction issue (fp64 0.60, fp32 0.34 of the HBM figure).
template <class T> struct Vec16;
template <> struct Vec16<double> { using type = double2; static constexpr int N = 2; };
template <> struct Vec16<float> { using type = float4; static constexpr int N = 4; };

template <class T>
__global__ void __launch_bounds__(256) classic2d_kernel(const T *__restrict__ src, T *__restrict__ dst, int64_t nx, int64_t ny, typename Heat2D<T>::Consts c) {
    using V = typename Vec16<T>::type;
    constexpr int N = Vec16<T>::N;
    const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * N, j = (int64_t)blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= nx || j >= ny) return;                       // nx is a power of two >= 8: a multiple of N
    const int64_t jn = (j + 1) & (ny - 1), js = (j - 1) & (ny - 1);
    const V vc = *reinterpret_cast<const V *>(src + j * nx + i), vn = *reinterpret_cast<const V *>(src + jn * nx + i), vs = *reinterpret_cast<const V *>(src + js * nx + i);
    const T *pc = reinterpret_cast<const T *>(&vc), *pn = reinterpret_cast<const T *>(&vn), *ps = reinterpret_cast<const T *>(&vs);
    const T uw = src[j * nx + ((i - 1) & (nx - 1))], ue = src[j * nx + ((i + N) & (nx - 1))];
    V out;
    T *po = reinterpret_cast<T *>(&out);
#pragma unroll
    for (int k = 0; k < N; ++k) po[k] = Heat2D<T>::point(c, pc[k], k < N - 1 ? pc[k < N - 1 ? k + 1 : k] : ue, k > 0 ? pc[k > 0 ? k - 1 : k] : uw, pn[k], ps[k]);
    *reinterpret_cast<V *>(dst + j * nx + i) = out;
}

// One region kind on the tiles whose origin is (ox, oy) + (tile index) * W.  REGION = R_BRIDGES: blockIdx.z = 0 runs the x-bridges
// (expanding in x, shrinking in y) at origin (ox, oy), blockIdx.z = 1 the y-bridges at origin (oy, ox).
template <class T, int W, int REGION>
__global__ void __launch_bounds__(W *W) swept2d_kernel(T *__restrict__ p0, T *__restrict__ p1, int64_t nx, int64_t ny, int ox, int oy, typename Heat2D<T>::Consts c) {
    constexpr int L = W / 2, C = W / 2, PS = W + 2;       // PS: plane stride (one halo point on every side)
    __shared__ T pl[2][PS * PS];
    const int x = (int)threadIdx.x, y = (int)threadIdx.y;
    const bool ybridge = REGION == R_BRIDGES && blockIdx.z == 1;
    const int64_t gx0 = (int64_t)blockIdx.x * W + (ybridge ? oy : ox), gy0 = (int64_t)blockIdx.y * W + (ybridge ? ox : oy);
    const int64_t mx = nx - 1, my = ny - 1;
    auto gidx = [&](int lx, int ly) -> int64_t { return ((gy0 + ly) & my) * nx + ((gx0 + lx) & mx); };
    // ---- load both planes: own point, and the halo ring by the first 4 W threads
    {
        const int64_t g = gidx(x, y);
        pl[0][(y + 1) * PS + x + 1] = p0[g];
        if (REGION != R_PYRAMID) pl[1][(y + 1) * PS + x + 1] = p1[g];
        const int t = y * W + x;
        if (t < 4 * W) {
            const int side = t / W, k = t % W;
            const int lx = side == 0 ? -1 : (side == 1 ? W : k), ly = side == 2 ? -1 : (side == 3 ? W : k);
            const int64_t gh = gidx(lx, ly);
            pl[0][(ly + 1) * PS + lx + 1] = p0[gh];
            if (REGION != R_PYRAMID) pl[1][(ly + 1) * PS + lx + 1] = p1[gh];
        }
    }
    __syncthreads();
    // ---- tiers
    constexpr int S0 = 1, S1 = REGION == R_PYRAMID ? L - 1 : (REGION == R_OCTAHEDRON ? 2 * L - 1 : L);
    int s_lo = 0, s_hi = 0;                               // tiers this thread updated: [s_lo, s_hi] (0 = none)
    const int me = (y + 1) * PS + x + 1;
#pragma unroll 1
    for (int s = S0; s <= S1; ++s) {
        int xa, xb, ya, yb;
        if (REGION == R_PYRAMID) { xa = ya = s; xb = yb = W - s; }
        else if (REGION == R_BRIDGES) {
            const int ea = C - s, eb = C + s, sa = s, sb = W - s;           // expanding / shrinking interval
            xa = ybridge ? sa : ea; xb = ybridge ? sb : eb;
            ya = ybridge ? ea : sa; yb = ybridge ? eb : sb;
        } else if (s <= L) { xa = ya = C - s; xb = yb = C + s; }
        else { xa = ya = s - L; xb = yb = W - (s - L); }
        if (x >= xa && x < xb && y >= ya && y < yb) {
            const T *src = pl[(s - 1) & 1];
            pl[s & 1][me] = Heat2D<T>::point(c, src[me], src[me + 1], src[me - 1], src[me + PS], src[me - PS]);
            if (s_lo == 0) s_lo = s;
            s_hi = s;
        }
        __syncthreads();
    }
    // ---- store what this thread updated
    if (s_hi > 0) {
        const int64_t g = gidx(x, y);
        T *newest = (s_hi & 1) ? p1 : p0, *other = (s_hi & 1) ? p0 : p1;
        newest[g] = pl[s_hi & 1][me];
        if (s_hi > s_lo) other[g] = pl[(s_hi - 1) & 1][me];
    }
}

// ---- register-resident tiles (W = 32): one WARP per tile, lane = x, the tile's 32 rows of both planes in registers -----------
// The paper-style kernel above keeps at most a third (octahedra) or a sixth (bridges) of a block's threads busy and pays a block
// barrier per tier.  Here a warp owns a 32 x 32 tile: lane x holds column x of plane 0 (newest even tier) and plane 1 (newest odd
// tier) in a0[32], a1[32]; the N/S neighbours of a point are registers of the same lane, the E/W neighbours two shuffles.  A tier
// updates the rows [ya, yb) of its rectangle (a warp-uniform branch per row, so rows outside cost nothing) on the lanes [xa, xb)
// (a predicate).  No shared-memory planes, no barrier: the 1-D register wavefront's idea (swept_wave.cuh) in its 2-D form.
// Halo: a rectangle reads one point beyond itself, and only the last tier of an inverted pyramid (s = L, the full tile) reaches
// beyond the tile: rows -1 and W come in two registers per lane, columns -1 and W through 2 x 32 values of shared memory per warp.
// Same regions, same tier order, same store rule as swept2d_kernel, so the two interoperate and are both bit-identical to the
// classic path.
constexpr int WARPS2D = 8;

template <class T, bool SRC0, bool HALO>
__device__ __forceinline__ void tier32(T (&a0)[32], T (&a1)[32], const int lane, const int xa, const int xb, const int ya, const int yb, const T hS, const T hN,
                                       const T *hl, const T *hr, const typename Heat2D<T>::Consts &c) {
    T(&src)[32] = SRC0 ? a0 : a1;
    T(&dst)[32] = SRC0 ? a1 : a0;
    // bit y of `rows`: row y is in [ya, yb) (warp-uniform); `mine`: ... and this lane is in [xa, xb)
    const unsigned rows = (yb >= 32 ? 0xffffffffu : (1u << yb) - 1u) & ~((1u << ya) - 1u);
    const unsigned mine = (lane >= xa && lane < xb) ? rows : 0u;
    // Rows in groups of RG: one warp-uniform branch per group, so that the group's 2 RG shuffles and RG dependent chains
    // (shuffle -> 2 adds -> add -> fma) overlap -- with a branch per row every chain ran exposed (ncu: `wait` 3.3 per issue, FP64 pipe
    // 10 %); rows of a group outside [ya, yb) are computed and dropped (3 rows per tier on average).
    constexpr int RG = sizeof(T) == 4 ? 8 : 4;
#pragma unroll
    for (int g = 0; g < 32 / RG; ++g) {
        if ((rows >> (RG * g)) & ((1u << RG) - 1u)) {     // warp-uniform
            T e[RG], w[RG], v[RG];
#pragma unroll
            for (int r = 0; r < RG; ++r) {
                const int y = RG * g + r;
                e[r] = __shfl_down_sync(0xffffffffu, src[y], 1);
                w[r] = __shfl_up_sync(0xffffffffu, src[y], 1);
                if (HALO) {
                    if (lane == 0) w[r] = hl[y];
                    if (lane == 31) e[r] = hr[y];
                }
            }
#pragma unroll
            for (int r = 0; r < RG; ++r) {
                const int y = RG * g + r;
                const T n = y < 31 ? src[y < 31 ? y + 1 : 31] : hN, so = y > 0 ? src[y > 0 ? y - 1 : 0] : hS;
                v[r] = Heat2D<T>::point(c, src[y], e[r], w[r], n, so);
            }
#pragma unroll
            for (int r = 0; r < RG; ++r) {
                const int y = RG * g + r;
                if ((mine >> y) & 1u) dst[y] = v[r];   // (a predicate on the fma itself -- inline PTX -- is turned back into these selects by ptxas)
            }
        }
    }
}

// Tiles of origin (ox, oy) + (tile index) * 32; REGION = R_BRIDGES: tiles [0, ntiles) are the x-bridges at origin (ox, oy), tiles
// [ntiles, 2 ntiles) the y-bridges at origin (oy, ox).
template <class T, int REGION, bool ybridge>
__device__ __forceinline__ void tile32(T *__restrict__ p0, T *__restrict__ p1, const int64_t nx, const int64_t ny, const int ox, const int oy, const int tiles_x, const int64_t t,
                                       T (*halo)[32], const int lane, const typename Heat2D<T>::Consts &c) {
    constexpr int W = 32, L = 16, C = 16;
    constexpr bool HALO_REGION = REGION == R_INVERTED || REGION == R_OCTAHEDRON;
    const int64_t gx0 = (t % tiles_x) * W + (ybridge ? oy : ox), gy0 = (t / tiles_x) * W + (ybridge ? ox : oy);
    const int64_t mx = nx - 1, my = ny - 1;
    auto gidx = [&](int lx, int ly) -> int64_t { return ((gy0 + ly) & my) * nx + ((gx0 + lx) & mx); };
    T a0[32], a1[32];
#pragma unroll
    for (int y = 0; y < 32; ++y) {
        const int64_t g = gidx(lane, y);
        a0[y] = p0[g];
        a1[y] = REGION != R_PYRAMID ? p1[g] : T(0);
    }
    T hS = T(0), hN = T(0);
    const T *hl = halo[0], *hr = halo[1];
    if (HALO_REGION) {                                    // tier L reads plane (L - 1) & 1 = 1 one point beyond the tile
        hS = p1[gidx(lane, -1)];
        hN = p1[gidx(lane, W)];
        halo[0][lane] = p1[gidx(-1, lane)];
        halo[1][lane] = p1[gidx(W, lane)];
        __syncwarp();
    }
    constexpr int S1 = REGION == R_OCTAHEDRON ? 2 * L - 1 : (REGION == R_INVERTED ? L : L - 1);   // (a bridge's tier L is empty)
    auto rect = [&](int s, int &xa, int &xb, int &ya, int &yb) {
        if (REGION == R_PYRAMID) { xa = ya = s; xb = yb = W - s; }
        else if (REGION == R_BRIDGES) {
            const int ea = C - s, eb = C + s, sa = s, sb = W - s;
            xa = ybridge ? sa : ea; xb = ybridge ? sb : eb;
            ya = ybridge ? ea : sa; yb = ybridge ? eb : sb;
        } else if (s <= L) { xa = ya = C - s; xb = yb = C + s; }
        else { xa = ya = s - L; xb = yb = W - (s - L); }
    };
#pragma unroll 1
    for (int s = 1; s <= S1; s += 2) {
        int xa, xb, ya, yb;
        rect(s, xa, xb, ya, yb);
        tier32<T, true, false>(a0, a1, lane, xa, xb, ya, yb, hS, hN, hl, hr, c);
        if (s + 1 <= S1) {
            rect(s + 1, xa, xb, ya, yb);
            if (HALO_REGION && s + 1 == L) tier32<T, false, true>(a0, a1, lane, xa, xb, ya, yb, hS, hN, hl, hr, c);
            else tier32<T, false, false>(a0, a1, lane, xa, xb, ya, yb, hS, hN, hl, hr, c);
        }
    }
    // ---- store what this lane updated: point (x, y) was updated at the tiers [s_lo, s_hi] (closed forms of the rectangles above);
    // the newest tier goes to its plane, the one before it -- if the point was updated twice or more -- to the other
    const int x = lane, ux = x < W - 1 - x ? x : W - 1 - x, dx = C - x > x - C + 1 ? C - x : x - C + 1;
#pragma unroll
    for (int y = 0; y < 32; ++y) {
        const int uy = y < W - 1 - y ? y : W - 1 - y, dy = C - y > y - C + 1 ? C - y : y - C + 1;
        const int umin = ux < uy ? ux : uy, dmax = dx > dy ? dx : dy;
        int s_lo, s_hi;
        if (REGION == R_PYRAMID) { s_lo = 1; s_hi = umin; }
        else if (REGION == R_BRIDGES) { s_lo = ybridge ? dy : dx; s_hi = ybridge ? ux : uy; }
        else if (REGION == R_INVERTED) { s_lo = dmax; s_hi = L; }
        else { s_lo = dmax; s_hi = L + umin; }
        if (s_hi >= s_lo && s_hi >= 1) {
            const int64_t g = gidx(x, y);
            const bool odd = (s_hi & 1) != 0;
            (odd ? p1 : p0)[g] = odd ? a1[y] : a0[y];
            if (s_hi > s_lo) (odd ? p0 : p1)[g] = odd ? a0[y] : a1[y];
        }
    }
}

// ---- the folded tile: two columns per lane, the upper 16 rows folded onto lanes 16..31 ----------------------------------------
// tile32 above spends 4 shuffles and ~10 bookkeeping instructions per 32-point row on 5 FP instructions.  Here lane (half, l) owns
// the columns 2l, 2l+1 of the rows r (half 0) or 31 - r (half 1), r = 0..15: a register row r is 64 points.  Of a point pair only
// the outer E / W neighbours cross lanes (one shuffle each, within the 16-lane half), so shuffles per point halve and the row
// bookkeeping is shared by two points.  Every rectangle is symmetric about the tile's centre row, so register row r is active in both
// halves at once ([ya, 32 - ya) = r >= ya) and nothing is wasted by the fold; the upper half runs its rows top-down, which swaps the
// roles of N and S -- harmless bit for bit, the update adds them (uN + uS = uS + uN).  The seam (rows 15 | 16) is one exchange
// between the halves per tier and column.
template <class T> struct alignas(2 * sizeof(T)) Pair2 { T a, b; };

template <class T, bool SRC0, bool HALO>
__device__ __forceinline__ void tier32f(T (&a0)[16][2], T (&a1)[16][2], const int half, const int l, const int xa, const int xb, const int ya, const T (&hrow)[2],
                                        const T *hl, const T *hr, const typename Heat2D<T>::Consts &c) {
    T(&src)[16][2] = SRC0 ? a0 : a1;
    T(&dst)[16][2] = SRC0 ? a1 : a0;
    // register rows per uniform branch (measured, 8192^2, GPts*steps/s: fp64 1: 345, 2: 414, 4: 425; fp32 2: 756, 4: 813, 8: 785, 16: 640)
    constexpr int RG = 4;
    const unsigned rows = 0xffffu & ~((1u << ya) - 1u);    // register rows ya .. 15 (warp-uniform)
    const int x0 = 2 * l;
    const unsigned mine0 = (x0 >= xa && x0 < xb) ? rows : 0u, mine1 = (x0 + 1 >= xa && x0 + 1 < xb) ? rows : 0u;
    T seam[2];                                            // row 16 for the lower half, row 15 for the upper: the other half's r = 15
#pragma unroll
    for (int k = 0; k < 2; ++k) seam[k] = __shfl_xor_sync(0xffffffffu, src[15][k], 16);
#pragma unroll
    for (int g = 0; g < 16 / RG; ++g) {
        if ((rows >> (RG * g)) & ((1u << RG) - 1u)) {     // warp-uniform
            T eR[RG], wL[RG], v0[RG], v1[RG];
#pragma unroll
            for (int q = 0; q < RG; ++q) {
                const int r = RG * g + q;
                eR[q] = __shfl_down_sync(0xffffffffu, src[r][0], 1, 16);   // lane l+1's left column: E of my right column
                wL[q] = __shfl_up_sync(0xffffffffu, src[r][1], 1, 16);     // lane l-1's right column: W of my left column
                if (HALO) {
                    const int y = half ? 31 - r : r;
                    if (l == 0) wL[q] = hl[y];
                    if (l == 15) eR[q] = hr[y];
                }
            }
#pragma unroll
            for (int q = 0; q < RG; ++q) {
                const int r = RG * g + q;
                const T up0 = r < 15 ? src[r < 15 ? r + 1 : 15][0] : seam[0], up1 = r < 15 ? src[r < 15 ? r + 1 : 15][1] : seam[1];
                const T dn0 = r > 0 ? src[r > 0 ? r - 1 : 0][0] : hrow[0], dn1 = r > 0 ? src[r > 0 ? r - 1 : 0][1] : hrow[1];
                v0[q] = Heat2D<T>::point(c, src[r][0], src[r][1], wL[q], up0, dn0);
                v1[q] = Heat2D<T>::point(c, src[r][1], eR[q], src[r][0], up1, dn1);
            }
#pragma unroll
            for (int q = 0; q < RG; ++q) {
                const int r = RG * g + q;
                if ((mine0 >> r) & 1u) dst[r][0] = v0[q];
                if ((mine1 >> r) & 1u) dst[r][1] = v1[q];
            }
        }
    }
}

template <class T, int REGION, bool ybridge>
__device__ __forceinline__ void tile32f(T *__restrict__ p0, T *__restrict__ p1, const int64_t nx, const int64_t ny, const int ox, const int oy, const int tiles_x, const int64_t t,
                                        T (*halo)[32], const int lane, const typename Heat2D<T>::Consts &c) {
    constexpr int W = 32, L = 16, C = 16;
    constexpr bool HALO_REGION = REGION == R_INVERTED || REGION == R_OCTAHEDRON;
    using V2 = Pair2<T>;
    const int half = lane >> 4, l = lane & 15, x0 = 2 * l;
    const int64_t gx0 = (t % tiles_x) * W + (ybridge ? oy : ox), gy0 = (t / tiles_x) * W + (ybridge ? ox : oy);
    const int64_t mx = nx - 1, my = ny - 1;
    auto gidx = [&](int lx, int ly) -> int64_t { return ((gy0 + ly) & my) * nx + ((gx0 + lx) & mx); };
    T a0[16][2], a1[16][2];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int64_t g = gidx(x0, half ? 31 - r : r);    // gx0 and x0 are even: the pair is aligned and does not straddle the wrap
        const V2 v = *reinterpret_cast<const V2 *>(p0 + g);
        a0[r][0] = v.a; a0[r][1] = v.b;
        if (REGION != R_PYRAMID) {
            const V2 u = *reinterpret_cast<const V2 *>(p1 + g);
            a1[r][0] = u.a; a1[r][1] = u.b;
        } else { a1[r][0] = a1[r][1] = T(0); }
    }
    T hrow[2] = {T(0), T(0)};                             // row -1 (lower half) / row 32 (upper half) of plane 1, this lane's columns
    const T *hl = halo[0], *hr = halo[1];
    if (HALO_REGION) {                                    // tier L reads plane (L - 1) & 1 = 1 one point beyond the tile
        const V2 u = *reinterpret_cast<const V2 *>(p1 + gidx(x0, half ? W : -1));
        hrow[0] = u.a; hrow[1] = u.b;
        halo[0][lane] = p1[gidx(-1, lane)];
        halo[1][lane] = p1[gidx(W, lane)];
        __syncwarp();
    }
    constexpr int S1 = REGION == R_OCTAHEDRON ? 2 * L - 1 : (REGION == R_INVERTED ? L : L - 1);
    auto rect = [&](int s, int &xa, int &xb, int &ya) {   // (yb = 32 - ya for every region)
        if (REGION == R_PYRAMID) { xa = ya = s; xb = W - s; }
        else if (REGION == R_BRIDGES) {
            xa = ybridge ? s : C - s; xb = ybridge ? W - s : C + s;
            ya = ybridge ? C - s : s;
        } else if (s <= L) { xa = ya = C - s; xb = C + s; }
        else { xa = ya = s - L; xb = W - (s - L); }
    };
#pragma unroll 1
    for (int s = 1; s <= S1; s += 2) {
        int xa, xb, ya;
        rect(s, xa, xb, ya);
        tier32f<T, true, false>(a0, a1, half, l, xa, xb, ya, hrow, hl, hr, c);
        if (s + 1 <= S1) {
            rect(s + 1, xa, xb, ya);
            if (HALO_REGION && s + 1 == L) tier32f<T, false, true>(a0, a1, half, l, xa, xb, ya, hrow, hl, hr, c);
            else tier32f<T, false, false>(a0, a1, half, l, xa, xb, ya, hrow, hl, hr, c);
        }
    }
    // ---- store (the rule of tile32): for register row r both halves have uy = r and dy = 16 - r
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int y = half ? 31 - r : r, uy = r, dy = C - r;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int x = x0 + k, ux = x < W - 1 - x ? x : W - 1 - x, dx = C - x > x - C + 1 ? C - x : x - C + 1;
            const int umin = ux < uy ? ux : uy, dmax = dx > dy ? dx : dy;
            int s_lo, s_hi;
            if (REGION == R_PYRAMID) { s_lo = 1; s_hi = umin; }
            else if (REGION == R_BRIDGES) { s_lo = ybridge ? dy : dx; s_hi = ybridge ? ux : uy; }
            else if (REGION == R_INVERTED) { s_lo = dmax; s_hi = L; }
            else { s_lo = dmax; s_hi = L + umin; }
            if (s_hi >= s_lo && s_hi >= 1) {
                const int64_t g = gidx(x, y);
                const bool odd = (s_hi & 1) != 0;
                (odd ? p1 : p0)[g] = odd ? a1[r][k] : a0[r][k];
                if (s_hi > s_lo) (odd ? p0 : p1)[g] = odd ? a0[r][k] : a1[r][k];
            }
        }
    }
}

template <class T, int REGION, bool FOLD = true>
__global__ void __launch_bounds__(32 * WARPS2D, sizeof(T) == 4 ? 2 : 1) swept2d_warp_kernel(T *__restrict__ p0, T *__restrict__ p1, int64_t nx, int64_t ny, int ox, int oy, int tiles_x, int64_t ntiles,
                                                                     typename Heat2D<T>::Consts c) {
    __shared__ T halo[WARPS2D][2][32];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    const int64_t t = (int64_t)blockIdx.x * WARPS2D + warp;
    if (t >= ntiles * (REGION == R_BRIDGES ? 2 : 1)) return;
    // the two kinds of bridge are two instances of the tile code: with the kind a run-time value the compiler re-derived it (and
    // the rectangle) from the block and thread index inside every row group rather than spend registers on it
    if constexpr (FOLD) {
        if (REGION == R_BRIDGES && t >= ntiles) tile32f<T, REGION, true>(p0, p1, nx, ny, ox, oy, tiles_x, t - ntiles, halo[warp], lane, c);
        else tile32f<T, REGION, false>(p0, p1, nx, ny, ox, oy, tiles_x, t, halo[warp], lane, c);
    } else {
        if (REGION == R_BRIDGES && t >= ntiles) tile32<T, REGION, true>(p0, p1, nx, ny, ox, oy, tiles_x, t - ntiles, halo[warp], lane, c);
        else tile32<T, REGION, false>(p0, p1, nx, ny, ox, oy, tiles_x, t, halo[warp], lane, c);
    }
}

template <class T> typename Heat2D<T>::Consts consts_of(const swept2d_ctx *h) { return *reinterpret_cast<const typename Heat2D<T>::Consts *>(h->cb.bytes); }

template <class T> cudaError_t classic2d(swept2d_ctx *h, void *d_u, int64_t nsteps, cudaStream_t st, int64_t *launches) {
    T *a = (T *)d_u, *b = (T *)h->work;
    constexpr int N = Vec16<T>::N;
    const dim3 block(32, 8), grid((unsigned)((h->nx / N + 31) / 32), (unsigned)((h->ny + 7) / 8));
    for (int64_t m = 0; m < nsteps; ++m) {
        classic2d_kernel<T><<<grid, block, 0, st>>>(a, b, h->nx, h->ny, consts_of<T>(h));
        T *t = a; a = b; b = t;
        ++*launches;
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && a != (T *)d_u) e = cudaMemcpyAsync(d_u, a, h->field_bytes, cudaMemcpyDeviceToDevice, st);
    return e;
}

template <class T, int W> cudaError_t sweep2d(swept2d_ctx *h, void *d_u, int64_t K, cudaStream_t st, int64_t *launches) {
    if (K <= 0) return cudaSuccess;
    T *p0 = (T *)d_u, *p1 = (T *)h->work;
    const dim3 block(W, W), grid((unsigned)(h->nx / W), (unsigned)(h->ny / W), 1), grid2(grid.x, grid.y, 2);
    const typename Heat2D<T>::Consts c = consts_of<T>(h);
    swept2d_kernel<T, W, R_PYRAMID><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, 0, 0, c);
    ++*launches;
    for (int64_t k = 0; k < K; ++k) {
        const int a = (int)(k & 1) * (W / 2), b = W / 2 - a;      // a: the alignment that shrinks in this half-cycle
        swept2d_kernel<T, W, R_BRIDGES><<<grid2, block, 0, st>>>(p0, p1, h->nx, h->ny, b, a, c);
        if (k == K - 1) swept2d_kernel<T, W, R_INVERTED><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, c);
        else swept2d_kernel<T, W, R_OCTAHEDRON><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, c);
        *launches += 2;
    }
    return cudaGetLastError();
}

template <class T, bool FOLD> cudaError_t sweep2d_warp(swept2d_ctx *h, void *d_u, int64_t K, cudaStream_t st, int64_t *launches) {
    if (K <= 0) return cudaSuccess;
    constexpr int W = 32;
    T *p0 = (T *)d_u, *p1 = (T *)h->work;
    const int tiles_x = (int)(h->nx / W);
    const int64_t ntiles = (h->nx / W) * (h->ny / W);
    const dim3 block(32 * WARPS2D), grid((unsigned)((ntiles + WARPS2D - 1) / WARPS2D)), grid2((unsigned)((2 * ntiles + WARPS2D - 1) / WARPS2D));
    const typename Heat2D<T>::Consts c = consts_of<T>(h);
    swept2d_warp_kernel<T, R_PYRAMID, FOLD><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, 0, 0, tiles_x, ntiles, c);
    ++*launches;
    for (int64_t k = 0; k < K; ++k) {
        const int a = (int)(k & 1) * (W / 2), b = W / 2 - a;      // a: the alignment that shrinks in this half-cycle
        swept2d_warp_kernel<T, R_BRIDGES, FOLD><<<grid2, block, 0, st>>>(p0, p1, h->nx, h->ny, b, a, tiles_x, ntiles, c);
        if (k == K - 1) swept2d_warp_kernel<T, R_INVERTED, FOLD><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, tiles_x, ntiles, c);
        else swept2d_warp_kernel<T, R_OCTAHEDRON, FOLD><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, tiles_x, ntiles, c);
        *launches += 2;
    }
    return cudaGetLastError();
}

template <class T> cudaError_t sweep2d_w(swept2d_ctx *h, void *d_u, int W, int64_t K, cudaStream_t st, int64_t *launches) {
    if (W == 32 && h->kernel != SWEPT2D_KERNEL_SMEM)
        return h->kernel == SWEPT2D_KERNEL_COLUMN ? sweep2d_warp<T, false>(h, d_u, K, st, launches) : sweep2d_warp<T, true>(h, d_u, K, st, launches);
    switch (W) {
        case 8: return sweep2d<T, 8>(h, d_u, K, st, launches);
        case 16: return sweep2d<T, 16>(h, d_u, K, st, launches);
        case 32: return sweep2d<T, 32>(h, d_u, K, st, launches);
        default: return cudaErrorInvalidValue;
    }
}

bool pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }

}  // namespace

extern "C" int swept2d_create(swept2d_handle_t *out, int64_t nx, int64_t ny, double dx, double dt, const swept2d_params_t *p) {
    if (!out) return swept_fail(SWEPT_EINVAL, "swept2d_create: out is NULL");
    *out = nullptr;
    const int dtype = p ? p->dtype : SWEPT_F64;
    const double alpha = p ? p->alpha : 1.0;
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return swept_fail(SWEPT_EINVAL, "swept2d_create: unknown dtype %d", dtype);
    // ny / 8 rows of blocks must fit gridDim.y (65535): the classic kernel and the narrowest shared-memory tiles put rows on blockIdx.y
    if (!pow2(nx) || !pow2(ny) || nx < 8 || ny < 8 || nx > ((int64_t)1 << 20) || ny > ((int64_t)1 << 18))
        return swept_fail(SWEPT_EINVAL, "swept2d_create: nx=%lld, ny=%lld must be powers of two, nx in [8, 2^20], ny in [8, 2^18]", (long long)nx, (long long)ny);
    if (!isfinite(dx) || !isfinite(dt) || dx <= 0.0 || dt <= 0.0 || !(isfinite(alpha) && alpha > 0.0))
        return swept_fail(SWEPT_EINVAL, "swept2d_create: dx, dt and alpha must be finite and positive");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_create: no CUDA device (this library has no CPU fallback): %s", cudaGetErrorString(e)); }
    swept2d_ctx *h = new (std::nothrow) swept2d_ctx();
    if (!h) return swept_fail(SWEPT_ENOMEM, "swept2d_create: out of host memory");
    h->dtype = dtype; h->device = dev; h->kernel = SWEPT2D_KERNEL_WARP; h->nx = nx; h->ny = ny; h->dx = dx; h->dt = dt; h->alpha = alpha;
    h->launches_last = h->launches_total = 0;
    h->host_stage = nullptr;
    const double Fo = alpha * dt / (dx * dx);                     // row A0: constants on the host in double, cast once
    memset(h->cb.bytes, 0, sizeof h->cb.bytes);
    if (dtype == SWEPT_F64) { Heat2D<double>::Consts c{Fo, 1.0 - 4.0 * Fo}; memcpy(h->cb.bytes, &c, sizeof c); }
    else { Heat2D<float>::Consts c{(float)Fo, (float)(1.0 - 4.0 * Fo)}; memcpy(h->cb.bytes, &c, sizeof c); }
    h->field_bytes = (size_t)nx * (size_t)ny * elem_size(dtype);
    e = cudaMalloc(&h->work, h->field_bytes);
    if (e != cudaSuccess) {
        delete h;
        cudaGetLastError();
        return swept_fail(e == cudaErrorMemoryAllocation ? SWEPT_ENOMEM : SWEPT_ECUDA, "swept2d_create: cudaMalloc workspace: %s", cudaGetErrorString(e));
    }
    *out = h;
    return SWEPT_OK;
}

static int args2d_ok(swept2d_ctx *h, void *d_u, int64_t nsteps, const char *who) {
    if (!h) return swept_fail(SWEPT_EINVAL, "%s: NULL handle", who);
    if (!d_u) return swept_fail(SWEPT_EINVAL, "%s: d_u is NULL", who);
    if (nsteps < 0) return swept_fail(SWEPT_EINVAL, "%s: nsteps < 0", who);
    if (((uintptr_t)d_u & 15) != 0) return swept_fail(SWEPT_EINVAL, "%s: d_u must be 16-byte aligned", who);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) { cudaGetLastError(); return swept_fail(SWEPT_EINVAL, "%s: the handle was created on device %d but device %d is current", who, h->device, dev); }
    return SWEPT_OK;
}

extern "C" int naive2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, void *cuda_stream) {
    int rc = args2d_ok(h, d_u, nsteps, "naive2d_run");
    if (rc) return rc;
    int64_t launches = 0;
    const cudaError_t e = h->dtype == SWEPT_F64 ? classic2d<double>(h, d_u, nsteps, (cudaStream_t)cuda_stream, &launches)
                                                : classic2d<float>(h, d_u, nsteps, (cudaStream_t)cuda_stream, &launches);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "naive2d_run: %s", cudaGetErrorString(e)); }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

extern "C" int swept2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, int tile_width, void *cuda_stream) {
    int rc = args2d_ok(h, d_u, nsteps, "swept2d_run");
    if (rc) return rc;
    int W = tile_width;
    if (W == 0) for (W = 32; W > 8 && (W > h->nx || W > h->ny); W >>= 1) {}
    if ((W != 8 && W != 16 && W != 32) || W > h->nx || W > h->ny)
        return swept_fail(SWEPT_EINVAL, "swept2d_run: tile_width %d: must be 8, 16 or 32 and at most nx, ny", tile_width);
    const int64_t L = W / 2, K = nsteps / L, r = nsteps % L;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int64_t launches = 0;
    cudaError_t e = h->dtype == SWEPT_F64 ? classic2d<double>(h, d_u, r, st, &launches) : classic2d<float>(h, d_u, r, st, &launches);
    if (e == cudaSuccess) e = h->dtype == SWEPT_F64 ? sweep2d_w<double>(h, d_u, W, K, st, &launches) : sweep2d_w<float>(h, d_u, W, K, st, &launches);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_run: %s", cudaGetErrorString(e)); }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

// End-to-end convenience (the `e2e` measurement of bench.py --heat2d): host buffer in, host buffer out.
extern "C" int swept2d_run_host(swept2d_handle_t h, void *h_u, int64_t nsteps, int tile_width, int use_swept, void *cuda_stream) {
    if (!h) return swept_fail(SWEPT_EINVAL, "swept2d_run_host: NULL handle");
    if (!h_u) return swept_fail(SWEPT_EINVAL, "swept2d_run_host: h_u is NULL");
    if (nsteps < 0) return swept_fail(SWEPT_EINVAL, "swept2d_run_host: nsteps < 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (!h->host_stage) {
        e = cudaMalloc(&h->host_stage, h->field_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); h->host_stage = nullptr; return swept_fail(SWEPT_ENOMEM, "swept2d_run_host: cudaMalloc: %s", cudaGetErrorString(e)); }
    }
    e = cudaMemcpyAsync(h->host_stage, h_u, h->field_bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_run_host: H2D: %s", cudaGetErrorString(e)); }
    const int rc = use_swept ? swept2d_run(h, h->host_stage, nsteps, tile_width, cuda_stream) : naive2d_run(h, h->host_stage, nsteps, cuda_stream);
    if (rc) return rc;
    e = cudaMemcpyAsync(h_u, h->host_stage, h->field_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_run_host: D2H: %s", cudaGetErrorString(e)); }
    return SWEPT_OK;
}

extern "C" int swept2d_set_option(swept2d_handle_t h, int option, int value) {
    if (!h) return swept_fail(SWEPT_EINVAL, "swept2d_set_option: NULL handle");
    if (option != SWEPT2D_OPT_KERNEL || (value != SWEPT2D_KERNEL_WARP && value != SWEPT2D_KERNEL_SMEM && value != SWEPT2D_KERNEL_COLUMN))
        return swept_fail(SWEPT_EINVAL, "swept2d_set_option: unknown option %d or value %d", option, value);
    h->kernel = value;
    return SWEPT_OK;
}

extern "C" int swept2d_get_info(swept2d_handle_t h, swept2d_info_t *info) {
    if (!h || !info) return swept_fail(SWEPT_EINVAL, "swept2d_get_info: NULL argument");
    info->dtype = h->dtype; info->nx = h->nx; info->ny = h->ny;
    info->workspace_bytes = (int64_t)h->field_bytes;
    info->launches_last_call = h->launches_last; info->launches_total = h->launches_total;
    return SWEPT_OK;
}

extern "C" int swept2d_destroy(swept2d_handle_t h) {
    if (!h) return swept_fail(SWEPT_EINVAL, "swept2d_destroy: NULL handle");
    if (h->work) cudaFree(h->work);
    if (h->host_stage) cudaFree(h->host_stage);
    delete h;
    return SWEPT_OK;
}
