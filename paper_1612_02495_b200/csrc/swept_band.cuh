// swept_band.cuh -- SWEPT_OPT_CHAIN = 2: the streaming form of the wavefront swept kernels (swept_wave.cuh).
//
// In the characteristic coordinates of swept_wave.cuh (i = x + H t, j = -x + H t - 1, up to constants) the tile that
// stitches on top of a diamond's upper-LEFT edge (Fig. 2b: the next half-cycle's tile, shifted by W/2 to the
// left) continues the SAME columns i to higher rows j.  A "band" is that chain of tiles: tile (band b, phase p) sits at
// g0 = b W - p W/2 (periodic), p = 0 the upright triangle, p = q the closing inverted triangle.  A warp that keeps a band
// keeps its column state in registers for the whole swept_run: the upper-left edge is never written to or re-read from
// global memory, and -- because the lanes' skewed wavefront simply runs on from one tile into the next -- the wavefront
// fills and drains once per launch instead of once per tile (swept_wave.cuh pays 31 of every NJ + 31 iterations).
//
// What still travels through the staircase arrays (R0 = d_u, R1 = workspace, row A4 of SURVEY.md section 8(a)) is the
// upper-RIGHT edge: lane 31's row outputs of tile (b, p) are the row feed of lane 0 of tile (b+1, p+1).  They are
// flushed / fetched in chunks of 32 super-rows (one coalesced access per lane) through two small shared-memory rings,
// and ordered by one monotone counter per band, prog[b] = output chunks of band b flushed so far (release store after
// the flush, acquire load before the fetch).  Chunk c of tile (b, p) needs prog[b-1] >= (p-1) NCH + c + 1, a chunk the
// left neighbour produced a whole half-cycle earlier, so bands advance in lockstep without waiting (tiles of NJ >= 64
// super-rows; the smallest tiles, NJ = 32, run on swept_chain_kernel instead).
//
// Bands are dealt statically: band n -> SM sub-partition slot n mod G (G = blocks x 4), so every sub-partition carries
// floor or ceil(ntiles / G) bands however ntiles and the SM count divide; a warp that owns k > 1 bands runs them
// phase-major (b_0 p, b_1 p, ..., b_0 p+1, ...) and parks the idle bands' columns in shared memory: at its own first
// super-row of a tile each lane swaps its PW columns with the parked copy (k - 1 rotating buffers per warp).  Every warp
// of the grid must be resident (the host sizes the grid by occupancy and launches it cooperatively); waits are on
// strictly earlier phases of other warps, so the schedule cannot deadlock.
#pragma once
#include <type_traits>

#include "swept_wave.cuh"

namespace swept {

// SR = super-rows a lane advances per iteration.  SR = 2 runs two consecutive super-rows one point apart (point n of the
// first with point n-1 of the second: they are independent), which doubles the independent FP chains per warp -- heat has
// only D = 2 rows to interleave and its DADD -> DFMA chain per point leaves the FP64 pipe idle at 4 warps per
// sub-partition -- and halves the per-iteration overhead (shuffles, ring accesses, loop control) per update.  W = 512 runs
// four: it is the width mid-size grids (2^17..2^20 points) pick, where a few warps per SM must each fill more of the pipe
// (SR = 4 needs NJ / 4 >= 64 iterations per tile, so W = 256 stays at two and fp64 W = 1024 has no registers left for it).
// KS already interleaves D = 4 rows; two super-rows per iteration at W = 512 still raise it from 0.68 to 0.84 of the FP64 pipe.
template <class P, int PW> constexpr int band_sr() {
    if (P::H == 2 && !P::GROUPED && (PW == 16 || (PW == 32 && sizeof(typename P::real) == 4))) return 2;   // KS: W = 512, and fp32 W = 1024
    return (P::H == 1 && (PW == 16 || (PW == 32 && sizeof(typename P::real) == 4))) ? 4 : ((P::H == 1 && PW >= 8) ? 2 : 1);
}

// Lane vector.  T = float / double: a warp slot is one band.  T = float2p: a slot is TWO bands advanced in lock step by packed
// arithmetic, component x the band n, component y the band n + nslots -- exactly half a domain away, so every global address of
// the y component is the x component's address + nx/2 (mod nx).  Progress counters stay per band.
template <class T> struct LaneVec { using E = T; static constexpr int V = 1; };
template <> struct LaneVec<float2p> { using E = float; static constexpr int V = 2; };
template <class T> __device__ __forceinline__ T lv_ldcg(const typename LaneVec<T>::E *base, int64_t a, int64_t half, int64_t mask) {
    if constexpr (LaneVec<T>::V == 1) return __ldcg(base + a);
    else return float2p(__ldcg(base + a), __ldcg(base + ((a + half) & mask)));
}
template <class T> __device__ __forceinline__ void lv_stcg(typename LaneVec<T>::E *base, int64_t a, int64_t half, int64_t mask, T v) {
    if constexpr (LaneVec<T>::V == 1) __stcg(base + a, v);
    else { __stcg(base + a, v.x); __stcg(base + ((a + half) & mask), v.y); }
}
template <> __device__ __forceinline__ float2p shfl_up1<float2p>(float2p v) {
    return float2p(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1));
}

template <class P, int PW> struct BandGeom {
    using T = typename P::real;
    static constexpr int H = P::H, NC = P::NC, D = 2 * H, SR = band_sr<P, PW>();
    static constexpr int W = 32 * PW, NJ = W / D, NP = PW / D, L = W / D, CTR = W / 2;
    static constexpr int NJI = NJ / SR;                  // iterations per tile
    static constexpr int NCH = NJI / 32;                 // chunks (32 iterations) per tile
    static constexpr int CS = 32 * (PW + 1);             // one field of a parked band: lane stride PW + 1 (conflict-free)
    static constexpr int FEED = NC * 32 * SR * D;        // values: feed ring (one chunk)
    static constexpr int OUTR = NC * 64 * SR * D;        // values: output ring (two chunks)
    static constexpr int EDGE = NC * 32 * D;             // values: per-lane hand-over of the last D columns at a swap
    static constexpr int COL = NC * CS;                  // values: one parked band
    static __host__ __device__ size_t warp_values(int kmax) { return (size_t)FEED + OUTR + EDGE + (size_t)(kmax > 1 ? kmax - 1 : 0) * COL; }
};

// Block size bound per instantiation: the column state alone is NC (D + PW) values per lane, so the number of warps an SM
// can hold is set by registers; the bound tells ptxas how many registers it may use (65536 / threads).
// TIGHT: a second build of the Euler fp64 narrow-tile kernel for 16 warps x 128 registers (with a spill) instead of 8 x 255: the
// Euler kernels are bound by resident warps, so the tight build wins once the grid has more bands than 8 warps per SM can own
// (nx = 2^19, W = 256: 37 -> 44.6 GPts*steps/s) and loses below that (2^18: 36.6 -> 32.3).
template <class P, int PW> constexpr bool band_has_tight() { return P::GROUPED && sizeof(typename P::real) == 8 && PW <= 8; }

template <class P, int PW, bool TIGHT = false> constexpr int band_max_threads() {
    // (measured: heat fp64 W = 512 with four super-rows per iteration is faster at 20 warps x 96 registers with an 80-byte
    // spill than at 16 warps x 128 registers without one, so SR does not enter the estimate)
    const int est = P::NC * (2 * P::H + PW) * (int)(sizeof(typename P::real) / 4) + (P::GROUPED ? 110 : 56 + 16 * (P::H - 1));
    int warps = 65536 / (32 * est);
    warps = warps >= 4 ? (warps & ~3) : (warps < 1 ? 1 : warps);
    // KS fp64 at 32 points per lane spills at the 170 registers 12 warps leave; 8 warps with up to 255 registers run faster
    if (P::H == 2 && !P::GROUPED && sizeof(typename P::real) == 8 && PW == 32) warps = 8;
    if (TIGHT) warps = 16;
    return 32 * (warps > 32 ? 32 : warps);
}

// SR consecutive super-rows of one lane (a super-row = the D rows in which each of its PW columns is updated exactly
// once; same update order as wave_tile in swept_wave.cuh).  Super-row s runs point n at step n + s, i.e. one point behind
// super-row s-1: (s, n) needs (s, n-1) and (s-1, n) only, so the SR streams are independent instruction chains.
// recv[s] = lane l-1's newest row values after ITS super-row s; keep[s] (s < SR-1) returns this lane's row values after
// super-row s, which super-row s+1 overwrites (the caller shuffles them to lane l+1 next iteration).  tb = tier of the
// lane's first point in super-row 0; a point of tier t is updated iff lo < t <= hi (ALL: every point -- the diamond
// phases' steady state, no tier tests, no selects).
// s / k for 0 <= s, s k < 2^32 without the integer-division sequence (the quotient of a multiply-high by ceil(2^32 / k) is exact
// in that range); k = 1 -- every grid with no more bands than warps -- costs nothing.  The chunk boundaries divide local tile
// numbers by the warp's band count several times each: ncu (heat fp64, nx = 2^12) put three MUFU.RCP division sequences per boundary.
struct DivK {
    unsigned m;
    int k;
    __device__ __forceinline__ explicit DivK(int kk) : m(kk > 1 ? (unsigned)((0x100000000ull + (unsigned)kk - 1) / (unsigned)kk) : 0u), k(kk) {}
    __device__ __forceinline__ int operator()(int s) const { return k > 1 ? (int)__umulhi((unsigned)s, m) : s; }
};

template <class P, int PW, int SR, bool ALL>
__device__ __forceinline__ void band_super_rows(typename P::real (&X)[P::NC][2 * P::H + PW], const typename P::real (&recv)[SR][P::NC][2 * P::H],
                                                typename P::real (&keep)[SR][P::NC][2 * P::H], const typename P::Consts &c, const int tb,
                                                const int lo, const int hi) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC, D = 2 * H, NP = PW / D;
    T old[SR][D][NC];
    if constexpr (!P::GROUPED && H == 1 && NC == 1 && P::S == 1) {
        // Heat: the SR x D point updates of one step are independent (super-row s + 1 runs one point behind super-row s): all sums,
        // then all products, then all fused multiply-adds, in that source order, so that a warp alone on its scheduler keeps SR D
        // chains in flight instead of the two or three the point-by-point order left it (ncu, nx = 2^18: `wait` 1.25 per issue)
#pragma unroll
        for (int step = 0; step < NP + SR - 1; ++step) {
            T t[SR][D], v[SR][D], o[SR][D];
#pragma unroll
            for (int s = 0; s < SR; ++s) {
                const int n = step - s;
                if (n == 0) {
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) X[0][D - 1 - rho] = recv[s][0][rho];
                }
            }
#pragma unroll
            for (int s = 0; s < SR; ++s) {
                const int n = step - s;
                if (n < 0 || n >= NP) continue;
#pragma unroll
                for (int rho = 0; rho < D; ++rho) {
                    const int qq = (D - 1 - rho) + D * n;
                    t[s][rho] = X[0][qq + 2] + X[0][qq];
                }
            }
#pragma unroll
            for (int s = 0; s < SR; ++s) {
                const int n = step - s;
                if (n < 0 || n >= NP) continue;
#pragma unroll
                for (int rho = 0; rho < D; ++rho) v[s][rho] = c.c0 * X[0][(D - 1 - rho) + D * n + 1];
            }
#pragma unroll
            for (int s = 0; s < SR; ++s) {
                const int n = step - s;
                if (n < 0 || n >= NP) continue;
#pragma unroll
                for (int rho = 0; rho < D; ++rho) o[s][rho] = fp<T>::fma(c.Fo, t[s][rho], v[s][rho]);
            }
#pragma unroll
            for (int s = 0; s < SR; ++s) {
                const int n = step - s;
                if (n < 0 || n >= NP) continue;
                const int tt = tb + s + n;
                const bool pact = ALL ? true : (tt > lo && tt <= hi);
#pragma unroll
                for (int rho = 0; rho < D; ++rho) {
                    const int qq = (D - 1 - rho) + D * n;
                    X[0][qq + D] = pact ? o[s][rho] : X[0][qq + D];
                }
                if (n == NP - 1) {
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) keep[s][0][rho] = X[0][PW + (D - 1 - rho)];
                }
            }
        }
        return;
    }
#pragma unroll
    for (int step = 0; step < NP + SR - 1; ++step) {
#pragma unroll
        for (int s = 0; s < SR; ++s) {
            const int n = step - s;
            if (n < 0 || n >= NP) continue;
            if (n == 0) {
#pragma unroll
                for (int rho = 0; rho < D; ++rho)
#pragma unroll
                    for (int kk = 0; kk < NC; ++kk) { old[s][rho][kk] = X[kk][D - 1 - rho]; X[kk][D - 1 - rho] = recv[s][kk][rho]; }
            }
            const int t = tb + s + n;
            const bool odd = (t & 1) != 0;
            const bool pact = ALL ? true : (t > lo && t <= hi);
            if constexpr (P::GROUPED) {
                T win[NC][2 * D], out[D][NC];
#pragma unroll
                for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                    for (int m = 0; m < 2 * D; ++m) win[kk][m] = X[kk][D * n + m];
                P::group_sel(c, odd, win, old[s], out);
#pragma unroll
                for (int rho = 0; rho < D; ++rho) {
                    const int qq = (D - 1 - rho) + D * n;
#pragma unroll
                    for (int kk = 0; kk < NC; ++kk) {
                        old[s][rho][kk] = X[kk][qq + D];
                        X[kk][qq + D] = pact ? out[rho][kk] : X[kk][qq + D];
                    }
                }
            } else {
#pragma unroll
                for (int rho = 0; rho < D; ++rho) {
                    const int qq = (D - 1 - rho) + D * n;   // window X[k][qq .. qq+D], target X[k][qq+D]
                    T win[NC][2 * H + 1], out[NC];
#pragma unroll
                    for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                        for (int m = 0; m <= D; ++m) win[kk][m] = X[kk][qq + m];
                    P::stage_sel(c, odd, win, old[s][rho], out);
#pragma unroll
                    for (int kk = 0; kk < NC; ++kk) {
                        old[s][rho][kk] = X[kk][qq + D];
                        X[kk][qq + D] = pact ? out[kk] : X[kk][qq + D];
                    }
                }
            }
            if (n == NP - 1) {                            // the lane's row values after super-row s: column PW-D+r, r = D-1-rho
#pragma unroll
                for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) keep[s][kk][rho] = X[kk][PW + (D - 1 - rho)];
            }
        }
    }
}

template <class P, int PW, bool TIGHT = false>
__global__ void __launch_bounds__((band_max_threads<P, PW, TIGHT>())) swept_band_kernel(typename LaneVec<typename P::real>::E *u, typename LaneVec<typename P::real>::E *w, int64_t nx,
                                                             int ntiles /* slots: bands / V */, int q, int rt, BandGrid grid, unsigned *prog, typename P::Consts c) {
    using T = typename P::real;
    using E = typename LaneVec<T>::E;
    constexpr int V = LaneVec<T>::V;
    const int64_t half = nx / 2;                          // (V = 2) offset of the y component's band
    using Gm = BandGeom<P, PW>;
    constexpr int H = Gm::H, NC = Gm::NC, D = Gm::D, W = Gm::W, NJI = Gm::NJI, NP = Gm::NP, L = Gm::L, CTR = Gm::CTR, NCH = Gm::NCH, CS = Gm::CS, SR = Gm::SR;
    static_assert(PW % D == 0, "points per lane must be a multiple of 2H");
    static_assert((NJI & (NJI - 1)) == 0 && NJI % 32 == 0, "iterations per tile must be a power of two multiple of 32");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    const int64_t mask = nx - 1;

    // ---- which bands this warp owns: band n -> slot n % G, round n / G -> warp (round % wps) of the slot, list index round / wps
    const int first = band_first(grid, (int)blockIdx.x, warp), stride = band_stride(grid);   // bands first, first + stride, ...
    const int k = band_count(grid, (int)blockIdx.x, warp, ntiles);
    if (k == 0) return;
    // rt > 0: the remainder as a truncated closing cycle (swept_ring.cuh; reading S3'): phase q runs on to tier L + rt and
    // one more phase q + 1 runs up to tier rt
    const int nph = q + 1 + (rt > 0 ? 1 : 0);
    const int n_items = k * nph;
    const int lt_end = n_items * NJI;                     // < 2^31: the host refuses longer runs

    T *base = reinterpret_cast<T *>(smem_raw) + (size_t)warp * Gm::warp_values(grid.kmax);
    T *feed = base, *outr = feed + Gm::FEED, *edge = outr + Gm::OUTR, *col = edge + Gm::EDGE;

    auto g0_of = [&](int band, int p) -> int64_t { return ((int64_t)band * W - (int64_t)p * (W / 2)) & mask; };

    // ---- column state.  X[k][0..D) = copy of lane l-1's last D columns, X[k][D + i] = own column i
    T X[NC][D + PW];
    {
        const int64_t g0 = g0_of(first, 0);
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int i = 0; i < PW; ++i) X[kk][D + i] = lv_ldcg<T>(u + (int64_t)kk * nx, (g0 + lane * PW + i) & mask, half, mask);
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int d = 0; d < D; ++d) X[kk][d] = shfl_up1(X[kk][PW + d]);
        // parked bands m = 1..k-1 start from the flat field too; band m is first swapped in at transition m - 1
        for (int m = 1; m < k; ++m) {
            const int64_t gm = g0_of(first + m * stride, 0);
            T *buf = col + (size_t)(m - 1) * Gm::COL;
            for (int i = lane; i < W; i += 32)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk) buf[kk * CS + i + i / PW] = lv_ldcg<T>(u + (int64_t)kk * nx, (gm + i) & mask, half, mask);
        }
        for (int i = lane; i < Gm::FEED; i += 32) feed[i] = T(0);
        __syncwarp();
    }

    const DivK divk(k);
    int p_cur = 0, lo = L, hi = 0x3fffffff;              // this lane's tile: phase, and the tiers (lo, hi] it updates
    bool interior = false;                               // p_cur is a diamond phase: every point of the tile is updated
    auto set_phase = [&](int s) {
        p_cur = divk(s);
        lo = p_cur == 0 ? L : 0;
        hi = p_cur < q ? 0x3fffffff : (p_cur == q ? L + rt : rt);
        interior = p_cur > 0 && p_cur < q;
    };
    // This lane enters tile s >= 1 of a warp that owns k > 1 bands: swap its PW columns with the parked copy of the incoming
    // band (transition s-1 uses buffer (s-1) mod (k-1)), and hand the incoming band's last D columns -- before this lane's
    // first super-row changes them -- to lane l+1, which swaps one iteration later.
    auto swap_bands = [&](int s) {
        T *buf = col + (size_t)((s - 1) % (k - 1)) * Gm::COL;
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int i = 0; i < PW; ++i) {
                T *a = buf + kk * CS + lane * (PW + 1) + i;
                const T t = *a;
                *a = X[kk][D + i];
                X[kk][D + i] = t;
            }
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int d = 0; d < D; ++d) {
                edge[(kk * 32 + lane) * D + d] = X[kk][PW + d];
                if (lane > 0) X[kk][d] = edge[(kk * 32 + lane - 1) * D + d];
            }
    };
    T keep[SR][NC][D];                                   // this lane's row values after each super-row of its last iteration
#pragma unroll
    for (int sr = 0; sr < SR; ++sr)
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int rho = 0; rho < D; ++rho) keep[sr][kk][rho] = X[kk][PW + (D - 1 - rho)];

    for (int K0 = 0; K0 < lt_end + 31; K0 += 32) {
        // ---- chunk boundary (warp-uniform).  Lane 0 first issues the acquire load of the left band's counter for the chunk it is
        // about to fetch, so that its round trip to L2 overlaps the flush below; (1) flush the row outputs lane 31 produced for
        // local times [K0-64, K0-32); (2) fetch the row feed of lane 0 for local times [K0, K0+32).
        __syncwarp();
        const int sf = K0 / NJI, pf = divk(sf), mf = sf - pf * k;
        const bool fetch = K0 < lt_end && pf > 0;
        // (V = 2: lane 0 polls / releases the counter of the slot's band, lane 1 that of the band half a domain away)
        const int nbands = ntiles * V;
        const int bandf = first + mf * stride, bandl = bandf + (lane < V ? lane : 0) * ntiles, left = bandl == 0 ? nbands - 1 : bandl - 1;
        unsigned seen = 0;
        if (fetch && lane < V) seen = ld_acquire_gpu(prog + left);
        const int lt0 = K0 - 64;
        if (lt0 >= 0 && lt0 < lt_end) {
            const int s = lt0 / NJI, p = divk(s), m = s - p * k;
            if (p < nph - 1) {
                const int band = first + m * stride;
                const int64_t g0 = g0_of(band, p);
#pragma unroll
                for (int sr = 0; sr < SR; ++sr) {
                    const int J = SR * ((lt0 & (NJI - 1)) + lane) + sr;        // super-row: rows j = J D + rho hold tier L + J
                    E *dst = (J & 1) ? w : u;
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) {
                        const int64_t g = (g0 + W - 1 - H * J - rho) & mask;
#pragma unroll
                        for (int kk = 0; kk < NC; ++kk)
                            lv_stcg<T>(dst + (int64_t)kk * nx, g, half, mask, outr[((kk * 64 + ((lt0 + lane) & 63)) * SR + sr) * D + rho]);
                    }
                }
                // the warp barrier orders every lane's stores before lane 0's release (cumulative at gpu scope)
                __syncwarp();
                if (lane < V) st_release_gpu(prog + band + lane * ntiles, (unsigned)(p * NCH + (lt0 & (NJI - 1)) / 32 + 1));
            }
        }
        if (K0 < lt_end) {
            if (fetch) {
                const unsigned need = (unsigned)((pf - 1) * NCH + (K0 & (NJI - 1)) / 32 + 1);
                bool dead = false;
                if (lane < V) {
                    unsigned ns = 20;
                    SpinWatch polls;
                    while (seen < need) {
                        __nanosleep(ns);
                        if (ns < 320) ns *= 2;
                        seen = ld_acquire_gpu(prog + left);
                        if (spin_gives_up(polls, abort_word_of(prog))) { dead = true; break; }
                    }
                }
                __syncwarp();                                     // orders the other lanes' loads behind the polling lanes' acquire
                if (__any_sync(0xffffffffu, dead)) return;
                const int64_t g0 = g0_of(bandf, pf);
#pragma unroll
                for (int sr = 0; sr < SR; ++sr) {
                    const int J = SR * ((K0 & (NJI - 1)) + lane) + sr;         // row j = J D + rho is fed from tier J of the left tile's right edge
                    const E *src = (J & 1) ? w : u;
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) {
                        const int64_t g = (g0 + CTR - H * J - rho - 1) & mask;
#pragma unroll
                        for (int kk = 0; kk < NC; ++kk) feed[((kk * 32 + lane) * SR + sr) * D + rho] = lv_ldcg<T>(src + (int64_t)kk * nx, g, half, mask);
                    }
                }
            }
            __syncwarp();
        }

        // ---- the chunk's 32 iterations.  Steady chunk: every lane is, for the whole chunk, inside diamond tiles (the tiles
        // of local times K0-31 and K0+31 are both diamond phases) -- nothing depends on the phase; in the first chunk of a tile
        // the lanes of a warp with k > 1 bands swap columns, each at its own iteration.
        bool steady = K0 >= 31 && K0 + 31 < lt_end;
        const bool swapchunk = k > 1 && (K0 & (NJI - 1)) == 0;
        if (steady) {
            const int pa = divk((K0 - 31) / NJI), pb = divk((K0 + 31) / NJI);
            steady = pa > 0 && pb < q;
        }
        if (steady) {
            // two instances of the loop: the chunk in which lanes swap bands carries the swap and a warp barrier per iteration,
            // the others (7 of 8 at W = 1024) stay free of both
            constexpr bool ONE_LOOP = P::GROUPED;
            auto steady_chunk = [&](auto swap_tag) {
                constexpr bool SWAP = decltype(swap_tag)::value;
                int J = (K0 - lane) & (NJI - 1);
                const T *fp = feed;
                T *op = outr + ((K0 - 31) & 63) * SR * D;     // lane 31's slot of local time K0 - 31
#pragma unroll 1
                for (int it = 0; it < 32; ++it) {
                    T recv[SR][NC][D];
#pragma unroll
                    for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                            for (int rho = 0; rho < D; ++rho) {
                                const T f = fp[(kk * 32 * SR + sr) * D + rho];
                                const T r = shfl_up1(keep[sr][kk][rho]);
                                recv[sr][kk][rho] = lane == 0 ? f : r;
                            }
                    if (SWAP && (!ONE_LOOP || swapchunk) && J == 0) swap_bands((K0 + it - lane) / NJI);
                    band_super_rows<P, PW, SR, true>(X, recv, keep, c, lane * NP + SR * J + 1, 0, 0);
                    if (lane == 31) {
#pragma unroll
                        for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                            for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                                for (int rho = 0; rho < D; ++rho) op[(kk * 64 * SR + sr) * D + rho] = keep[sr][kk][rho];
                    }
                    J = (J + 1) & (NJI - 1);
                    fp += SR * D;
                    op += SR * D;
                    if (op == outr + 64 * SR * D) op = outr;
                    if (SWAP && (!ONE_LOOP || swapchunk)) __syncwarp();   // lane l+1 reads the hand-over slot lane l wrote this iteration
                }
            };
            // Euler's loop body is 40 KB of code: two instances of it, taken in turn by a warp with k > 1 bands, thrash the instruction
            // cache (ncu, fp64, nx = 2^20: `no_instruction` the top stall, 28 % of the samples) -- one instance, the swap a run-time flag
            // (also for a warp with one band, which never swaps: warps with one and with two bands share an SM, and the plain instance
            // beside the merged one is the same 84 KB again -- measured: ring 2^19 36.4 -> 26.6)
            if (ONE_LOOP || swapchunk) steady_chunk(std::true_type{});
            else steady_chunk(std::false_type{});
            continue;
        }
        {
            const int ltc = K0 - lane;                    // phase of the tile this lane is in when the chunk starts
            if (ltc >= 0) set_phase((ltc < lt_end ? ltc : lt_end - 1) / NJI);
        }
        for (int K = K0; K < K0 + 32 && K < lt_end + 31; ++K) {
            const int lt = K - lane;                      // this lane's local time: tile lt / NJI of the warp's list, iteration lt % NJI
            const bool act = lt >= 0 && lt < lt_end;
            const int J = lt & (NJI - 1);
            // lane 0's row inputs come from the feed ring (all lanes read the same address: one broadcast)
            T fd[SR][NC][D];
#pragma unroll
            for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) fd[sr][kk][rho] = feed[((kk * 32 + (K & 31)) * SR + sr) * D + rho];
            // lane l-1's row values after each super-row of its previous iteration (= the super-rows this lane runs now)
            T recv[SR][NC][D];
#pragma unroll
            for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) recv[sr][kk][rho] = shfl_up1(keep[sr][kk][rho]);
            if (act && J == 0) {
                // ---- this lane enters a new tile: update its phase; with k > 1 swap columns with the parked band
                const int s = lt / NJI;
                set_phase(s);
                if (k > 1 && s > 0) swap_bands(s);
            }
            const bool fed = lane == 0 && p_cur > 0;
#pragma unroll
            for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) recv[sr][kk][rho] = fed ? fd[sr][kk][rho] : recv[sr][kk][rho];
            const int tb = lane * NP + SR * J + 1;        // tier of the lane's first point in the first super-row
            if (__all_sync(0xffffffffu, act && interior)) {
                band_super_rows<P, PW, SR, true>(X, recv, keep, c, tb, lo, hi);
            } else if (act) {
                band_super_rows<P, PW, SR, false>(X, recv, keep, c, tb, lo, hi);
            }
            if (act && lane == 31 && p_cur < nph - 1) {   // the row outputs of the SR super-rows
#pragma unroll
                for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                    for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                        for (int rho = 0; rho < D; ++rho) outr[((kk * 64 + (lt & 63)) * SR + sr) * D + rho] = keep[sr][kk][rho];
            }
            __syncwarp();
        }
    }

    // ---- With a truncated closing cycle phase q has a consumer, and its row outputs lie in the span the flat field is stored over:
    // wait until every warp of the grid is through its last tile (swept_ring.cuh explains the hazard)
    if (rt > 0) {
        bool dead = false;
        __syncwarp();
        if (lane == 0) {
            const int stride_all = band_stride(grid);
            const unsigned total = (unsigned)(ntiles < stride_all ? ntiles : stride_all);
            __threadfence();
            atomicAdd(prog + ntiles * V, 1u);
            unsigned ns = 100;
            SpinWatch polls;
            while (ld_acquire_gpu(prog + ntiles * V) < total) {
                __nanosleep(ns);
                if (ns < 6400) ns *= 2;
                if (spin_gives_up(polls, abort_word_of(prog))) { dead = true; break; }
            }
        }
        __syncwarp();                                     // orders the other lanes' loads behind the polling lanes' acquire
        if (__any_sync(0xffffffffu, dead)) return;
    }
    // ---- all phases done: column i of a band ended at x = g0(band, q) + i - H rt; registers hold band k-1's flat values, the
    // parked copies the other bands'
    {
        const int64_t sh = (rt > 0 ? W / 2 : 0) - H * rt + nx;   // g0(q) = g0(last phase) + W/2 when the extra phase ran
        const int64_t g0 = g0_of(first + (k - 1) * stride, nph - 1) + sh;
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int i = 0; i < PW; ++i) lv_stcg<T>(u + (int64_t)kk * nx, (g0 + lane * PW + i) & mask, half, mask, X[kk][D + i]);
        for (int m = 0; m + 1 < k; ++m) {
            const int64_t gm = g0_of(first + m * stride, nph - 1) + sh;
            const T *buf = col + (size_t)(((nph - 1) * k + m) % (k - 1)) * Gm::COL;   // band m's last tile was swapped out at transition (nph-1) k + m
            for (int i = lane; i < W; i += 32)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk) lv_stcg<T>(u + (int64_t)kk * nx, (gm + i) & mask, half, mask, buf[kk * CS + i + i / PW]);
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
// Size the grid: one block per SM, as many warps as the kernel's registers allow (all must be resident), bands dealt
// round-robin over the SM sub-partitions.  Returns false if the launch-free band schedule does not fit (too few
// bands to spread over two warps, or the parked bands exceed shared memory): the caller falls back to swept_chain_kernel.
template <class P, int PW, bool TIGHT = false>
bool band_grid(int64_t nx, int sm_count, int max_smem, int max_warps, BandGrid *out, size_t *smem_bytes) {
    using Gm = BandGeom<P, PW>;
    using T = typename P::real;
    constexpr int V = LaneVec<T>::V;
    if ((nx / Gm::W) % V != 0) return false;
    const int64_t ntiles64 = nx / Gm::W / V;                      // warp slots (V bands each)
    // One chunk per tile (NJI = 32): lane 0 would need, at the start of a tile, the chunk its left neighbour's lane 31 is
    // still 31 super-rows from finishing -- with every band in lockstep that is a cycle of waits, not a bubble
    if (Gm::NCH < 2) return false;
    if (ntiles64 < 2 || ntiles64 > (1 << 24)) return false;
    const int ntiles = (int)ntiles64;
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, swept_band_kernel<P, PW, TIGHT>) != cudaSuccess) { cudaGetLastError(); return false; }
    int regs = fa.numRegs < 16 ? 16 : fa.numRegs;
    regs = (regs + 7) & ~7;                                       // allocation granularity: 8 registers per thread
    int wmax = 65536 / (regs * 32);
    if (wmax > 32) wmax = 32;
    if (wmax > band_max_threads<P, PW, TIGHT>() / 32) wmax = band_max_threads<P, PW, TIGHT>() / 32;
    if (max_warps > 0 && wmax > max_warps) wmax = max_warps;    // SWEPT_OPT_BLOCKS_PER_SM x 4 warps: fewer resident warps on request
    static const int cand[] = {32, 28, 24, 20, 16, 12, 8, 4, 2, 1};
    int wneed = 32;                                               // smallest block that gives every band its own warp
    for (int wpb : cand)
        if ((int64_t)sm_count * wpb >= ntiles64) wneed = wpb;
    for (int wpb : cand) {
        if (wpb > wmax || wpb > wneed) continue;
        const BandGrid g = band_layout(ntiles, sm_count, wpb);
        if (g.G < 2) continue;
        const size_t smem = (size_t)wpb * Gm::warp_values(g.kmax) * sizeof(T);
        if (smem > (size_t)max_smem) continue;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, swept_band_kernel<P, PW, TIGHT>, wpb * 32, smem) != cudaSuccess) { cudaGetLastError(); continue; }
        if (per_sm < 1) continue;
        *out = g;
        *smem_bytes = smem;
        return true;
    }
    return false;
}

// `sync` = prog[ntiles] (zeroed here).  Returns cudaErrorNotSupported when the band schedule does not fit.
template <class P, int PW, bool TIGHT = false>
cudaError_t wave_band_pw(void *u, void *w, int64_t nx, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps,
                         cudaStream_t st) {
    using T = typename P::real;
    using Gm = BandGeom<P, PW>;
    if constexpr (!TIGHT && band_has_tight<P, PW>()) {
        // more bands than the roomy build has warps, and no more than the tight build has (one band per warp: its spills make
        // the band swaps of k > 1 slower than the roomy build's)
        if (nx / Gm::W > (int64_t)sm_count * (band_max_threads<P, PW, false>() / 32) && nx / Gm::W <= (int64_t)sm_count * (band_max_threads<P, PW, true>() / 32))
            return wave_band_pw<P, PW, true>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
    }
    BandGrid g;
    size_t smem = 0;
    if (q < 0 || (q == 0 && rt == 0) || rt < 0 || rt >= Gm::L || q > (1 << 24) / Gm::NCH || !band_grid<P, PW, TIGHT>(nx, sm_count, max_smem, max_warps, &g, &smem))
        return cudaErrorNotSupported;
    if ((int64_t)(q + 2) * g.kmax * Gm::NJI >= ((int64_t)1 << 30)) return cudaErrorNotSupported;   // the kernel's local time is an int
    using E = typename LaneVec<T>::E;
    constexpr int V = LaneVec<T>::V;
    typename P::Consts c;
    if constexpr (V == 1) c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    else c = P::expand(cb.bytes);                                 // the scalar problem's constants, both components
    const int nbands = (int)(nx / Gm::W), ntiles = nbands / V;    // ntiles: warp slots
    cudaError_t e = cudaMemsetAsync(sync, 0, sizeof(unsigned) * (size_t)(nbands + 1), st);   // prog[nbands] + the end-of-run arrival count
    if (e != cudaSuccess) return e;
    // Cooperative launch: the warps wait on one another, so the whole grid must be resident at once -- also when another
    // stream's kernel shares the device (a plain launch could leave two such grids each half scheduled, waiting forever).
    E *up = (E *)u, *wp = (E *)w;
    int qi = (int)q, nt = ntiles, rti = rt;
    unsigned *pr = (unsigned *)sync;
    typename P::Consts cc = c;
    void *args[] = {&up, &wp, &nx, &nt, &qi, &rti, &g, &pr, &cc};
    return cudaLaunchCooperativeKernel((const void *)swept_band_kernel<P, PW, TIGHT>, dim3((unsigned)g.nblocks), dim3((unsigned)(g.wpb * 32)), args, smem, st);
}

template <class P, int PW> cudaError_t band_prepare_pw(int max_smem) {
    if constexpr (band_has_tight<P, PW>()) {
        cudaError_t e = cudaFuncSetAttribute(swept_band_kernel<P, PW, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e != cudaSuccess) return e;
    }
    return cudaFuncSetAttribute(swept_band_kernel<P, PW>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}

}  // namespace swept
