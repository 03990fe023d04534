// swept_wave.cuh -- SWEPT_KERNEL_WAVE: the B200 design of the swept kernels.  One WARP owns one tile of W = 32*PW
// points; the tile's values live in registers, neighbouring lanes talk through one warp shuffle per tier row, and
// there is no block barrier and no shared-memory traffic in the inner loop (generalises the paper's register-only
// one-warp node, which kept idle lanes and a 32-point node).
//
// Geometry.  A diamond (Fig. 1b) in tile-local (x, t), t = tier, is the square 0 <= i, j < W in the
// characteristic coordinates
//     i = (x - c) + H t + (.5 - .5),  j = -(x - c) + H t - 1      <=>   x = c + (i - j - 1)/2,  t = (i + j + 1)/(2H),
// (c = W/2), restricted to the lattice (i + j + 1) = 0 mod 2H.  The stencil of point (i, j) is the anti-diagonal
// (i-2H+m, j-m), m = 0..2H, of the previous tier; the final stage of a two-stage scheme also reads (i-2H, j-2H).  All
// dependencies point to lower i and lower j.  Lane l owns the PW columns [l*PW, (l+1)*PW) and sweeps the rows j upwards;
// per row it needs ONE new value from lane l-1 (that lane's newest value of the same row), so lanes run as a
// wavefront, lane l one "super-row" (D = 2H rows, in which every column is updated exactly once) behind lane l-1.
// Every lane is busy in every iteration except while the wavefront fills and drains (31 of W/D + 31 iterations) --
// the half-idle lanes of a one-thread-per-point triangle are gone.
//   rows j < 0      (initial column state)  = right halves of the staircase rows R0/R1   (lower-right edge, Fig. 2b)
//   columns i < 0   (fed to lane 0 per row) = left halves of R0/R1                        (lower-left edge)
//   last D rows     (final column state)    = left halves of the new R0/R1               (upper-left edge)
//   last D columns  (lane 31, one per row)  = right halves of the new R0/R1              (upper-right edge)
// which is exactly the in-place staircase exchange of swept_smem.cu (row A4), so both kernel families interoperate.
// MODE_UP computes only the points above the anti-diagonal t = L (the tile's initial row, x = i), MODE_DOWN only those
// up to it.
#pragma once
#include "internal.h"
#include "stencils.cuh"

namespace swept {

// Global index of tile-local position g (which may lie up to W/2 + h outside [0, nx)).  Periodic: `& (nx-1)`.
// Insulated ends (INS; the paper's heat problem, Eq. 9, reading G7 of DESIGN.md: the ghost
// value is the adjacent interior value, T_0 = T_1): a tile that straddles an end of the rod -- the paper's "node split
// across the spatial boundary" -- reads the mirror image -1-g / 2nx-1-g, computes the whole (symmetric)
// diamond and stores only the positions inside the rod.
template <bool INS> __device__ __forceinline__ int64_t dom_map(int64_t g, int64_t nx) {
    if (!INS) return g & (nx - 1);
    return g < 0 ? -1 - g : (g >= nx ? 2 * nx - 1 - g : g);
}
template <bool INS> __device__ __forceinline__ bool dom_in(int64_t g, int64_t nx) { return !INS || (g >= 0 && g < nx); }

template <class T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// Staircase loads/stores.  CG = true (chained persistent kernel): cache at L2 only, because another SM may have
// rewritten the line since this SM last read it (the flag acquire orders the accesses, .cg keeps L1 out of it).
template <bool CG, class T> __device__ __forceinline__ T ld_stair(const T *p) { return CG ? __ldcg(p) : *p; }
template <bool CG, class T> __device__ __forceinline__ void st_stair(T *p, T v) { if (CG) __stcg(p, v); else *p = v; }

// One tile (one warp): g0 = global index of the tile's first point (before the periodic wrap), io = the warp's
// shared-memory row buffer of NC*W values.
template <class P, int PW, int MODE, bool CG, bool INS = false>
__device__ __forceinline__ void wave_tile(typename P::real *u, typename P::real *w, const int64_t nx, const int64_t g0,
                                          typename P::real *io, const typename P::Consts &c, const int lane) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC, D = 2 * H;
    constexpr int W = 32 * PW, NJ = W / D, NP = PW / D, L = W / D, CTR = W / 2;
    static_assert(PW % D == 0, "points per lane must be a multiple of 2H");

    // X[k][0..D) = copy of lane l-1's last D columns, X[k][D + q] = own column q
    T X[NC][D + PW];

    if (MODE == MODE_UP) {
#pragma unroll
        for (int k = 0; k < NC; ++k)
#pragma unroll
            for (int q = 0; q < PW; ++q) X[k][D + q] = ld_stair<CG>(u + (int64_t)k * nx + dom_map<INS>(g0 + lane * PW + q, nx));
    } else {
        // column i = 2H m + r starts from tier m of the right neighbour triangle's left edge: R_{m&1}[c + H m + r]
#pragma unroll
        for (int q = 0; q < PW; ++q) {
            const int m = lane * NP + q / D, r = q % D;
            const T *src = (m & 1) ? w : u;
            const int64_t g = dom_map<INS>(g0 + CTR + H * m + r, nx);
#pragma unroll
            for (int k = 0; k < NC; ++k) X[k][D + q] = ld_stair<CG>(src + (int64_t)k * nx + g);
        }
        // row j = 2H m + rho is fed from tier m of the left neighbour triangle's right edge: R_{m&1}[c - H m - rho - 1]
        for (int j = lane; j < W; j += 32) {
            const int m = j / D, rho = j % D;
            const T *src = (m & 1) ? w : u;
            const int64_t g = dom_map<INS>(g0 + CTR - H * m - rho - 1, nx);
#pragma unroll
            for (int k = 0; k < NC; ++k) io[k * W + j] = ld_stair<CG>(src + (int64_t)k * nx + g);
        }
        __syncwarp();
    }
#pragma unroll
    for (int k = 0; k < NC; ++k)
#pragma unroll
        for (int d = 0; d < D; ++d) X[k][d] = shfl_up1(X[k][PW + d]);

    for (int K = 0; K < NJ + 31; ++K) {
        const int J = K - lane;                       // this lane's super-row
        const bool act = (unsigned)J < (unsigned)NJ;
        const int tb = lane * NP + J + 1;             // tier of the lane's first point in every row of the super-row
        T feed[NC][D];
        if (MODE != MODE_UP) {
            const int fj = (K < NJ ? K : NJ - 1) * D;
#pragma unroll
            for (int k = 0; k < NC; ++k)
#pragma unroll
                for (int d = 0; d < D; ++d) feed[k][d] = io[k * W + fj + d];
        }
        // Lane l-1's newest value of row rho is its column PW-D+r (r = D-1-rho), last written one super-row ago and not
        // yet overwritten, so all D row inputs can be fetched before any of this super-row's updates.
        T recv[NC][D];
#pragma unroll
        for (int rho = 0; rho < D; ++rho)
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                recv[k][rho] = shfl_up1(X[k][PW + (D - 1 - rho)]);
                if (MODE != MODE_UP) recv[k][rho] = (lane == 0) ? feed[k][rho] : recv[k][rho];
            }
        if (act) {
            // Point n of row rho reads this super-row's point n-1 of rows <= rho and the previous super-row's values of
            // the columns rows > rho will write at point n: looping n outside, rho inside keeps the in-place update
            // correct and leaves the D points of one n independent of each other (instruction-level parallelism D).
            T old[D][NC];
#pragma unroll
            for (int rho = 0; rho < D; ++rho)
#pragma unroll
                for (int k = 0; k < NC; ++k) { old[rho][k] = X[k][D - 1 - rho]; X[k][D - 1 - rho] = recv[k][rho]; }
#pragma unroll
            for (int n = 0; n < NP; ++n) {
                const int t = tb + n;
                const bool odd = (t & 1) != 0;
                const bool pact = (MODE == MODE_DIAMOND) ? true : (MODE == MODE_UP ? (t > L) : (t <= L));
                if constexpr (P::GROUPED) {
                    // the D points of this n lie on one tier at neighbouring x and read X[k][D n .. D n + 2D) only, none of
                    // which another of them writes before reading: one call that shares work between them
                    T win[NC][2 * D], out[D][NC];
#pragma unroll
                    for (int k = 0; k < NC; ++k)
#pragma unroll
                        for (int m = 0; m < 2 * D; ++m) win[k][m] = X[k][D * n + m];
                    P::group_sel(c, odd, win, old, out);
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) {
                        const int q = (D - 1 - rho) + D * n;
#pragma unroll
                        for (int k = 0; k < NC; ++k) {
                            old[rho][k] = X[k][q + D];
                            X[k][q + D] = pact ? out[rho][k] : X[k][q + D];
                        }
                    }
                } else {
#pragma unroll
                for (int rho = 0; rho < D; ++rho) {
                    const int q = (D - 1 - rho) + D * n;   // row residue r = D-1-rho; window X[k][q .. q+D], target X[k][q+D]
                    T win[NC][2 * H + 1], out[NC];
#pragma unroll
                    for (int k = 0; k < NC; ++k)
#pragma unroll
                        for (int m = 0; m <= D; ++m) win[k][m] = X[k][q + m];
                    P::stage_sel(c, odd, win, old[rho], out);
#pragma unroll
                    for (int k = 0; k < NC; ++k) {
                        old[rho][k] = X[k][q + D];
                        X[k][q + D] = pact ? out[k] : X[k][q + D];
                    }
                }
                }
            }
            if (MODE != MODE_DOWN && lane == 31) {    // the row outputs: newest value of row rho is column PW-D+r
#pragma unroll
                for (int k = 0; k < NC; ++k)
#pragma unroll
                    for (int rho = 0; rho < D; ++rho) io[k * W + J * D + rho] = X[k][PW + (D - 1 - rho)];
            }
        }
    }

    if (MODE == MODE_DOWN) {
#pragma unroll
        for (int k = 0; k < NC; ++k)
#pragma unroll
            for (int q = 0; q < PW; ++q)
                if (dom_in<INS>(g0 + lane * PW + q, nx)) st_stair<CG>(u + (int64_t)k * nx + dom_map<INS>(g0 + lane * PW + q, nx), X[k][D + q]);
    } else {
        // final column state: column i = 2H m + r holds tier L+m at x = H m + r  -> R_{m&1}[H m + r]
#pragma unroll
        for (int q = 0; q < PW; ++q) {
            const int m = lane * NP + q / D, r = q % D;
            T *dst = (m & 1) ? w : u;
            const int64_t g = dom_map<INS>(g0 + H * m + r, nx);
            if (dom_in<INS>(g0 + H * m + r, nx))
#pragma unroll
                for (int k = 0; k < NC; ++k) st_stair<CG>(dst + (int64_t)k * nx + g, X[k][D + q]);
        }
        __syncwarp();
        // lane 31's row outputs: row j = 2H m + rho holds tier L+m at x = W-1-H m-rho -> R_{m&1}[W - 1 - H m - rho]
        for (int j = lane; j < W; j += 32) {
            const int m = j / D, rho = j % D;
            T *dst = (m & 1) ? w : u;
            const int64_t g = dom_map<INS>(g0 + W - 1 - H * m - rho, nx);
            if (dom_in<INS>(g0 + W - 1 - H * m - rho, nx))
#pragma unroll
                for (int k = 0; k < NC; ++k) st_stair<CG>(dst + (int64_t)k * nx + g, io[k * W + j]);
        }
    }
}

// One launch per phase (SWEPT_OPT_CHAIN = 0): stream order between the launches is the only synchronisation.
// INS (insulated ends): a shifted launch (offset = W/2) has ntiles + 1 tiles, tile j on [jW - W/2, jW + W/2); tiles 0 and
// ntiles straddle the ends of the rod (see dom_map).
template <class P, int PW, int MODE, bool INS = false>
__global__ void __launch_bounds__(256) swept_wave_kernel(typename P::real *u, typename P::real *w, int64_t nx, int64_t offset,
                                                          int ntiles, typename P::Consts c) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    const int tile = (int)blockIdx.x * (int)(blockDim.x >> 5) + warp;
    if (tile >= ntiles) return;                      // whole warps only
    T *io = reinterpret_cast<T *>(smem_raw) + (size_t)warp * P::NC * W;   // io[k*W + j]: row feed in, right edge out
    const int64_t g0 = (INS && offset != 0) ? (int64_t)tile * W - W / 2 : (int64_t)tile * W + offset;
    wave_tile<P, PW, MODE, false, INS>(u, w, nx, g0, io, c, lane);
}

// ---- launch-free sweep (SWEPT_OPT_CHAIN = 1) ----------------------------
// ONE launch runs all q half-cycles: phase 0 = upright triangles (offset 0), phases 1..q-1 = diamonds (offset W/2, 0,
// W/2, ...), phase q = closing inverted triangles.  Work items (phase, tile) are handed out in phase-major order by an
// atomic counter; a warp that draws (p, t) waits until the two tiles of phase p-1 it stitches together (PAPER.md:86,
// Fig. 2b: tile slots t and t+1 when phase p is the shifted one, t-1 and t otherwise) have published their staircases:
// done[slot] = number of phases slot has completed (release store after the tile's last global store, acquire load
// before the next tile's first global load).  Those two are the only tiles whose output (p, t) reads or overwrites
// (DESIGN.md section 5.5), so no other ordering is needed, and because items are drawn in dependency order by warps
// that are already running, the item with the smallest id in flight never waits: no co-residency requirement, no
// grid-wide barrier.  Phase p+1 starts on the SMs that run out of phase-p tiles, so there is no tail between
// half-cycles, and at small nx the cost of a kernel launch per half-cycle is gone.
__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned *p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Bounded waits.  The launch-free kernels wait on flags / counters that other warps of the SAME launch publish; a flag
// that never comes (a grid that is not fully resident, a handle misused from two host threads) would otherwise spin for ever
// and take the GPU with it.  Every SPIN_CHECK polls a waiting warp looks at the clock and at the handle's abort word -- the 4
// bytes SYNC_HEADER bytes before the sync area the helpers zero; after SPIN_LIMIT_NS of waiting it sets that word itself.
// A warp that sees the word set leaves the kernel; the host reports SWEPT_ECUDA from the next call on the handle (api.cu).
// The result of such a run is garbage.
struct SpinWatch { unsigned polls = 0; unsigned long long t0 = 0; };
constexpr unsigned SPIN_CHECK = 1024;
constexpr unsigned long long SPIN_LIMIT_NS = 4000000000ull;
__device__ __forceinline__ unsigned *abort_word_of(void *sync_area) { return reinterpret_cast<unsigned *>(reinterpret_cast<char *>(sync_area) - SYNC_HEADER); }
__device__ __forceinline__ bool spin_gives_up(SpinWatch &sw, unsigned *abortw) {
    if ((++sw.polls & (SPIN_CHECK - 1)) != 0) return false;
    if (*reinterpret_cast<volatile unsigned *>(abortw) != 0) return true;
    unsigned long long now;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
    if (sw.t0 == 0) { sw.t0 = now; return false; }
    if (now - sw.t0 < SPIN_LIMIT_NS) return false;
    atomicExch(abortw, 1u);
    return true;
}

// Launch bounds of the tile-flag kernel: the Euler kernels are bound by resident warps, so the narrow
// Euler tiles are compiled for 4 blocks of 4 warps per SM (128 registers, a 200-byte spill for fp64 at 8 points per lane:
// 29.5 GPts*steps/s at 2 blocks, 36.2 at 3, 37.2 at 4); everything else keeps 256 threads x 1 block.
template <class P, int PW> constexpr bool chain_tight() { return P::GROUPED && sizeof(typename P::real) == 8 && PW <= 8; }   // Euler fp64, W <= 256 (fp32 W = 512 is slower that way)
template <class P, int PW> constexpr int chain_max_threads() { return chain_tight<P, PW>() ? 128 : 256; }
template <class P, int PW> constexpr int chain_min_blocks() { return chain_tight<P, PW>() ? 4 : 1; }

template <class P, int PW>
__global__ void __launch_bounds__((chain_max_threads<P, PW>()), (chain_min_blocks<P, PW>())) swept_chain_kernel(typename P::real *u, typename P::real *w, int64_t nx, int ntiles, int q,
                                                           unsigned long long *counter, unsigned *done, typename P::Consts c) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    T *io = reinterpret_cast<T *>(smem_raw) + (size_t)warp * P::NC * W;
    const unsigned long long total = (unsigned long long)(q + 1) * (unsigned long long)ntiles;
    for (;;) {
        unsigned long long id = 0;
        if (lane == 0) id = atomicAdd(counter, 1ull);
        id = __shfl_sync(0xffffffffu, id, 0);
        if (id >= total) break;
        const int p = (int)(id / (unsigned long long)ntiles);
        const int t = (int)(id - (unsigned long long)p * (unsigned long long)ntiles);
        if (p > 0) {
            bool dead = false;
            if (lane < 2) {
                int slot = t;
                if (lane == 1) slot = (p & 1) ? (t + 1 == ntiles ? 0 : t + 1) : (t == 0 ? ntiles - 1 : t - 1);
                unsigned ns = 20;
                    SpinWatch polls;
                while (ld_acquire_gpu(done + slot) < (unsigned)p) {
                    __nanosleep(ns);
                    if (ns < 640) ns *= 2;
                    if (spin_gives_up(polls, abort_word_of(counter))) { dead = true; break; }
                }
            }
            __syncwarp();                                     // orders the other lanes' loads behind the polling lanes' acquire
            if (__any_sync(0xffffffffu, dead)) return;
        }
        const int64_t g0 = (int64_t)t * W + ((p & 1) ? W / 2 : 0);
        if (p == 0) wave_tile<P, PW, MODE_UP, true>(u, w, nx, g0, io, c, lane);
        else if (p == q) wave_tile<P, PW, MODE_DOWN, true>(u, w, nx, g0, io, c, lane);
        else wave_tile<P, PW, MODE_DIAMOND, true>(u, w, nx, g0, io, c, lane);
        __threadfence();
        __syncwarp();
        if (lane == 0) st_release_gpu(done + t, (unsigned)(p + 1));
    }
}

// Tile-flag kernel for insulated ends.  Even phases have ntiles tiles on [tW, (t+1)W), odd phases ntiles + 1 tiles on
// [jW - W/2, jW + W/2); odd tile j stitches even tiles j-1 and j (where they exist), even tile t stitches odd tiles t and t+1.
// doneE[t] / doneO[j] = 1 + the last phase of that parity the slot completed.  Items are numbered phase-major (an even
// phase and the odd phase after it form a group of 2 ntiles + 1 items), so the smallest id in flight never waits.
template <class P, int PW>
__global__ void __launch_bounds__(256) swept_chain_ins_kernel(typename P::real *u, typename P::real *w, int64_t nx, int ntiles, int q,
                                                               unsigned long long *counter, unsigned *doneE, unsigned *doneO, typename P::Consts c) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    T *io = reinterpret_cast<T *>(smem_raw) + (size_t)warp * P::NC * W;
    const unsigned long long group = 2ull * (unsigned long long)ntiles + 1ull;
    const unsigned long long total = (unsigned long long)(q + 1) * (unsigned long long)ntiles + (unsigned long long)((q + 1) / 2);
    for (;;) {
        unsigned long long id = 0;
        if (lane == 0) id = atomicAdd(counter, 1ull);
        id = __shfl_sync(0xffffffffu, id, 0);
        if (id >= total) break;
        const unsigned long long pair = id / group;
        const int rem = (int)(id - pair * group);
        const bool odd = rem >= ntiles;
        const int p = 2 * (int)pair + (odd ? 1 : 0), t = odd ? rem - ntiles : rem;
        if (p > 0) {
            bool dead = false;
            if (lane < 2) {
                const unsigned *flag = nullptr;
                if (odd) {
                    const int s = t - 1 + lane;                  // even tiles t-1 and t
                    if (s >= 0 && s < ntiles) flag = doneE + s;
                } else {
                    flag = doneO + t + lane;                     // odd tiles t and t+1
                }
                if (flag) {
                    unsigned ns = 20;
                    SpinWatch polls;
                    while (ld_acquire_gpu(flag) < (unsigned)p) {
                        __nanosleep(ns);
                        if (ns < 640) ns *= 2;
                        if (spin_gives_up(polls, abort_word_of(counter))) { dead = true; break; }
                    }
                }
            }
            __syncwarp();                                     // orders the other lanes' loads behind the polling lanes' acquire
            if (__any_sync(0xffffffffu, dead)) return;
        }
        const int64_t g0 = odd ? (int64_t)t * W - W / 2 : (int64_t)t * W;
        if (p == 0) wave_tile<P, PW, MODE_UP, true, true>(u, w, nx, g0, io, c, lane);
        else if (p == q) wave_tile<P, PW, MODE_DOWN, true, true>(u, w, nx, g0, io, c, lane);
        else wave_tile<P, PW, MODE_DIAMOND, true, true>(u, w, nx, g0, io, c, lane);
        __threadfence();
        __syncwarp();
        if (lane == 0) st_release_gpu((odd ? doneO : doneE) + t, (unsigned)(p + 1));
    }
}

// ---- host side, instantiated per problem in swept_wave_<problem>.cu -------------------------------------------
template <class P, int PW>
cudaError_t wave_launch_pw(int mode, void *u, void *w, int64_t nx, int64_t offset, const ConstBlock &cb, int wpb, size_t smem_floor,
                           int bc, cudaStream_t st) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int ntiles = (int)(nx / W) + ((bc && offset != 0) ? 1 : 0);
    if (wpb > 8) wpb = 8;
    if (wpb > ntiles) wpb = ntiles;
    const unsigned blocks = (unsigned)((ntiles + wpb - 1) / wpb);
    size_t smem = (size_t)wpb * P::NC * W * sizeof(T);
    if (smem < smem_floor) smem = smem_floor;
    if (bc) {
        if constexpr (P::INSULATED_OK) {
            if (mode == MODE_UP) swept_wave_kernel<P, PW, MODE_UP, true><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
            else if (mode == MODE_DIAMOND) swept_wave_kernel<P, PW, MODE_DIAMOND, true><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
            else swept_wave_kernel<P, PW, MODE_DOWN, true><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
            return cudaGetLastError();
        } else {
            return cudaErrorNotSupported;
        }
    }
    if (mode == MODE_UP) swept_wave_kernel<P, PW, MODE_UP><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    else if (mode == MODE_DIAMOND) swept_wave_kernel<P, PW, MODE_DIAMOND><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    else swept_wave_kernel<P, PW, MODE_DOWN><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    return cudaGetLastError();
}

// Chain launch: grid = min(warps needed, resident warps) / wpb blocks; `sync` = counter (8 bytes) + done[ntiles] (zeroed here);
// the handle's abort word sits SYNC_HEADER bytes before it (not zeroed here).
template <class P, int PW>
cudaError_t wave_chain_pw(void *u, void *w, int64_t nx, int64_t q, void *sync, const ConstBlock &cb, int wpb, size_t smem_floor, int sm_count,
                          int bc, cudaStream_t st) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int ntiles = (int)(nx / W);
    if (bc) {
        // insulated ends: sync = counter (8 bytes) + doneE[ntiles] + doneO[ntiles + 1]
        if constexpr (P::INSULATED_OK) {
            if (wpb > 8) wpb = 8;
            while (wpb > 1 && (int64_t)wpb * sm_count > ntiles) wpb >>= 1;
            size_t smem = (size_t)wpb * P::NC * W * sizeof(T);
            if (smem < smem_floor) smem = smem_floor;
            int per_sm = 0;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, swept_chain_ins_kernel<P, PW>, wpb * 32, smem);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) return cudaErrorLaunchOutOfResources;
            int64_t blocks = (ntiles + 1 + wpb - 1) / wpb;
            if (blocks > (int64_t)per_sm * sm_count) blocks = (int64_t)per_sm * sm_count;
            e = cudaMemsetAsync(sync, 0, 8 + sizeof(unsigned) * (size_t)(2 * ntiles + 1), st);
            if (e != cudaSuccess) return e;
            unsigned *doneE = (unsigned *)((char *)sync + 8);
            swept_chain_ins_kernel<P, PW><<<(unsigned)blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, ntiles, (int)q, (unsigned long long *)sync, doneE,
                                                                                    doneE + ntiles, c);
            return cudaGetLastError();
        } else {
            return cudaErrorNotSupported;
        }
    }
    if (wpb > chain_max_threads<P, PW>() / 32) wpb = chain_max_threads<P, PW>() / 32;
    while (wpb > 1 && (int64_t)wpb * sm_count > ntiles) wpb >>= 1;   // few tiles: spread the warps over the SMs
    size_t smem = (size_t)wpb * P::NC * W * sizeof(T);
    if (smem < smem_floor) smem = smem_floor;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, swept_chain_kernel<P, PW>, wpb * 32, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    int64_t blocks = (ntiles + wpb - 1) / wpb;
    if (blocks > (int64_t)per_sm * sm_count) blocks = (int64_t)per_sm * sm_count;
    e = cudaMemsetAsync(sync, 0, 8 + sizeof(unsigned) * (size_t)ntiles, st);
    if (e != cudaSuccess) return e;
    swept_chain_kernel<P, PW><<<(unsigned)blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, ntiles, (int)q, (unsigned long long *)sync,
                                                                          (unsigned *)((char *)sync + 8), c);
    return cudaGetLastError();
}

template <class P, int PW> cudaError_t wave_prepare_pw(int max_smem) {
    cudaError_t e = cudaFuncSetAttribute(swept_chain_kernel<P, PW>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_UP>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DIAMOND>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DOWN>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if constexpr (P::INSULATED_OK) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(swept_chain_ins_kernel<P, PW>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_UP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DIAMOND, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DOWN, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    }
    return e;
}

}  // namespace swept
