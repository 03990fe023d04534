// swept_ring.cuh -- SWEPT_OPT_CHAIN = 3 (default): the streaming band kernel (swept_band.cuh) with the edge exchange taken
// off the computing warps.
//
// swept_band_kernel keeps a band's columns in registers for the whole run and moves only the upper-right edge
// (Fig. 2b) through the staircase arrays R0 = d_u / R1 = workspace.  There the
// computing warp itself does the exchange every 32 iterations: acquire-load of the left band's counter, flush of its own
// output chunk, fence + release, fetch of its feed chunk -- four dependent L2 round trips (ncu, heat fp64, one warp per SM:
// 2 900 of the 12 400 cycles between two chunk boundaries; every warp also meets its left neighbour at every boundary, because a chunk
// is published exactly when the consumer asks for it).  On grids that give an SM only a few warps that is a quarter of
// the run time, and it is what makes narrow tiles (many warps, short dependent chains per iteration) lose.
//
// Here each block carries one extra COMMUNICATION WARP, and the exchange is split in three asynchronous parts:
//   flush    the computing warp stores the output chunk lane 31 has just finished (out ring in shared memory -> staircase arrays,
//            coalesced st.cg) at its chunk boundary and goes on; nothing waits for those stores;
//   release  the computing warp publishes its position K0 in shared memory (st.release.cta); the communication warp (lane w serves
//            computing warp w) acquires it and publishes the chunk to the right neighbour: st.release.gpu of prog[band].  The fence
//            of that release is cumulative over the two scopes, so it covers the computing warp's stores -- and it is the
//            communication warp, not a computing warp, that sits out its L2 round trip;
//   feed     the communication warp polls the left bands' counters (ld.acquire.gpu), stages every chunk that has been published up
//            to CAP - CH iterations ahead of its consumer into the consumer's feed ring with cp.async (LDGSTS, no register
//            staging), and publishes a counter in shared memory behind cp.async.wait_all.
// A computing warp touches global memory only with those fire-and-forget stores; at a boundary it reads one shared-memory
// counter.  The chunk (CH = 8 .. 32 iterations) no longer has to be the warp width, so a chunk is published up to 24 iterations
// before the neighbour needs it and neighbouring bands no longer run in lockstep.
//
// The remainder (nsteps mod (L/S), "results can only be read out every n-th timestep") runs INSIDE the same
// launch as a truncated cycle: with rt = S * (nsteps mod L/S) tiers left over, the last full phase q is not closed at tier L
// but runs on to tier L + rt, and one more phase q + 1 runs up to tier rt (swept_band_kernel's per-phase window (lo, hi] of
// tiers, nothing else).  In the characteristic coordinates column i of a band then ends at x = g0(q) + i - H rt: columns
// i < 2 H rt in phase q + 1, the others in phase q, so the flat field is stored with one shifted copy.  swept_run is ONE
// launch for any nsteps.
//
// Deadlock freedom: as swept_band_kernel (every wait is for an event of strictly smaller local time; all warps resident:
// cooperative launch), plus the communication warp, which never waits for anything but polls.  A chunk of outputs is complete
// when its warp has passed local time (chunk end + 31) and is published at the next boundary, so a tile must be at least
// CH * ceil((CH + 31) / CH) = 48 / 64 iterations long: NJI >= 64.  Every wait is bounded (spin_gives_up, swept_wave.cuh).
#pragma once
#include "swept_band.cuh"

namespace swept {

template <class P, int PW> struct RingGeom {
    using T = typename P::real;
    static constexpr int H = P::H, NC = P::NC, D = 2 * H;
    static constexpr int W = 32 * PW, NJ = W / D, NP = PW / D, L = W / D, CTR = W / 2;
    static constexpr int SR = band_sr<P, PW>();
    static constexpr int NJI = NJ / SR;                       // iterations per tile
    // Iterations per chunk and ring capacity.  Heat iterations are short (60..150 cycles for a warp alone on its scheduler), so the
    // rings must cover a few thousand cycles of exchange latency: chunks of 16 (32 for the long tiles), four (two) chunks of ring.
    // KS / Euler iterations cost hundreds to thousands of cycles and their rows are wide (D = 4, Euler 3 fields): chunks of 8 (16)
    // and two chunks of ring keep the rings at 1..3 KB per warp, which is what lets the parked bands of the largest grids fit.
    static constexpr int CH = H == 1 ? (NJI >= 128 ? 32 : 16) : (NJI >= 128 ? 16 : 8);
    static constexpr int NCH = NJI / CH;                      // chunks per tile
    static constexpr int CAP = (H == 1 && CH == 16 ? 4 : 2) * CH;   // feed ring capacity in iterations (prefetch depth CAP - CH)
    static constexpr int LAGC = (31 + CH) / CH;               // chunks between the end of a chunk and the boundary at which lane 31 is through it
    static constexpr int OCAP = 2 * CH;                       // out ring capacity in iterations: at a boundary K0 it holds the local times
                                                              // [K0 - CH (1 + LAGC), K0 - 31), CH (1 + LAGC) - 31 = 33 / 17 / 9 of them
    static constexpr int ITV = SR * D;                        // values per iteration and field
    static constexpr int RING = NC * CAP * ITV;               // values: feed ring
    static constexpr int ORING = NC * OCAP * ITV;             // values: out ring
    static constexpr int CS = 32 * (PW + 1);                  // one field of a parked band: lane stride PW + 1 (conflict-free)
    static constexpr int COL = NC * CS;                       // values: one parked band
    static constexpr int EDGE = 2 * NC * D;                   // values: hand-over of the incoming band's last D columns (two slots)
    static constexpr bool OK = NJI >= 64 && (NJI & (NJI - 1)) == 0;
    static __host__ __device__ size_t warp_values(int k) { return (size_t)RING + ORING + EDGE + (size_t)(k > 1 ? k - 1 : 0) * COL; }
};

// Computing warps per block an instantiation is compiled for.  The register file is per SM sub-partition (16384 registers, the
// warps of a block are dealt round-robin over the four), so a block of 4n warps -- 4n - 1 computing warps and the communication
// warp -- gets 16384 / (32 n) registers per thread: NWMAX = 4n - 1.  The column state is NC (D + PW) values per lane plus what
// the stencil needs.  ROOMY: a second build for 3 computing warps (up to 255 registers, no spills) where the wide build is
// register-starved; used when the grid has no more bands than 3 warps per SM can own -- small and mid-size grids, where every
// warp must be as fast as it can.
constexpr int RING_ROOMY = 3;
template <class P, int PW> constexpr int ring_nwmax() {
    const int est = P::NC * (2 * P::H + PW) * (int)(sizeof(typename P::real) / 4) + (P::GROUPED ? 110 : 56 + 16 * (P::H - 1));
    int warps = 65536 / (32 * est);
    if (P::H == 2 && !P::GROUPED && sizeof(typename P::real) == 8 && PW == 32) warps = 8;   // KS fp64, 32 points per lane: spills below ~200 registers
    warps = warps >= 4 ? (warps & ~3) : 4;
    return (warps > 28 ? 28 : warps) - 1;
}
// heat: up to 7 computing warps per SM (8 warps x 255 registers is still the whole register file) -- measured, W = 512: nx = 2^18 2849 -> 2993,
// 2^19 3819 -> 4068 GPts*steps/s; KS W = 256 loses with 7 (2^17 210 -> 179) and keeps 3
template <class P> constexpr int ring_roomy() { return P::H == 1 ? 7 : RING_ROOMY; }
template <class P, int PW> constexpr bool ring_has_roomy() { return ring_nwmax<P, PW>() > ring_roomy<P>() && 65536 / (32 * (ring_nwmax<P, PW>() + 1)) < (P::GROUPED ? 255 : 128); }

// Bands are dealt over the computing warps of the grid: band n -> warp (n mod (blocks x wpb)) / blocks of block n mod blocks, so
// that neighbouring bands sit on different SMs and every warp owns floor or ceil(ntiles / (blocks x wpb)) of them (the BandGrid
// helpers of internal.h with one slot per block).
__host__ __device__ inline BandGrid ring_layout(int ntiles, int sm_count, int wpb) {
    BandGrid g;
    g.wpb = wpb;
    g.SL = 1;
    g.wps = wpb;
    const int nb = (ntiles + wpb - 1) / wpb;
    g.nblocks = nb < sm_count ? nb : sm_count;
    g.G = g.nblocks;
    const int stride = g.G * g.wps;
    g.kmax = (ntiles + stride - 1) / stride;
    return g;
}

struct RingCtl { unsigned k0, feed, pad0, pad1; };
constexpr unsigned RING_END = 0x7fffffffu;
constexpr int RING_CTL_BYTES = 32 * (int)sizeof(RingCtl);

__device__ __forceinline__ unsigned ld_acquire_cta_shared(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"((unsigned)__cvta_generic_to_shared(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_cta_shared(unsigned *p, unsigned v) {
    asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_relaxed_gpu(const unsigned *p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// one element global -> shared, asynchronously (LDGSTS); completion: cp_async_wait_all
template <class T> __device__ __forceinline__ void cp_async_elem(T *smem_dst, const T *gsrc) {
    static_assert(sizeof(T) == 4 || sizeof(T) == 8, "element size");
    if (sizeof(T) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Shared-memory offset (in values) of computing warp `warp`'s area: the areas are packed by each warp's own band count.
template <class Gm> __device__ __forceinline__ size_t ring_warp_offset(const BandGrid &grid, int block, int warp, int ntiles) {
    size_t off = 0;
    for (int w = 0; w < warp; ++w) off += Gm::warp_values(band_count(grid, block, w, ntiles));
    return off;
}

// Vector of 16 bytes of T
template <class T> struct vec16;
template <> struct vec16<double> { using type = double2; static constexpr int N = 2; };
template <> struct vec16<float> { using type = float4; static constexpr int N = 4; };

// ---- the communication warp ---------------------------------------------------------------------------------------
template <class P, int PW>
__device__ __forceinline__ void ring_comm_warp(typename P::real *u, typename P::real *w, const int64_t nx, const int ntiles, const int nph, const BandGrid &grid,
                                               unsigned *prog, unsigned char *smem_raw, const int lane) {
    using T = typename P::real;
    using Gm = RingGeom<P, PW>;
    constexpr int H = Gm::H, NC = Gm::NC, D = Gm::D, W = Gm::W, NJI = Gm::NJI, CTR = Gm::CTR, NCH = Gm::NCH, SR = Gm::SR, CH = Gm::CH, CAP = Gm::CAP, ITV = Gm::ITV;
    constexpr int NEL = NC * CH * ITV;                     // values of one chunk
    const int64_t mask = nx - 1;
    const int NW = grid.wpb;
    RingCtl *ctl = reinterpret_cast<RingCtl *>(smem_raw);
    T *areas = reinterpret_cast<T *>(smem_raw + RING_CTL_BYTES);
    const int stride = band_stride(grid);

    // lane w serves computing warp w
    const bool mine = lane < NW;
    const int first = mine ? band_first(grid, (int)blockIdx.x, lane) : 0;
    const int k = mine ? band_count(grid, (int)blockIdx.x, lane, ntiles) : 0;
    const int lt_end = k * nph * NJI;
    const DivK divk(k > 0 ? k : 1);
    T *area = areas + (mine ? ring_warp_offset<Gm>(grid, (int)blockIdx.x, lane, ntiles) : 0);
    int fnext = 0, snext = 0;                             // next feed chunk to stage / next output chunk to publish (local time of its first iteration)
    unsigned seen = 0;                                    // last value read from the left band's counter
    int seen_band = -1;
    SpinWatch idle;

    for (;;) {
        bool f_ready = false, f_data = false;
        int f_band = 0, f_p = 0, n_pub = 0;
        if (k > 0 && (fnext < lt_end || snext < lt_end)) {
            const unsigned k0u = ld_acquire_cta_shared(&ctl[lane].k0);
            const int k0 = k0u == RING_END ? lt_end + 64 + CH : (int)k0u;
            // the warp flushes chunk [c, c + CH) at the boundary K0 = c + CH (1 + LAGC), before it publishes K0
            n_pub = snext < lt_end ? (k0 - CH * Gm::LAGC - snext) / CH : 0;
            if (n_pub < 0) n_pub = 0;
            if (snext + n_pub * CH > lt_end) n_pub = (lt_end - snext) / CH;
            if (fnext < lt_end && fnext + CH - CAP <= k0) {             // the ring slots of the chunk are consumed
                const int s = fnext / NJI;
                f_p = divk(s);
                f_band = first + (s - f_p * k) * stride;
                if (f_p == 0) f_ready = true;                           // the upright triangle takes no row inputs
                else {
                    const int left = f_band == 0 ? ntiles - 1 : f_band - 1;
                    const unsigned need = (unsigned)((f_p - 1) * NCH + (fnext & (NJI - 1)) / CH + 1);
                    if (seen_band != left || seen < need) { seen = ld_acquire_gpu(prog + left); seen_band = left; }
                    if (seen >= need) f_ready = f_data = true;
                }
            }
        }
        const unsigned mf = __ballot_sync(0xffffffffu, f_data);
        const unsigned any = __ballot_sync(0xffffffffu, f_ready || n_pub > 0);
        const unsigned busy = __ballot_sync(0xffffffffu, k > 0 && (fnext < lt_end || snext < lt_end));
        if (!busy) break;
        if (!any) {
            __nanosleep(32);
            if (spin_gives_up(idle, abort_word_of(prog))) return;
            continue;
        }
        idle = SpinWatch();
        // ---- publish: the computing warp stored its chunk(s) before it released K0 and this lane acquired K0, so the release below
        // orders those stores before the counter for every observer (causality is cumulative across the two scopes)
        for (; n_pub > 0; --n_pub, snext += CH) {
            const int s = snext / NJI, p = divk(s);
            if (p < nph - 1) st_release_gpu(prog + first + (s - p * k) * stride, (unsigned)(p * NCH + (snext & (NJI - 1)) / CH + 1));
        }
        // ---- stage the feeds whose chunk the left band has published (the acquire loads above order the copies behind it for the
        // lane that polled; the warp barrier extends that to the lanes that copy)
        if (mf) {
            __syncwarp();
            for (unsigned m = mf; m; m &= m - 1) {
                const int src = __ffs(m) - 1;
                const int band = __shfl_sync(0xffffffffu, f_band, src), p = __shfl_sync(0xffffffffu, f_p, src), lt0 = __shfl_sync(0xffffffffu, fnext, src);
                T *ring = areas + __shfl_sync(0xffffffffu, (unsigned long long)(area - areas), src);       // that warp's feed ring
                const int64_t g0 = ((int64_t)band * W - (int64_t)p * (W / 2)) & mask;
                const int it0 = lt0 & (NJI - 1);
                for (int e = lane; e < NEL; e += 32) {
                    const int rho = e % D, sr = (e / D) % SR, it = (e / ITV) % CH, kk = e / (ITV * CH);
                    const int J = SR * (it0 + it) + sr;                 // row j = J D + rho is fed from tier J of the left tile's right edge
                    const T *from = ((J & 1) ? w : u) + (int64_t)kk * nx + ((g0 + CTR - H * J - rho - 1) & mask);
                    cp_async_elem(ring + ((kk * CAP + ((lt0 + it) & (CAP - 1))) * SR + sr) * D + rho, from);
                }
            }
            cp_async_wait_all();
        }
        __syncwarp();
        if (f_ready) { fnext += CH; st_release_cta_shared(&ctl[lane].feed, (unsigned)fnext); }
    }
}

// ---- the kernel ---------------------------------------------------------------------------------------------------------
// grid.wpb = computing warps per block; the block has one more warp (the last), the communication warp.
// nph = number of phases = q + 1 (+ 1 if rt > 0); phase p updates the tiers (lo, hi]: lo = L for p = 0 (the upright triangle starts
// from the flat field), hi = L + rt for p = q, rt for p = q + 1 (the truncated closing cycle).
template <class P, int PW, int NWMAX>
__global__ void __launch_bounds__(32 * (NWMAX + 1)) swept_ring_kernel(typename P::real *u, typename P::real *w, int64_t nx, int ntiles, int q, int rt,
                                                                       BandGrid grid, unsigned *prog, typename P::Consts c) {
    using T = typename P::real;
    using Gm = RingGeom<P, PW>;
    using V = typename vec16<T>::type;
    constexpr int VN = vec16<T>::N;
    constexpr int H = Gm::H, NC = Gm::NC, D = Gm::D, W = Gm::W, NJI = Gm::NJI, NP = Gm::NP, L = Gm::L, CS = Gm::CS, SR = Gm::SR, CH = Gm::CH, CAP = Gm::CAP, OCAP = Gm::OCAP, ITV = Gm::ITV, CTR = Gm::CTR;
    static_assert(CH * (1 + Gm::LAGC) - 31 <= OCAP, "the chunk being flushed must still be in the out ring");
    static_assert(Gm::OK, "a tile must be at least 64 iterations long");
    static_assert(PW % D == 0 && PW % VN == 0, "points per lane: a multiple of 2H and of a 16-byte vector");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    const int64_t mask = nx - 1;
    const int nph = q + 1 + (rt > 0 ? 1 : 0);
    RingCtl *ctl = reinterpret_cast<RingCtl *>(smem_raw);
    if (threadIdx.x < 32) { ctl[threadIdx.x].k0 = 0; ctl[threadIdx.x].feed = 0; }
    __syncthreads();
    if (warp == grid.wpb) {
        ring_comm_warp<P, PW>(u, w, nx, ntiles, nph, grid, prog, smem_raw, lane);
        return;
    }

    const int first = band_first(grid, (int)blockIdx.x, warp), stride = band_stride(grid);   // bands first, first + stride, ...
    const int k = band_count(grid, (int)blockIdx.x, warp, ntiles);
    if (k == 0) return;
    const int n_items = k * nph;
    const int lt_end = n_items * NJI;                     // < 2^31: the host refuses longer runs
    RingCtl *my = ctl + warp;

    T *base = reinterpret_cast<T *>(smem_raw + RING_CTL_BYTES) + ring_warp_offset<Gm>(grid, (int)blockIdx.x, warp, ntiles);
    T *feed = base, *outr = feed + Gm::RING, *edge = outr + Gm::ORING, *col = edge + Gm::EDGE;

    auto g0_of = [&](int band, int p) -> int64_t { return ((int64_t)band * W - (int64_t)p * (W / 2)) & mask; };

    // ---- column state.  X[k][0..D) = copy of lane l-1's last D columns, X[k][D + i] = own column i (16-byte loads)
    T X[NC][D + PW];
    {
        const int64_t g0 = g0_of(first, 0);
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int i = 0; i < PW; i += VN) {
                const V v = __ldcg(reinterpret_cast<const V *>(u + (int64_t)kk * nx + ((g0 + lane * PW + i) & mask)));
                const T *pv = reinterpret_cast<const T *>(&v);
#pragma unroll
                for (int e = 0; e < VN; ++e) X[kk][D + i + e] = pv[e];
            }
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
                for (int kk = 0; kk < NC; ++kk) buf[kk * CS + i + i / PW] = __ldcg(u + (int64_t)kk * nx + ((gm + i) & mask));
        }
        __syncwarp();
    }

    const DivK divk(k);
    int p_cur = 0, lo = L, hi = 0x3fffffff;               // this lane's tile: phase, and the tiers (lo, hi] it updates
    bool interior = false;                               // p_cur is a diamond phase: every point of the tile is updated
    auto set_phase = [&](int s) {
        p_cur = divk(s);
        lo = p_cur == 0 ? L : 0;
        hi = p_cur < q ? 0x3fffffff : (p_cur == q ? L + rt : rt);
        interior = p_cur > 0 && p_cur < q;
    };
    // This lane enters tile s >= 1 of a warp that owns k > 1 bands: swap its PW columns with the parked copy of the incoming
    // band (transition s-1 uses buffer (s-1) mod (k-1)), and hand the incoming band's last D columns -- before this lane's
    // first super-row changes them -- to lane l+1, which swaps one iteration later (slot = parity of the lane).
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
                edge[((lane & 1) * NC + kk) * D + d] = X[kk][PW + d];
                if (lane > 0) X[kk][d] = edge[(((lane - 1) & 1) * NC + kk) * D + d];
            }
    };
    T keep[SR][NC][D];                                   // this lane's row values after each super-row of its last iteration
#pragma unroll
    for (int sr = 0; sr < SR; ++sr)
#pragma unroll
        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
            for (int rho = 0; rho < D; ++rho) keep[sr][kk][rho] = X[kk][PW + (D - 1 - rho)];

    for (int K0 = 0; K0 < lt_end + 31; K0 += CH) {
        // ---- chunk boundary.  (1) Flush the output chunk lane 31 has just got through, local times [K0 - CH (1 + LAGC), + CH): plain
        // coalesced stores, nothing waits for them.  (2) Publish K0 (release at CTA scope: the communication warp then releases the
        // chunk to the right neighbour at GPU scope).  (3) Wait for the feed of [K0, K0 + CH) -- staged chunks ahead, so normally
        // there already.  EVERY lane polls the counter (one address: a broadcast read; each lane's own acquire orders its ring
        // reads): the boundary has no lane-dependent branch, so the warp stays converged for the shuffles of the loop (a
        // lane-0-only spin left the warp split in two for whole chunks: ncu showed 40 % of the iterations issued twice, through
        // the divergent-shuffle path).
        __syncwarp();
        {
            const int lt0 = K0 - CH * (1 + Gm::LAGC);
            if (lt0 >= 0 && lt0 < lt_end) {
                const int s = lt0 / NJI, p = divk(s);
                if (p < nph - 1) {
                    const int64_t g0 = g0_of(first + (s - p * k) * stride, p);
                    const int it0 = lt0 & (NJI - 1);
                    constexpr int NEL = NC * CH * ITV;
#pragma unroll
                    for (int e0 = 0; e0 < NEL; e0 += 32) {
                        const int e = e0 + lane;
                        if (NEL % 32 == 0 || e < NEL) {
                            const int rho = e % D, sr = (e / D) % SR, it = (e / ITV) % CH, kk = e / (ITV * CH);
                            const int J = SR * (it0 + it) + sr;         // rows j = J D + rho hold tier L + J
                            T *to = ((J & 1) ? w : u) + (int64_t)kk * nx + ((g0 + W - 1 - H * J - rho) & mask);
                            __stcg(to, outr[((kk * OCAP + ((lt0 + it) & (OCAP - 1))) * SR + sr) * D + rho]);
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) st_release_cta_shared(&my->k0, (unsigned)K0);
        {
            const int need_feed = K0 < lt_end ? (K0 + CH < lt_end ? K0 + CH : lt_end) : 0;
            SpinWatch polls;
            bool dead = false;
            while ((int)ld_acquire_cta_shared(&my->feed) < need_feed) {
                if (spin_gives_up(polls, abort_word_of(prog))) { dead = true; break; }
            }
            if (__any_sync(0xffffffffu, dead)) return;
        }

        // ---- the chunk's CH iterations.  Steady chunk: every lane is, for the whole chunk, inside diamond tiles -- nothing depends on
        // the phase; in the first 32 iterations of a tile the lanes of a warp with k > 1 bands swap columns, each at its own iteration.
        bool steady = K0 >= 31 && K0 + CH - 1 < lt_end;
        const bool swapchunk = k > 1 && (K0 & (NJI - 1)) < 32;
        if (steady) {
            const int pa = divk((K0 - 31) / NJI), pb = divk((K0 + CH - 1) / NJI);
            steady = pa > 0 && pb < q;
        }
        if (steady) {
            constexpr bool ONE_LOOP = P::GROUPED;
            auto steady_chunk = [&](auto swap_tag) {
                constexpr bool SWAP = decltype(swap_tag)::value;
                int J = (K0 - lane) & (NJI - 1);
                int fs = K0 & (CAP - 1), os = (K0 - 31) & (OCAP - 1);     // ring slots: lane 0's local time K0, lane 31's K0 - 31
#pragma unroll 1
                for (int it = 0; it < CH; ++it) {
                    const T *fp = feed + fs * SR * D;
                    T recv[SR][NC][D];
#pragma unroll
                    for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                        for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                            for (int rho = 0; rho < D; ++rho) {
                                const T f = fp[(kk * CAP * SR + sr) * D + rho];
                                const T r = shfl_up1(keep[sr][kk][rho]);
                                recv[sr][kk][rho] = lane == 0 ? f : r;
                            }
                    if (SWAP && (!ONE_LOOP || swapchunk) && J == 0) swap_bands((K0 + it - lane) / NJI);
                    band_super_rows<P, PW, SR, true>(X, recv, keep, c, lane * NP + SR * J + 1, 0, 0);
                    if (lane == 31) {
                        T *op = outr + os * SR * D;
#pragma unroll
                        for (int sr = 0; sr < SR; ++sr)
#pragma unroll
                            for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                                for (int rho = 0; rho < D; ++rho) op[(kk * OCAP * SR + sr) * D + rho] = keep[sr][kk][rho];
                    }
                    J = (J + 1) & (NJI - 1);
                    fs = (fs + 1) & (CAP - 1);
                    os = (os + 1) & (OCAP - 1);
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
        for (int K = K0; K < K0 + CH && K < lt_end + 31; ++K) {
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
                    for (int rho = 0; rho < D; ++rho) fd[sr][kk][rho] = feed[((kk * CAP + (K & (CAP - 1))) * SR + sr) * D + rho];
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
                        for (int rho = 0; rho < D; ++rho) outr[((kk * OCAP + (lt & (OCAP - 1))) * SR + sr) * D + rho] = keep[sr][kk][rho];
            }
            __syncwarp();
        }
    }
    // ---- tail: the chunks lane 31 finished during the last boundaries' worth of iterations (the loop above flushes chunk c at the
    // boundary c + CH (1 + LAGC), and ends at lt_end + 31)
    __syncwarp();
    for (int lt0 = ((lt_end + 31 + CH - 1) / CH) * CH - CH * (1 + Gm::LAGC); lt0 < lt_end; lt0 += CH) {
        if (lt0 < 0) continue;
        const int s = lt0 / NJI, p = divk(s);
        if (p >= nph - 1) continue;
        const int64_t g0 = g0_of(first + (s - p * k) * stride, p);
        const int it0 = lt0 & (NJI - 1);
        constexpr int NEL = NC * CH * ITV;
        for (int e = lane; e < NEL; e += 32) {
            const int rho = e % D, sr = (e / D) % SR, it = (e / ITV) % CH, kk = e / (ITV * CH);
            const int J = SR * (it0 + it) + sr;
            T *to = ((J & 1) ? w : u) + (int64_t)kk * nx + ((g0 + W - 1 - H * J - rho) & mask);
            __stcg(to, outr[((kk * OCAP + ((lt0 + it) & (OCAP - 1))) * SR + sr) * D + rho]);
        }
    }
    __syncwarp();
    if (lane == 0) st_release_cta_shared(&my->k0, RING_END);

    // ---- With a truncated closing cycle (rt > 0) phase q has a consumer, so its row outputs sit in the right half of this band's
    // phase-q span -- the span the flat field is about to be stored over -- until the right neighbour has fetched them for its
    // phase q + 1.  (Without it, phase q has no outputs and every band overwrites only what it consumed itself.)  All bands finish
    // within a few iterations of one another: wait until every computing warp of the grid is through its last tile.
    if (rt > 0) {
        bool dead = false;
        if (lane == 0) {
            const unsigned total = (unsigned)(ntiles < grid.G * grid.wps ? ntiles : grid.G * grid.wps);
            __threadfence();
            atomicAdd(prog + ntiles, 1u);
            unsigned ns = 100;
            SpinWatch polls;
            while (ld_acquire_gpu(prog + ntiles) < total) {
                __nanosleep(ns);
                if (ns < 6400) ns *= 2;
                if (spin_gives_up(polls, abort_word_of(prog))) { dead = true; break; }
            }
        }
        if (__any_sync(0xffffffffu, dead)) return;
    }

    // ---- all phases done.  Column i of a band ended at x = g0(band, q) + i - H rt (in phase q + 1 if i < 2 H rt, else in phase q):
    // registers hold band k-1's values, the parked copies the other bands'
    {
        const int64_t sh = (rt > 0 ? W / 2 : 0) - H * rt + nx;   // g0(q) = g0(last phase) + W/2 when the extra phase ran
        const int64_t g0 = g0_of(first + (k - 1) * stride, nph - 1) + sh;
        if ((H * rt) % VN == 0) {
#pragma unroll
            for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                for (int i = 0; i < PW; i += VN) {
                    V v;
                    T *pv = reinterpret_cast<T *>(&v);
#pragma unroll
                    for (int e = 0; e < VN; ++e) pv[e] = X[kk][D + i + e];
                    __stcg(reinterpret_cast<V *>(u + (int64_t)kk * nx + ((g0 + lane * PW + i) & mask)), v);
                }
        } else {
#pragma unroll
            for (int kk = 0; kk < NC; ++kk)
#pragma unroll
                for (int i = 0; i < PW; ++i) __stcg(u + (int64_t)kk * nx + ((g0 + lane * PW + i) & mask), X[kk][D + i]);
        }
        for (int m = 0; m + 1 < k; ++m) {
            const int64_t gm = g0_of(first + m * stride, nph - 1) + sh;
            const T *buf = col + (size_t)(((nph - 1) * k + m) % (k - 1)) * Gm::COL;   // band m's last tile was swapped out at transition (nph-1) k + m
            for (int i = lane; i < W; i += 32)
#pragma unroll
                for (int kk = 0; kk < NC; ++kk) __stcg(u + (int64_t)kk * nx + ((gm + i) & mask), buf[kk * CS + i + i / PW]);
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------
// Size the grid: one block per SM, computing warps as the launch bound (registers) and shared memory allow, all resident.
template <class P, int PW, int NWMAX>
bool ring_grid(int64_t nx, int sm_count, int max_smem, int max_warps, BandGrid *out, size_t *smem_bytes) {
    using Gm = RingGeom<P, PW>;
    using T = typename P::real;
    const int64_t ntiles64 = nx / Gm::W;
    if (ntiles64 < 2 || ntiles64 > (1 << 24)) return false;
    const int ntiles = (int)ntiles64;
    int wmax = NWMAX;
    if (max_warps > 0 && wmax > max_warps) wmax = max_warps;    // SWEPT_OPT_BLOCKS_PER_SM x 4 warps: fewer resident warps on request
    // computing warps per block: the fewest that give every band its own warp on sm_count SMs (the bands then spread over all SMs);
    // with more bands than warps, the most the build allows, less in steps of 4 while the parked bands do not fit shared memory
    int wneed = (int)((ntiles64 + sm_count - 1) / sm_count);
    if (wneed < 1) wneed = 1;
    for (int wpb = wneed < wmax ? wneed : wmax; wpb >= 1; wpb -= (wpb > 4 ? 4 : 1)) {
        const BandGrid g = ring_layout(ntiles, sm_count, wpb);
        size_t worst = 0;                                         // the areas are packed per warp's own band count: size the fullest block
        for (int b = 0; b < g.nblocks; ++b) {
            size_t v = 0;
            for (int wv = 0; wv < wpb; ++wv) v += Gm::warp_values(band_count(g, b, wv, ntiles));
            if (v > worst) worst = v;
        }
        const size_t smem = RING_CTL_BYTES + worst * sizeof(T);
        if (smem > (size_t)max_smem) continue;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, swept_ring_kernel<P, PW, NWMAX>, (wpb + 1) * 32, smem) != cudaSuccess) { cudaGetLastError(); continue; }
        if (per_sm < 1) continue;
        *out = g;
        *smem_bytes = smem;
        return true;
    }
    return false;
}

// `sync` = prog[ntiles] (zeroed here).  q half-cycles + rt remainder tiers in ONE launch.  cudaErrorNotSupported when the
// schedule does not fit (the caller falls back to swept_band_kernel / swept_chain_kernel).
template <class P, int PW, int NWMAX>
cudaError_t wave_ring_pw(void *u, void *w, int64_t nx, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps,
                         cudaStream_t st) {
    using T = typename P::real;
    using Gm = RingGeom<P, PW>;
    BandGrid g;
    size_t smem = 0;
    if (q < 0 || (q == 0 && rt == 0) || q > (1 << 24) / Gm::NCH || rt < 0 || rt >= Gm::L) return cudaErrorNotSupported;
    if (!ring_grid<P, PW, NWMAX>(nx, sm_count, max_smem, max_warps, &g, &smem)) return cudaErrorNotSupported;
    if ((int64_t)(q + 2) * g.kmax * Gm::NJI >= ((int64_t)1 << 30)) return cudaErrorNotSupported;   // the kernel's local time is an int
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int ntiles = (int)(nx / Gm::W);
    cudaError_t e = cudaMemsetAsync(sync, 0, sizeof(unsigned) * (size_t)(ntiles + 1), st);   // prog[ntiles] + the end-of-run arrival count
    if (e != cudaSuccess) return e;
    T *up = (T *)u, *wp = (T *)w;
    int qi = (int)q, nt = ntiles, rti = rt;
    unsigned *pr = (unsigned *)sync;
    typename P::Consts cc = c;
    void *args[] = {&up, &wp, &nx, &nt, &qi, &rti, &g, &pr, &cc};
    return cudaLaunchCooperativeKernel((const void *)swept_ring_kernel<P, PW, NWMAX>, dim3((unsigned)g.nblocks), dim3((unsigned)((g.wpb + 1) * 32)), args, smem, st);
}

template <class P, int PW, int NWMAX> cudaError_t ring_prepare_pw(int max_smem) {
    return cudaFuncSetAttribute(swept_ring_kernel<P, PW, NWMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}

// One (problem, points per lane): the wide build, or the roomy one when the grid is small enough for it.
template <class P, int PW>
cudaError_t wave_ring(void *u, void *w, int64_t nx, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    if constexpr (!RingGeom<P, PW>::OK) return cudaErrorNotSupported;
    else {
        if constexpr (ring_has_roomy<P, PW>()) {
            if (nx / RingGeom<P, PW>::W <= (int64_t)ring_roomy<P>() * sm_count) return wave_ring_pw<P, PW, ring_roomy<P>()>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        }
        return wave_ring_pw<P, PW, ring_nwmax<P, PW>()>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
    }
}
template <class P, int PW> cudaError_t ring_prepare(int max_smem) {
    if constexpr (!RingGeom<P, PW>::OK) return cudaSuccess;
    else {
        if constexpr (ring_has_roomy<P, PW>()) {
            cudaError_t e = ring_prepare_pw<P, PW, ring_roomy<P>()>(max_smem);
            if (e != cudaSuccess) return e;
        }
        return ring_prepare_pw<P, PW, ring_nwmax<P, PW>()>(max_smem);
    }
}
template <class P, int PW> constexpr bool ring_supports() { return RingGeom<P, PW>::OK; }

}  // namespace swept
