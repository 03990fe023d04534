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

template <class T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

template <class P, int PW, int MODE>
__global__ void __launch_bounds__(256) swept_wave_kernel(typename P::real *u, typename P::real *w, int64_t nx, int64_t offset,
                                                          int ntiles, typename P::Consts c) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC, D = 2 * H;
    constexpr int W = 32 * PW, NJ = W / D, NP = PW / D, L = W / D, CTR = W / 2;
    static_assert(PW % D == 0, "points per lane must be a multiple of 2H");
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int lane = (int)(threadIdx.x & 31), warp = (int)(threadIdx.x >> 5);
    const int tile = (int)blockIdx.x * (int)(blockDim.x >> 5) + warp;
    if (tile >= ntiles) return;                      // whole warps only
    T *io = reinterpret_cast<T *>(smem_raw) + (size_t)warp * NC * W;   // io[k*W + j]: row feed in, right edge out
    const int64_t mask = nx - 1;
    const int64_t g0 = (int64_t)tile * W + offset;

    // X[k][0..D) = copy of lane l-1's last D columns, X[k][D + q] = own column q
    T X[NC][D + PW];

    if (MODE == MODE_UP) {
#pragma unroll
        for (int k = 0; k < NC; ++k)
#pragma unroll
            for (int q = 0; q < PW; ++q) X[k][D + q] = u[(int64_t)k * nx + ((g0 + lane * PW + q) & mask)];
    } else {
        // column i = 2H m + r starts from tier m of the right neighbour triangle's left edge: R_{m&1}[c + H m + r]
#pragma unroll
        for (int q = 0; q < PW; ++q) {
            const int m = lane * NP + q / D, r = q % D;
            const T *src = (m & 1) ? w : u;
            const int64_t g = (g0 + CTR + H * m + r) & mask;
#pragma unroll
            for (int k = 0; k < NC; ++k) X[k][D + q] = src[(int64_t)k * nx + g];
        }
        // row j = 2H m + rho is fed from tier m of the left neighbour triangle's right edge: R_{m&1}[c - H m - rho - 1]
        for (int j = lane; j < W; j += 32) {
            const int m = j / D, rho = j % D;
            const T *src = (m & 1) ? w : u;
            const int64_t g = (g0 + CTR - H * m - rho - 1) & mask;
#pragma unroll
            for (int k = 0; k < NC; ++k) io[k * W + j] = src[(int64_t)k * nx + g];
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
            for (int q = 0; q < PW; ++q) u[(int64_t)k * nx + ((g0 + lane * PW + q) & mask)] = X[k][D + q];
    } else {
        // final column state: column i = 2H m + r holds tier L+m at x = H m + r  -> R_{m&1}[H m + r]
#pragma unroll
        for (int q = 0; q < PW; ++q) {
            const int m = lane * NP + q / D, r = q % D;
            T *dst = (m & 1) ? w : u;
            const int64_t g = (g0 + H * m + r) & mask;
#pragma unroll
            for (int k = 0; k < NC; ++k) dst[(int64_t)k * nx + g] = X[k][D + q];
        }
        __syncwarp();
        // lane 31's row outputs: row j = 2H m + rho holds tier L+m at x = W-1-H m-rho -> R_{m&1}[W - 1 - H m - rho]
        for (int j = lane; j < W; j += 32) {
            const int m = j / D, rho = j % D;
            T *dst = (m & 1) ? w : u;
            const int64_t g = (g0 + W - 1 - H * m - rho) & mask;
#pragma unroll
            for (int k = 0; k < NC; ++k) dst[(int64_t)k * nx + g] = io[k * W + j];
        }
    }
}

// ---- host side, instantiated per problem in swept_wave_<problem>.cu -------------------------------------------
template <class P, int PW>
cudaError_t wave_launch_pw(int mode, void *u, void *w, int64_t nx, int64_t offset, const ConstBlock &cb, int wpb, size_t smem_floor,
                           cudaStream_t st) {
    using T = typename P::real;
    constexpr int W = 32 * PW;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int ntiles = (int)(nx / W);
    if (wpb > 8) wpb = 8;
    if (wpb > ntiles) wpb = ntiles;
    const unsigned blocks = (unsigned)((ntiles + wpb - 1) / wpb);
    size_t smem = (size_t)wpb * P::NC * W * sizeof(T);
    if (smem < smem_floor) smem = smem_floor;
    if (mode == MODE_UP) swept_wave_kernel<P, PW, MODE_UP><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    else if (mode == MODE_DIAMOND) swept_wave_kernel<P, PW, MODE_DIAMOND><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    else swept_wave_kernel<P, PW, MODE_DOWN><<<blocks, wpb * 32, smem, st>>>((T *)u, (T *)w, nx, offset, ntiles, c);
    return cudaGetLastError();
}

template <class P, int PW> cudaError_t wave_prepare_pw(int max_smem) {
    cudaError_t e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_UP>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DIAMOND>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(swept_wave_kernel<P, PW, MODE_DOWN>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
}

}  // namespace swept
