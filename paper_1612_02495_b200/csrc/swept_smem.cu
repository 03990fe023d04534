// swept_smem.cu -- the paper's swept kernels (SWEPT_KERNEL_SMEM): one thread block per tile ("node"), one
// thread per point, a two-row shared-memory matrix (row 0 = even tiers, row 1 = odd tiers,
// interior overwritten as it is used), a block barrier after every tier (Fig. 5).
//
//   MODE_UP       upTriangle, Fig. 5:  tiers 1..L-1 on [H t, W - H t)            (row A3)
//   MODE_DIAMOND  PAPER.md:86, 98, 114; Fig. 2b:        tiers 1..L on [c - H t, c + H t), then
//                                                        tiers L+1..2L-1 on [H(t-L), W - H(t-L))    (row A5)
//   MODE_DOWN     closing inverted triangle PAPER.md:98: tiers 1..L on [c - H t, c + H t)           (row A6)
//
// Edge exchange (row A4): the paper copies each tier's two edge values into global `left`/`right` arrays and
// swaps them on re-insertion (Fig. 2).  Even (odd) tier edges do not overlap, so
// row 0 over [0,W) and row 1 over [H, W-H) ARE the two edges; they are written back in place -- row 0 into the
// field u itself, row 1 into the workspace w -- and the next, half-a-tile shifted, kernel reads row 0 on [0,W)
// and row 1 on [-H, W+H).  No block writes what another block of the same launch reads.
#include "internal.h"
#include "stencils.cuh"

namespace swept {

template <class P, bool ODD>
__device__ __forceinline__ void smem_tier(typename P::real *s, int RS, int lo, int hi, const typename P::Consts &c) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC;
    // row r, field k, point x (valid for x in [-H, W+H)) lives at s[(r*NC + k)*RS + H + x]
    T *src = s + (ODD ? 0 : NC * RS) + H;
    T *dst = s + (ODD ? NC * RS : 0) + H;
    T *row0 = s + H;
    for (int x = lo + (int)threadIdx.x; x < hi; x += (int)blockDim.x) {
        T win[NC][2 * H + 1], b[NC], out[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) {
#pragma unroll
            for (int j = 0; j < 2 * H + 1; ++j) win[k][j] = src[k * RS + x + j - H];
            b[k] = (P::S == 2 && !ODD) ? row0[k * RS + x] : T(0);
        }
        P::template stage<ODD>(c, win, b, out);
#pragma unroll
        for (int k = 0; k < NC; ++k) dst[k * RS + x] = out[k];
    }
    __syncthreads();
}

template <class P, int MODE>
__global__ void __launch_bounds__(P::NC == 3 ? 512 : 1024) swept_smem_kernel(typename P::real *u, typename P::real *w, int64_t nx, int W,
                                                           int64_t offset, typename P::Consts c) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *s = reinterpret_cast<T *>(smem_raw);
    const int RS = W + 2 * H;
    const int64_t mask = nx - 1;
    const int64_t g0 = (int64_t)blockIdx.x * W + offset;
    const int tid = (int)threadIdx.x, nt = (int)blockDim.x;
    const int L = W / (2 * H), ctr = W / 2;

    for (int x = tid; x < W; x += nt)
#pragma unroll
        for (int k = 0; k < NC; ++k) s[k * RS + H + x] = u[(int64_t)k * nx + ((g0 + x) & mask)];
    if (MODE != MODE_UP) {
        for (int x = tid - H; x < W + H; x += nt)
#pragma unroll
            for (int k = 0; k < NC; ++k) s[(NC + k) * RS + H + x] = w[(int64_t)k * nx + ((g0 + x) & mask)];
    }
    __syncthreads();

    if (MODE != MODE_UP) {   // expanding part: inverted triangle between the two neighbouring triangles
        for (int t = 1; t <= L; ++t) {
            if (t & 1) smem_tier<P, true>(s, RS, ctr - H * t, ctr + H * t, c);
            else       smem_tier<P, false>(s, RS, ctr - H * t, ctr + H * t, c);
        }
    }
    if (MODE != MODE_DOWN) {  // shrinking part: upright triangle (L is even, so tier parity = t & 1 in both modes)
        for (int t = 1; t <= L - 1; ++t) {
            if (t & 1) smem_tier<P, true>(s, RS, H * t, W - H * t, c);
            else       smem_tier<P, false>(s, RS, H * t, W - H * t, c);
        }
    }

    for (int x = tid; x < W; x += nt)
#pragma unroll
        for (int k = 0; k < NC; ++k) u[(int64_t)k * nx + ((g0 + x) & mask)] = s[k * RS + H + x];
    if (MODE != MODE_DOWN) {
        for (int x = tid + H; x < W - H; x += nt)
#pragma unroll
            for (int k = 0; k < NC; ++k) w[(int64_t)k * nx + ((g0 + x) & mask)] = s[(NC + k) * RS + H + x];
    }
}

size_t swept_smem_bytes(int problem, int dtype, int W) {
    return (size_t)2 * (size_t)(W + 2 * radius_of(problem)) * (size_t)ncomp_of(problem) * elem_size(dtype);
}

template <class P> static cudaError_t prepare_smem(size_t max_bytes) {
    cudaError_t e;
    e = cudaFuncSetAttribute(swept_smem_kernel<P, MODE_UP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(swept_smem_kernel<P, MODE_DIAMOND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(swept_smem_kernel<P, MODE_DOWN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_bytes);
}

cudaError_t swept_smem_prepare(int problem, int dtype, size_t max_bytes) {
    cudaError_t e = cudaSuccess;
    SWEPT_DISPATCH(problem, dtype, P, e = prepare_smem<P>(max_bytes));
    return e;
}

template <class P>
static cudaError_t launch_smem(int mode, void *u, void *w, int64_t nx, int W, int64_t offset, const ConstBlock &cb,
                               size_t smem, cudaStream_t st) {
    using T = typename P::real;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const unsigned blocks = (unsigned)(nx / W);
    const int cap = P::NC == 3 ? 512 : 1024;   // Euler's flux arithmetic needs more than 64 registers per thread
    const int threads = W < cap ? (W < 32 ? 32 : W) : cap;
    if (mode == MODE_UP) swept_smem_kernel<P, MODE_UP><<<blocks, threads, smem, st>>>((T *)u, (T *)w, nx, W, offset, c);
    else if (mode == MODE_DIAMOND) swept_smem_kernel<P, MODE_DIAMOND><<<blocks, threads, smem, st>>>((T *)u, (T *)w, nx, W, offset, c);
    else swept_smem_kernel<P, MODE_DOWN><<<blocks, threads, smem, st>>>((T *)u, (T *)w, nx, W, offset, c);
    return cudaGetLastError();
}

cudaError_t launch_swept_smem(int problem, int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset,
                              const ConstBlock &cb, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    const size_t smem = swept_smem_bytes(problem, dtype, W);
    SWEPT_DISPATCH(problem, dtype, P, e = launch_smem<P>(mode, u, w, nx, W, offset, cb, smem, st));
    return e;
}

}  // namespace swept
