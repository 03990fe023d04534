// naive.cu -- the classic decomposition (section IV.D; Fig. 6): one kernel per
// sub-timestep, one thread per grid point, neighbours through the periodic index `& (nx-1)`
// (PAPER.md:171), global memory in and out.  SURVEY.md section 8(a) row A2.
#include "internal.h"
#include "stencils.cuh"

namespace swept {

// INS: insulated ends (Eq. 9): a neighbour index outside the rod is mirrored back, -1 -> 0 and
// nx -> nx-1 (the ghost value is the adjacent interior value).
template <class P, bool ODD, bool INS = false>
__global__ void __launch_bounds__(256) classic_kernel(const typename P::real *__restrict__ src, const typename P::real *base,
                                                       typename P::real *dst, int64_t nx, typename P::Consts c) {
    using T = typename P::real;
    constexpr int H = P::H, NC = P::NC;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nx) return;
    T win[NC][2 * H + 1], b[NC], out[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
#pragma unroll
        for (int j = 0; j < 2 * H + 1; ++j) {
            int64_t g = i + j - H;
            if (INS) g = g < 0 ? -1 - g : (g >= nx ? 2 * nx - 1 - g : g);
            else g &= nx - 1;
            win[k][j] = src[(int64_t)k * nx + g];
        }
        b[k] = (P::S == 2 && !ODD) ? base[(int64_t)k * nx + i] : T(0);
    }
    P::template stage<ODD>(c, win, b, out);
#pragma unroll
    for (int k = 0; k < NC; ++k) dst[(int64_t)k * nx + i] = out[k];
}

template <class P>
static cudaError_t launch_classic(int odd, const void *src, const void *base, void *dst, int64_t nx, const ConstBlock &cb, int bc,
                                  cudaStream_t st) {
    using T = typename P::real;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int tpb = 256;
    const unsigned blocks = (unsigned)((nx + tpb - 1) / tpb);
    if (bc) {
        if constexpr (P::INSULATED_OK) {
            classic_kernel<P, P::S == 2, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);   // heat: S = 1, never odd
            return cudaGetLastError();
        } else {
            return cudaErrorNotSupported;
        }
    }
    if (odd) classic_kernel<P, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
    else     classic_kernel<P, false><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
    return cudaGetLastError();
}

cudaError_t launch_classic_stage(int problem, int dtype, int odd, const void *win_src, const void *base, void *dst, int64_t nx,
                                 const ConstBlock &cb, int bc, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    SWEPT_DISPATCH(problem, dtype, P, e = launch_classic<P>(odd, win_src, base, dst, nx, cb, bc, st));
    return e;
}

}  // namespace swept
