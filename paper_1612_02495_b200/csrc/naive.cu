// naive.cu -- the classic decomposition (section IV.D; Fig. 6): one kernel per
// sub-timestep, a thread per 16 bytes of grid points, neighbours through the periodic index `& (nx-1)`
// (PAPER.md:171), global memory in and out.  SURVEY.md section 8(a) row A2.
#include "internal.h"
#include "stencils.cuh"

namespace swept {

// INS: insulated ends (Eq. 9): a neighbour index outside the rod is mirrored back, -1 -> 0 and
// nx -> nx-1 (the ghost value is the adjacent interior value).
//
// A thread updates V = 16 / sizeof(T) consecutive points: one aligned 16-byte load and store per field for the points
// themselves and 2H scalar loads for the halo (the naive path is bound by memory bandwidth; with one
// point per thread it is bound by instruction issue instead -- fp32 heat reached 42 % of the HBM copy bandwidth at nx = 2^28).
// Every point still goes through the same P::stage<ODD> as in the swept kernels.
template <class T> struct vec16;
template <> struct vec16<double> { using type = double2; static constexpr int V = 2; };
template <> struct vec16<float> { using type = float4; static constexpr int V = 4; };

template <bool INS> __device__ __forceinline__ int64_t classic_index(int64_t g, int64_t nx) {
    if (INS) return g < 0 ? -1 - g : (g >= nx ? 2 * nx - 1 - g : g);
    return g & (nx - 1);
}

template <class P, bool ODD, bool INS = false, bool SHARE = false>
__global__ void __launch_bounds__(256) classic_kernel(const typename P::real *__restrict__ src, const typename P::real *base,
                                                       typename P::real *dst, int64_t nx, typename P::Consts c) {
    using T = typename P::real;
    using VT = typename vec16<T>::type;
    constexpr int H = P::H, NC = P::NC, V = vec16<T>::V;
    const int64_t i0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * V;
    if (i0 >= nx) return;
    T w[NC][V + 2 * H], b[NC][V], out[V][NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const VT v = *reinterpret_cast<const VT *>(src + (int64_t)k * nx + i0);
        const T *pv = reinterpret_cast<const T *>(&v);
#pragma unroll
        for (int j = 0; j < V; ++j) w[k][H + j] = pv[j];
#pragma unroll
        for (int j = 0; j < H; ++j) {
            w[k][j] = src[(int64_t)k * nx + classic_index<INS>(i0 - H + j, nx)];
            w[k][H + V + j] = src[(int64_t)k * nx + classic_index<INS>(i0 + V + j, nx)];
        }
        if (P::S == 2 && !ODD) {
            const VT bv = *reinterpret_cast<const VT *>(base + (int64_t)k * nx + i0);
            const T *pb = reinterpret_cast<const T *>(&bv);
#pragma unroll
            for (int j = 0; j < V; ++j) b[k][j] = pb[j];
        } else {
#pragma unroll
            for (int j = 0; j < V; ++j) b[k][j] = T(0);
        }
    }
    if constexpr (SHARE && P::GROUPED) {
        // SWEPT_OPT_NAIVE_SHARE: the faces between the thread's V cells are evaluated once (V + 1 faces instead of 2 V)
        T bb[V][NC];
#pragma unroll
        for (int j = 0; j < V; ++j)
#pragma unroll
            for (int k = 0; k < NC; ++k) bb[j][k] = b[k][j];
        P::template cells<V>(c, ODD, w, bb, out);
    } else {
#pragma unroll
    for (int j = 0; j < V; ++j) {
        T win[NC][2 * H + 1], bb[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) {
#pragma unroll
            for (int m = 0; m < 2 * H + 1; ++m) win[k][m] = w[k][j + m];
            bb[k] = b[k][j];
        }
        P::template stage<ODD>(c, win, bb, out[j]);
    }
    }
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        VT v;
        T *pv = reinterpret_cast<T *>(&v);
#pragma unroll
        for (int j = 0; j < V; ++j) pv[j] = out[j][k];
        *reinterpret_cast<VT *>(dst + (int64_t)k * nx + i0) = v;
    }
}

template <class P>
static cudaError_t launch_classic(int odd, const void *src, const void *base, void *dst, int64_t nx, const ConstBlock &cb, int bc, int share,
                                  cudaStream_t st) {
    using T = typename P::real;
    const typename P::Consts c = *reinterpret_cast<const typename P::Consts *>(cb.bytes);
    const int tpb = 256;
    const int64_t threads = nx / vec16<T>::V;                 // nx is a power of two >= 8
    const unsigned blocks = (unsigned)((threads + tpb - 1) / tpb);
    if (bc) {
        if constexpr (P::INSULATED_OK) {
            classic_kernel<P, P::S == 2, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);   // heat: S = 1, never odd
            return cudaGetLastError();
        } else {
            return cudaErrorNotSupported;
        }
    }
    if constexpr (P::GROUPED) {
        if (share) {
            if (odd) classic_kernel<P, true, false, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
            else     classic_kernel<P, false, false, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
            return cudaGetLastError();
        }
    }
    if (odd) classic_kernel<P, true><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
    else     classic_kernel<P, false><<<blocks, tpb, 0, st>>>((const T *)src, (const T *)base, (T *)dst, nx, c);
    return cudaGetLastError();
}

cudaError_t launch_classic_stage(int problem, int dtype, int odd, const void *win_src, const void *base, void *dst, int64_t nx,
                                 const ConstBlock &cb, int bc, int share, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    SWEPT_DISPATCH(problem, dtype, P, e = launch_classic<P>(odd, win_src, base, dst, nx, cb, bc, share, st));
    return e;
}

}  // namespace swept
