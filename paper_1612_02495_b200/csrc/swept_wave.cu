// swept_wave.cu -- problem dispatch for the wavefront swept kernels (instantiated in swept_wave_<problem>.cu).
#include "internal.h"

namespace swept {

#define DECL(prob)                                                                                                              \
    cudaError_t launch_swept_wave_##prob(int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset,              \
                                         const ConstBlock &cb, int wpb, size_t smem_floor, int bc, cudaStream_t st);            \
    cudaError_t launch_swept_chain_##prob(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, void *sync,                \
                                          const ConstBlock &cb, int wpb, size_t smem_floor, int sm_count, int bc, cudaStream_t st); \
    cudaError_t swept_wave_prepare_##prob(int dtype, int max_smem);                                                             \
    cudaError_t launch_swept_band_##prob(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync,         \
                                         const ConstBlock &cb, int sm_count, int max_smem, int max_warps, int pack, cudaStream_t st); \
    cudaError_t swept_band_prepare_##prob(int dtype, int max_smem);                                                             \
    cudaError_t launch_swept_ring_##prob(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync,         \
                                         const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st);     \
    cudaError_t swept_ring_prepare_##prob(int dtype, int max_smem);                                                             \
    int swept_ring_supports_##prob(int W);                                                                                      \
    int swept_wave_supports_##prob(int W);
DECL(heat)
DECL(ks)
DECL(euler)
#undef DECL

// Shared memory request that caps resident blocks per SM at `cap` (SWEPT_OPT_BLOCKS_PER_SM): each block is charged its
// request plus 1 KB of system use against the SM's 228 KB.
size_t smem_floor_for_cap(int cap) {
    if (cap <= 0) return 0;
    const size_t total = 228 * 1024, sys = 1024, limit = 227 * 1024;
    size_t req = total / (size_t)cap - sys;
    return req > limit ? limit : req;
}

cudaError_t launch_swept_wave(int problem, int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset,
                              const ConstBlock &cb, int warps_per_block, int blocks_per_sm, int bc, cudaStream_t st) {
    const size_t floor = smem_floor_for_cap(blocks_per_sm);
    if (problem == SWEPT_HEAT) return launch_swept_wave_heat(dtype, mode, u, w, nx, W, offset, cb, warps_per_block, floor, bc, st);
    if (problem == SWEPT_KS) return launch_swept_wave_ks(dtype, mode, u, w, nx, W, offset, cb, warps_per_block, floor, bc, st);
    return launch_swept_wave_euler(dtype, mode, u, w, nx, W, offset, cb, warps_per_block, floor, bc, st);
}

cudaError_t launch_swept_chain(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, void *sync, const ConstBlock &cb,
                               int warps_per_block, int blocks_per_sm, int sm_count, int bc, cudaStream_t st) {
    const size_t floor = smem_floor_for_cap(blocks_per_sm);
    if (problem == SWEPT_HEAT) return launch_swept_chain_heat(dtype, u, w, nx, W, q, sync, cb, warps_per_block, floor, sm_count, bc, st);
    if (problem == SWEPT_KS) return launch_swept_chain_ks(dtype, u, w, nx, W, q, sync, cb, warps_per_block, floor, sm_count, bc, st);
    return launch_swept_chain_euler(dtype, u, w, nx, W, q, sync, cb, warps_per_block, floor, sm_count, bc, st);
}

cudaError_t launch_swept_band(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb,
                              int sm_count, int max_smem, int max_warps, int pack, cudaStream_t st) {
    if (problem == SWEPT_HEAT) return launch_swept_band_heat(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, pack, st);
    if (problem == SWEPT_KS) return launch_swept_band_ks(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, pack, st);
    return launch_swept_band_euler(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, 0, st);
}

cudaError_t launch_swept_ring(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb,
                              int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    if (problem == SWEPT_HEAT) return launch_swept_ring_heat(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
    if (problem == SWEPT_KS) return launch_swept_ring_ks(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
    return launch_swept_ring_euler(dtype, u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
}

int swept_ring_supports(int problem, int W) {
    if (problem == SWEPT_HEAT) return swept_ring_supports_heat(W);
    if (problem == SWEPT_KS) return swept_ring_supports_ks(W);
    return swept_ring_supports_euler(W);
}

int swept_wave_supports(int problem, int dtype, int W) {
    (void)dtype;
    if (problem == SWEPT_HEAT) return swept_wave_supports_heat(W);
    if (problem == SWEPT_KS) return swept_wave_supports_ks(W);
    return swept_wave_supports_euler(W);
}

cudaError_t swept_wave_prepare(int problem, int dtype) {
    int dev = 0, max_smem = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaError_t e;
    if (problem == SWEPT_HEAT) {
        if ((e = swept_wave_prepare_heat(dtype, max_smem)) != cudaSuccess) return e;
        if ((e = swept_ring_prepare_heat(dtype, max_smem)) != cudaSuccess) return e;
        return swept_band_prepare_heat(dtype, max_smem);
    }
    if (problem == SWEPT_KS) {
        if ((e = swept_wave_prepare_ks(dtype, max_smem)) != cudaSuccess) return e;
        if ((e = swept_ring_prepare_ks(dtype, max_smem)) != cudaSuccess) return e;
        return swept_band_prepare_ks(dtype, max_smem);
    }
    if ((e = swept_wave_prepare_euler(dtype, max_smem)) != cudaSuccess) return e;
    if ((e = swept_ring_prepare_euler(dtype, max_smem)) != cudaSuccess) return e;
    return swept_band_prepare_euler(dtype, max_smem);
}

}  // namespace swept
