// swept_ring_ks.cu -- instantiations of the ring kernel (swept_ring.cuh) for the ks problem.
#include "swept_ring.cuh"
namespace swept {
template <class T> static cudaError_t ring_t(void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    switch (W / 32) {
        case 8: return wave_ring<KS<T>, 8>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 16: return wave_ring<KS<T>, 16>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 32: return wave_ring<KS<T>, 32>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        default: return cudaErrorNotSupported;
    }
}
template <class T> static cudaError_t prepare_t(int max_smem) {
    cudaError_t e = cudaSuccess;
    if ((e = ring_prepare<KS<T>, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = ring_prepare<KS<T>, 16>(max_smem)) != cudaSuccess) return e;
    if ((e = ring_prepare<KS<T>, 32>(max_smem)) != cudaSuccess) return e;
    return e;
}
cudaError_t launch_swept_ring_ks(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    return dtype == SWEPT_F64 ? ring_t<double>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st) : ring_t<float>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
}
cudaError_t swept_ring_prepare_ks(int dtype, int max_smem) { return dtype == SWEPT_F64 ? prepare_t<double>(max_smem) : prepare_t<float>(max_smem); }
int swept_ring_supports_ks(int W) {
    switch (W) {
        case 256: return ring_supports<KS<double>, 8>() ? 1 : 0;
        case 512: return ring_supports<KS<double>, 16>() ? 1 : 0;
        case 1024: return ring_supports<KS<double>, 32>() ? 1 : 0;
        default: return 0;
    }
}
}  // namespace swept
