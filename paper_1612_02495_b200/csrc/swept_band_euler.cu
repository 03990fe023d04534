// swept_band_euler.cu -- instantiations of the streaming band kernel (swept_band.cuh) for the euler problem.
#include "swept_band.cuh"
namespace swept {
template <class T> static cudaError_t band_t(void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    switch (W / 32) {
        case 4: return wave_band_pw<Euler<T>, 4>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 8: return wave_band_pw<Euler<T>, 8>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 16: return wave_band_pw<Euler<T>, 16>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        default: return cudaErrorNotSupported;
    }
}
template <class T> static cudaError_t prepare_t(int max_smem) {
    cudaError_t e = cudaSuccess;
    if ((e = band_prepare_pw<Euler<T>, 4>(max_smem)) != cudaSuccess) return e;
    if ((e = band_prepare_pw<Euler<T>, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = band_prepare_pw<Euler<T>, 16>(max_smem)) != cudaSuccess) return e;
    return e;
}
cudaError_t launch_swept_band_euler(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, int, cudaStream_t st) {
    return dtype == SWEPT_F64 ? band_t<double>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st) : band_t<float>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
}
cudaError_t swept_band_prepare_euler(int dtype, int max_smem) { return dtype == SWEPT_F64 ? prepare_t<double>(max_smem) : prepare_t<float>(max_smem); }
}  // namespace swept
