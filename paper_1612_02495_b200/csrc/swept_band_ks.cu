// swept_band_ks.cu -- instantiations of the streaming band kernel (swept_band.cuh) for the ks problem.
#include "swept_band.cuh"
namespace swept {
template <class T> static cudaError_t band_t(void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, cudaStream_t st) {
    switch (W / 32) {
        case 4: return wave_band_pw<KS<T>, 4>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 8: return wave_band_pw<KS<T>, 8>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 16: return wave_band_pw<KS<T>, 16>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        case 32: return wave_band_pw<KS<T>, 32>(u, w, nx, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        default: return cudaErrorNotSupported;
    }
}
template <class T> static cudaError_t prepare_t(int max_smem) {
    cudaError_t e = cudaSuccess;
    if ((e = band_prepare_pw<KS<T>, 4>(max_smem)) != cudaSuccess) return e;
    if ((e = band_prepare_pw<KS<T>, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = band_prepare_pw<KS<T>, 16>(max_smem)) != cudaSuccess) return e;
    if ((e = band_prepare_pw<KS<T>, 32>(max_smem)) != cudaSuccess) return e;
    return e;
}
cudaError_t launch_swept_band_ks(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb, int sm_count, int max_smem, int max_warps, int pack, cudaStream_t st) {
    if (dtype == SWEPT_F32 && pack) {
        // two bands per warp slot on packed f32x2 arithmetic (as heat fp32); falls through to one band per slot where the paired schedule does not fit
        const cudaError_t e = band_t<float2p>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
        if (e != cudaErrorNotSupported && e != cudaErrorCooperativeLaunchTooLarge) return e;
        cudaGetLastError();
    }
    return dtype == SWEPT_F64 ? band_t<double>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st) : band_t<float>(u, w, nx, W, q, rt, sync, cb, sm_count, max_smem, max_warps, st);
}
cudaError_t swept_band_prepare_ks(int dtype, int max_smem) {
    if (dtype == SWEPT_F64) return prepare_t<double>(max_smem);
    const cudaError_t e = prepare_t<float2p>(max_smem);
    return e != cudaSuccess ? e : prepare_t<float>(max_smem);
}
}  // namespace swept
