// swept_wave_ks.cu -- instantiations of the wavefront swept kernels (swept_wave.cuh) for the ks problem.
#include "swept_wave.cuh"
namespace swept {
template <class T> static cudaError_t launch_t(int mode, void *u, void *w, int64_t nx, int W, int64_t offset, const ConstBlock &cb, int wpb, size_t smem_floor, int bc, cudaStream_t st) {
    switch (W / 32) {
        case 4: return wave_launch_pw<KS<T>, 4>(mode, u, w, nx, offset, cb, wpb, smem_floor, bc, st);
        case 8: return wave_launch_pw<KS<T>, 8>(mode, u, w, nx, offset, cb, wpb, smem_floor, bc, st);
        case 16: return wave_launch_pw<KS<T>, 16>(mode, u, w, nx, offset, cb, wpb, smem_floor, bc, st);
        case 32: return wave_launch_pw<KS<T>, 32>(mode, u, w, nx, offset, cb, wpb, smem_floor, bc, st);
        default: return cudaErrorInvalidValue;
    }
}
template <class T> static cudaError_t chain_t(void *u, void *w, int64_t nx, int W, int64_t q, void *sync, const ConstBlock &cb, int wpb, size_t smem_floor, int sm_count, int bc, cudaStream_t st) {
    switch (W / 32) {
        case 4: return wave_chain_pw<KS<T>, 4>(u, w, nx, q, sync, cb, wpb, smem_floor, sm_count, bc, st);
        case 8: return wave_chain_pw<KS<T>, 8>(u, w, nx, q, sync, cb, wpb, smem_floor, sm_count, bc, st);
        case 16: return wave_chain_pw<KS<T>, 16>(u, w, nx, q, sync, cb, wpb, smem_floor, sm_count, bc, st);
        case 32: return wave_chain_pw<KS<T>, 32>(u, w, nx, q, sync, cb, wpb, smem_floor, sm_count, bc, st);
        default: return cudaErrorInvalidValue;
    }
}
template <class T> static cudaError_t prepare_t(int max_smem) {
    cudaError_t e = cudaSuccess;
    if ((e = wave_prepare_pw<KS<T>, 4>(max_smem)) != cudaSuccess) return e;
    if ((e = wave_prepare_pw<KS<T>, 8>(max_smem)) != cudaSuccess) return e;
    if ((e = wave_prepare_pw<KS<T>, 16>(max_smem)) != cudaSuccess) return e;
    if ((e = wave_prepare_pw<KS<T>, 32>(max_smem)) != cudaSuccess) return e;
    return e;
}
cudaError_t launch_swept_wave_ks(int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset, const ConstBlock &cb, int wpb, size_t smem_floor, int bc, cudaStream_t st) {
    return dtype == SWEPT_F64 ? launch_t<double>(mode, u, w, nx, W, offset, cb, wpb, smem_floor, bc, st) : launch_t<float>(mode, u, w, nx, W, offset, cb, wpb, smem_floor, bc, st);
}
cudaError_t launch_swept_chain_ks(int dtype, void *u, void *w, int64_t nx, int W, int64_t q, void *sync, const ConstBlock &cb, int wpb, size_t smem_floor, int sm_count, int bc, cudaStream_t st) {
    return dtype == SWEPT_F64 ? chain_t<double>(u, w, nx, W, q, sync, cb, wpb, smem_floor, sm_count, bc, st) : chain_t<float>(u, w, nx, W, q, sync, cb, wpb, smem_floor, sm_count, bc, st);
}
cudaError_t swept_wave_prepare_ks(int dtype, int max_smem) { return dtype == SWEPT_F64 ? prepare_t<double>(max_smem) : prepare_t<float>(max_smem); }
int swept_wave_supports_ks(int W) {
    switch (W) {
        case 128: return 1;
        case 256: return 1;
        case 512: return 1;
        case 1024: return 1;
        default: return 0;
    }
}
}  // namespace swept
