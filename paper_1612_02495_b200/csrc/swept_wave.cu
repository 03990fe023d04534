// swept_wave.cu -- placeholder until the register-resident wavefront kernels land.
#include "internal.h"
namespace swept {
cudaError_t launch_swept_wave(int, int, int, void *, void *, int64_t, int, int64_t, const ConstBlock &, int, int, cudaStream_t) { return cudaErrorNotSupported; }
int swept_wave_supports(int, int, int) { return 0; }
cudaError_t swept_wave_prepare(int, int) { return cudaSuccess; }
}
