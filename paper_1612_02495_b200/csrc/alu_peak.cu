// alu_peak.cu -- FMA-chain microbenchmark: the plain-ALU peak (FP64 or FP32 pipe) that bounds the swept
// kernels ("Swept path -> plain ALUs ... never tensor cores").  Each thread runs
// CHAINS independent fused multiply-adds per iteration, so the pipe, not latency, limits it.
#include "internal.h"

namespace swept {

template <class T, int CHAINS>
__global__ void __launch_bounds__(256) alu_peak_kernel(T *out, int iters, T a, T b) {
    T acc[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) acc[i] = (T)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < CHAINS; ++i) acc[i] = (sizeof(T) == 8) ? (T)fma((double)acc[i], (double)a, (double)b) : (T)fmaf((float)acc[i], (float)a, (float)b);
    }
    T sum = 0;
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) sum += acc[i];
    if (sum == (T)123456789) out[0] = sum;   // never true for the given a, b; keeps the chain alive
}

template <class T> static cudaError_t run_peak(int sm_count, double *instr_per_s, double *ms_out, cudaStream_t st) {
    constexpr int CHAINS = 8;
    T *d = nullptr;
    cudaError_t e = cudaMalloc(&d, sizeof(T));
    if (e != cudaSuccess) return e;
    const int blocks = sm_count * 8, threads = 256;
    const int iters = sizeof(T) == 8 ? 8192 : 16384;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // first repetition is the warm-up
        cudaEventRecord(e0, st);
        alu_peak_kernel<T, CHAINS><<<blocks, threads, 0, st>>>(d, iters, (T)0.999, (T)0.001);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double n = (double)blocks * threads * (double)iters * CHAINS;
    if (instr_per_s) *instr_per_s = n / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return cudaSuccess;
}

// Shared-memory read peak: every thread reads 16 bytes per instruction (LDS.128, consecutive threads consecutive addresses:
// conflict-free), 8 independent loads in flight; nominal 128 B per clock per SM (B300_MICROARCH guide: smem crossbar).
__global__ void __launch_bounds__(1024) smem_peak_kernel(float *out, int iters) {
    __shared__ float4 buf[2048];                                      // 32 KB
    for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int idx = threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const float4 v = buf[(idx + 256 * k) & 2047];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        idx = (idx + 32) & 2047;
    }
    if (acc.x + acc.y + acc.z + acc.w == 123456789.f) out[0] = acc.x;   // keeps the loads alive
}

cudaError_t run_smem_peak(int sm_count, double *bytes_per_s, double *ms_out, cudaStream_t st) {
    float *d = nullptr;
    cudaError_t e = cudaMalloc(&d, sizeof(float));
    if (e != cudaSuccess) return e;
    const int blocks = sm_count * 2, threads = 1024, iters = 4096;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        smem_peak_kernel<<<blocks, threads, 0, st>>>(d, iters);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (bytes_per_s) *bytes_per_s = (double)blocks * threads * (double)iters * 8 * 16 / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return cudaSuccess;
}

// Latency probes (one warp, dependent chains, clock64 around N repetitions): the numbers behind DESIGN.md's small-grid bound.
//   [0] dependent DFMA                      [1] the heat update's chain: DADD -> DFMA (+ an independent DMUL)
//   [2] dependent 64-bit __shfl_up          [3] a lock-step tier: two 64-bit shuffles -> DADD -> DFMA
//   [4] a tier through shared memory with one block barrier, 256 threads (store, barrier, two loads, DADD, DFMA)
template <int WHICH>
__global__ void latency_probe_kernel(double *out, double a, double b, int n) {
    __shared__ double sh[2][1024 + 2];
    double x = (double)threadIdx.x, l = 1.0, r = 2.0;
    if (WHICH == 4) {    // the two guard cells beside the 256 values no thread stores to
        if (threadIdx.x < 2) { sh[threadIdx.x][0] = 0.0; sh[threadIdx.x][blockDim.x + 1] = 0.0; }
        __syncthreads();
    }
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) {
        if (WHICH == 0) x = fma(x, a, b);
        else if (WHICH == 1) { const double t = x + l, v = b * r; x = fma(a, t, v); }
        else if (WHICH == 2) x = __shfl_up_sync(0xffffffffu, x, 1);
        else if (WHICH == 3) {
            const double lo = __shfl_up_sync(0xffffffffu, x, 1), hi = __shfl_down_sync(0xffffffffu, x, 1);
            const double t = lo + hi, v = b * x;
            x = fma(a, t, v);
        } else {
            double *s = sh[i & 1];
            s[threadIdx.x + 1] = x;
            __syncthreads();
            const double t = s[threadIdx.x] + s[threadIdx.x + 2], v = b * x;
            x = fma(a, t, v);
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) out[WHICH] = (double)(t1 - t0) / n;
    if (x == 123456789.0) out[7] = x;
}

cudaError_t run_latency_probes(double *cycles, cudaStream_t st) {
    double *d = nullptr;
    cudaError_t e = cudaMalloc(&d, 8 * sizeof(double));
    if (e != cudaSuccess) return e;
    cudaMemsetAsync(d, 0, 8 * sizeof(double), st);
    constexpr int N = 4096;
    for (int rep = 0; rep < 2; ++rep) {                       // the first pass warms the instruction cache
        latency_probe_kernel<0><<<1, 32, 0, st>>>(d, 1.0000001, 1e-9, N);
        latency_probe_kernel<1><<<1, 32, 0, st>>>(d, 0.25, 0.5, N);
        latency_probe_kernel<2><<<1, 32, 0, st>>>(d, 0.0, 0.0, N);
        latency_probe_kernel<3><<<1, 32, 0, st>>>(d, 0.25, 0.5, N);
        latency_probe_kernel<4><<<1, 256, 0, st>>>(d, 0.25, 0.5, N);
    }
    e = cudaMemcpyAsync(cycles, d, 5 * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t run_alu_peak(int dtype, int sm_count, double *instr_per_s, double *ms, cudaStream_t st) {
    return dtype == SWEPT_F64 ? run_peak<double>(sm_count, instr_per_s, ms, st) : run_peak<float>(sm_count, instr_per_s, ms, st);
}

}  // namespace swept
