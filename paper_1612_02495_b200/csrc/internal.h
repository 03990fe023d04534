// internal.h -- declarations shared by the translation units of libswept1d.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/swept1d.h"

namespace swept {

// Scheme constants of one handle, stored as the bytes of P<T>::Consts (row A0; the paper keeps them in a
// __constant__ struct, PAPER.md:42, 193 -- here they travel as a by-value kernel parameter, which lives in
// the same constant bank).
struct ConstBlock {
    alignas(8) unsigned char bytes[64];
};

enum { MODE_UP = 0, MODE_DIAMOND = 1, MODE_DOWN = 2 };

// Bytes in front of a handle's sync area (flags / counters of the launch-free kernels); word 0 is the abort word of the
// bounded waits (swept_wave.cuh: spin_gives_up).  The launch helpers zero the sync area, never the header.
constexpr int SYNC_HEADER = 16;

// One classic sub-timestep over all nx points (naive.cu).  odd: predictor stage of a two-stage scheme.
// dst[i] = stage(win_src[i-H..i+H], base[i]); base may alias dst.
// bc: SWEPT_BC_PERIODIC | SWEPT_BC_INSULATED (heat only: ghost value = adjacent interior value).
// share: Euler only -- the faces between the cells one thread updates are evaluated once (SWEPT_OPT_NAIVE_SHARE).
cudaError_t launch_classic_stage(int problem, int dtype, int odd, const void *win_src, const void *base, void *dst,
                                 int64_t nx, const ConstBlock &cb, int bc, int share, cudaStream_t st);

// Paper-style shared-memory swept kernels (swept_smem.cu): one block per tile of W points.
// mode: MODE_UP | MODE_DIAMOND | MODE_DOWN; offset: tile-grid shift (0 or W/2).
cudaError_t launch_swept_smem(int problem, int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset,
                              const ConstBlock &cb, cudaStream_t st);
size_t swept_smem_bytes(int problem, int dtype, int W);
cudaError_t swept_smem_prepare(int problem, int dtype, size_t max_bytes);

// Register-resident wavefront swept kernels (swept_wave.cu): one warp per tile of W points.
cudaError_t launch_swept_wave(int problem, int dtype, int mode, void *u, void *w, int64_t nx, int W, int64_t offset,
                              const ConstBlock &cb, int warps_per_block, int blocks_per_sm, int bc, cudaStream_t st);
// Launch-free sweep: ONE launch runs q half-cycles (1 upright + (q-1) diamond + 1 closing phase), tiles ordered by per-tile
// flags in `sync` (8 + 4*nx/W bytes, zeroed by the launch helper).
cudaError_t launch_swept_chain(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, void *sync, const ConstBlock &cb,
                               int warps_per_block, int blocks_per_sm, int sm_count, int bc, cudaStream_t st);
// Streaming band kernel (swept_band.cuh): ONE launch runs q half-cycles with every band's columns resident in registers /
// shared memory; `sync` = prog[nx/W] counters (zeroed by the helper).  cudaErrorNotSupported if the schedule does not fit
// the device (the caller then uses launch_swept_chain).  max_warps > 0 caps the resident warps per SM.
// pack != 0 (heat and KS fp32 only): two bands per warp slot, advanced by packed f32x2 arithmetic (stencils.cuh float2p).
// rt > 0: the remainder tiers as a truncated closing cycle inside the launch (as launch_swept_ring).
cudaError_t launch_swept_band(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb,
                              int sm_count, int max_smem, int max_warps, int pack, cudaStream_t st);
// Ring kernel (swept_ring.cuh): the band kernel with a communication warp per block (cp.async-staged edge exchange); ONE launch
// runs q half-cycles plus rt remainder tiers (rt = S x remaining timesteps < L).  `sync` = prog[nx/W] counters (zeroed by the
// helper).  cudaErrorNotSupported if the width / schedule does not fit (the caller then uses the band or the tile-flag kernel).
cudaError_t launch_swept_ring(int problem, int dtype, void *u, void *w, int64_t nx, int W, int64_t q, int rt, void *sync, const ConstBlock &cb,
                              int sm_count, int max_smem, int max_warps, cudaStream_t st);
int swept_ring_supports(int problem, int W);
int swept_wave_supports(int problem, int dtype, int W);
cudaError_t swept_wave_prepare(int problem, int dtype);

// ---- streaming-band schedule (swept_band.cuh): which warp owns which band.  Host logic shared by the kernel, the launch
// helper and swept_band_layout / swept_band_owner (C ABI, CPU-testable).
struct BandGrid {
    int nblocks, wpb, SL, wps, G, kmax;   // blocks, warps per block, sub-partition slots per block (min(wpb, 4)), warps per
                                          // slot, G = nblocks * SL slots in the grid, kmax = most bands any warp owns
};
// Grid for ntiles bands on sm_count SMs with wpb warps per block: one block per SM at most, no more blocks than needed.
__host__ __device__ inline BandGrid band_layout(int ntiles, int sm_count, int wpb) {
    BandGrid g;
    g.wpb = wpb;
    g.SL = wpb < 4 ? wpb : 4;
    g.wps = wpb / g.SL;
    const int nb = (ntiles + wpb - 1) / wpb;
    g.nblocks = nb < sm_count ? nb : sm_count;
    g.G = g.nblocks * g.SL;
    const int stride = g.G * g.wps;
    g.kmax = (ntiles + stride - 1) / stride;
    return g;
}
// Band n goes to slot n mod G (a slot = the warps of one block that share an SM sub-partition: warp % SL), dealing
// round n / G to warp (round mod wps) of the slot as its (round / wps)-th band: every slot carries floor or ceil of
// ntiles / G bands whatever ntiles and the SM count are.
__host__ __device__ inline int band_first(const BandGrid &g, int block, int warp) { return block * g.SL + warp % g.SL + g.G * (warp / g.SL); }
__host__ __device__ inline int band_stride(const BandGrid &g) { return g.G * g.wps; }
__host__ __device__ inline int band_count(const BandGrid &g, int block, int warp, int ntiles) {
    const int first = band_first(g, block, warp);
    return first < ntiles ? (ntiles - 1 - first) / band_stride(g) + 1 : 0;
}
__host__ __device__ inline void band_owner(const BandGrid &g, int band, int *block, int *warp, int *index) {
    const int slot = band % g.G, round = band / g.G;
    *block = slot / g.SL;
    *warp = slot % g.SL + g.SL * (round % g.wps);
    *index = round / g.wps;
}

// Record an error message for swept_last_error() (thread-local, api.cu) and return `code`.
int swept_fail(int code, const char *fmt, ...) __attribute__((format(printf, 2, 3)));

// FMA-chain microbenchmark (alu_peak.cu)
cudaError_t run_alu_peak(int dtype, int sm_count, double *instr_per_s, double *ms, cudaStream_t st);
cudaError_t run_smem_peak(int sm_count, double *bytes_per_s, double *ms, cudaStream_t st);
cudaError_t run_latency_probes(double *cycles, cudaStream_t st);

inline int radius_of(int problem) { return problem == SWEPT_HEAT ? 1 : 2; }
inline int stages_of(int problem) { return problem == SWEPT_HEAT ? 1 : 2; }
inline int ncomp_of(int problem) { return problem == SWEPT_EULER ? 3 : 1; }
inline size_t elem_size(int dtype) { return dtype == SWEPT_F64 ? 8 : 4; }

}  // namespace swept

// Dispatch a (problem, dtype) pair to a template taking <P<T>>: SWEPT_DISPATCH(problem, dtype, P, expr-using-P)
#define SWEPT_DISPATCH(problem, dtype, PNAME, ...)                                                        \
    do {                                                                                                  \
        if ((dtype) == SWEPT_F64) {                                                                       \
            if ((problem) == SWEPT_HEAT) { using PNAME = ::swept::Heat<double>; __VA_ARGS__; }            \
            else if ((problem) == SWEPT_KS) { using PNAME = ::swept::KS<double>; __VA_ARGS__; }           \
            else { using PNAME = ::swept::Euler<double>; __VA_ARGS__; }                                   \
        } else {                                                                                          \
            if ((problem) == SWEPT_HEAT) { using PNAME = ::swept::Heat<float>; __VA_ARGS__; }             \
            else if ((problem) == SWEPT_KS) { using PNAME = ::swept::KS<float>; __VA_ARGS__; }            \
            else { using PNAME = ::swept::Euler<float>; __VA_ARGS__; }                                    \
        }                                                                                                 \
    } while (0)
