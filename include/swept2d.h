/* swept2d.h -- C ABI of the 2-D part of libswept1d.so: the swept rule for the 2-D heat equation.
 *
 * The paper names "implementing the 2D swept rule on the GPU" as future work and gives neither a scheme nor a
 * decomposition.  Scheme here: the paper's own heat discretisation (forward in time, second-order central in space, Eq. (5)-(8)
 * PAPER.md:250-263) on a square mesh dx = dy with periodic ends in both directions:
 *     T_{i,j}^{m+1} = Fo (T_{i+1,j} + T_{i-1,j} + T_{i,j+1} + T_{i,j-1}) + (1 - 4 Fo) T_{i,j},     Fo = alpha dt / dx^2.
 * Decomposition: the product of the paper's 1-D rule with itself.  With tiles of W x W
 * points and L = W/2 tiers per half-cycle, every point is at tier s = 1..L in exactly one of: the shrinking square [s, W-s)^2 of
 * an aligned tile (upright pyramid), an x-bridge [c-s, c+s) x [s, W-s) or a y-bridge, or the growing square [c-s, c+s)^2 of a tile
 * shifted by (W/2, W/2) (inverted pyramid).  Pyramids need nothing but themselves, bridges need the pyramids, inverted pyramids
 * need all three; the inverted pyramid of one half-cycle and the upright pyramid of the next share a tile and run as one
 * octahedron.  A half-cycle of L timesteps is therefore two launches (bridges, octahedra) and touches global memory twice per
 * point instead of L times.  Values are exchanged in place through d_u (newest even tier of every point) and the handle's
 * workspace (newest odd tier), the 2-D form of the staircase rows of swept1d.h.
 *
 * Conventions as in swept1d.h: d_* are device pointers; the field is [ny][nx] row-major (x fastest), 16-byte aligned, advanced
 * in place and asynchronously on `cuda_stream`; 0 on success, negative SWEPT_E* otherwise with the message in swept_last_error();
 * no CPU fallback.  The result of swept2d_run is bit-identical to naive2d_run (one shared device stencil function).
 */
#ifndef SWEPT2D_H
#define SWEPT2D_H

#include <stdint.h>

#include "swept1d.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swept2d_ctx *swept2d_handle_t; /* opaque; owned by the library */

typedef struct {
    int dtype;    /* SWEPT_F32 | SWEPT_F64 */
    double alpha; /* thermal diffusivity   */
} swept2d_params_t;

typedef struct {
    int dtype;
    int64_t nx, ny;
    int64_t workspace_bytes;    /* the odd-tier array / the classic path's second buffer */
    int64_t launches_last_call; /* kernels the last swept2d_run / naive2d_run enqueued    */
    int64_t launches_total;
} swept2d_info_t;

/* nx, ny: powers of two >= 8 (periodic neighbours by `& (n-1)`), nx <= 2^20, ny <= 2^18 (rows of blocks go on
 * blockIdx.y, which the device limits to 65535); dx = dy; `p` may be NULL (f64, alpha = 1).
 * Allocates nx*ny elements of workspace on the current device.  Errors: SWEPT_EINVAL, SWEPT_ENOMEM, SWEPT_ECUDA. */
int swept2d_create(swept2d_handle_t *out, int64_t nx, int64_t ny, double dx, double dt, const swept2d_params_t *p);

/* Advance d_u by nsteps timesteps with the 2-D swept rule.  tile_width W in {8, 16, 32} (W <= nx, ny; L = W/2 even so that the
 * flat field lands on the even-tier array d_u); 0 = 32 (or the largest that fits).  nsteps = K L + r: the r remainder timesteps
 * run first on the classic kernel, then 1 pyramid launch + K x (bridges, octahedra) launches, the last octahedra launch only up
 * to its waist.  Errors: SWEPT_EINVAL (NULL, nsteps < 0, illegal width), SWEPT_ECUDA. */
int swept2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, int tile_width, void *cuda_stream);

/* The classic decomposition: one kernel per timestep over all nx*ny points, ping-pong with the workspace. */
int naive2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, void *cuda_stream);

/* End-to-end convenience used for the `e2e` measurement: copy h_u (HOST, [ny][nx], ideally pinned) to an internal device buffer
 * (allocated on first use), swept2d_run (use_swept != 0) or naive2d_run on it, copy the result back into h_u, and synchronise
 * the stream.  Errors as the run calls, SWEPT_ENOMEM. */
int swept2d_run_host(swept2d_handle_t h, void *h_u, int64_t nsteps, int tile_width, int use_swept, void *cuda_stream);

/* SWEPT2D_OPT_KERNEL: which kernels run tiles of W = 32 (W = 8, 16 always run on the shared-memory kernels).
 *   SWEPT2D_KERNEL_WARP (default)  one warp per tile, both planes of the tile in registers, no barrier; a lane holds two columns of 16
 *                                  rows (the tile's upper half folded onto lanes 16..31): one shuffle per point
 *   SWEPT2D_KERNEL_SMEM            the paper's design in 2-D (Fig. 5): block = tile, thread = point, two shared-memory planes
 *   SWEPT2D_KERNEL_COLUMN          one warp per tile, a lane holds one column of 32 rows: two shuffles per point (the first register
 *                                  kernel; kept for comparison)
 * Same regions, tier order and store rule: all are interchangeable launch by launch and bit-identical.  Errors: SWEPT_EINVAL. */
#define SWEPT2D_OPT_KERNEL 0
#define SWEPT2D_KERNEL_WARP 0
#define SWEPT2D_KERNEL_SMEM 1
#define SWEPT2D_KERNEL_COLUMN 2
int swept2d_set_option(swept2d_handle_t h, int option, int value);

int swept2d_get_info(swept2d_handle_t h, swept2d_info_t *info);
int swept2d_destroy(swept2d_handle_t h);

#ifdef __cplusplus
}
#endif
#endif /* SWEPT2D_H */
