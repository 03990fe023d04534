/* swept1d.h -- C ABI of the B200-native swept time-space decomposition library (libswept1d.so).
 *
 * Method: Magee & Niemeyer, "An initial investigation of the performance of GPU-based swept
 * time-space decomposition" (arXiv 1612.02495), cited below as PAPER.md:<line>.  The library
 * advances an explicit 1-D scheme on a periodic grid of nx points either
 *   - by the swept rule: every tile of W points advances through an
 *     upright triangle, then diamonds on tiles shifted by W/2, then a closing inverted triangle,
 *     touching global memory once per W/(2h) sub-timesteps, or
 *   - by the classic decomposition (Fig. 6): one kernel per sub-timestep.
 * Both evaluate the same device stencil functions, so their results are bit-identical.
 *
 * Conventions for every entry point
 *   - All pointers named d_* are DEVICE pointers, h_* are HOST pointers; sizes are element counts.
 *   - Field layout: [ncomp][nx] contiguous, structure of arrays (Euler: rho row, m = rho*u row,
 *     E row; heat and KS: one row), dtype as given at creation, base address 16-byte aligned.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     swept_run / naive_run only ENQUEUE work on that stream: they never synchronise and never
 *     allocate.  The field holds the solution at time +nsteps*dt when the stream reaches the end
 *     of the enqueued work.
 *   - Return value: 0 on success, negative on error (SWEPT_EINVAL / ENOMEM / ECUDA); the message is
 *     available from swept_last_error() (thread-local).  Nothing is printed, nothing aborts.
 *     Numerical blow-up is not an error: values become Inf/NaN exactly as the classic path's would.
 *   - No CPU fallback exists: without a CUDA device every compute call fails with SWEPT_ECUDA.
 *   - A handle owns device scratch (workspace, flags, cached graphs) on the device that was current at swept_create; every
 *     later call must be made with that device current (SWEPT_EINVAL otherwise).  Use a handle from one host thread at a
 *     time.  Calls on one handle from different streams are legal: each call first makes its stream wait (on the device,
 *     cudaStreamWaitEvent) for the handle's previous call, so they run one after the other.  Different handles are
 *     independent and run concurrently on different streams.  (A call made inside the caller's own stream capture skips
 *     that wait; the caller's graph must then order the handle's uses itself.)
 *   - The launch-free kernels wait on flags other warps of the same launch publish; every such wait is bounded (seconds).
 *     A wait that gives up makes the kernel exit and marks the handle: the field that launch ran on is invalid, and so is the
 *     result of every sweep enqueued on the handle behind it, until the mark is reported.  It is reported ONCE, as SWEPT_ECUDA,
 *     by swept_check(h) (which waits for the handle's work), by swept_run_host (which synchronises anyway), or by the first
 *     swept_run / naive_run / swept_tune on the handle that is called after the marked launch has finished on the device; a call
 *     made while it is still running cannot know yet.  Reporting clears the mark: the handle works again.  A caller that
 *     synchronises its own stream and reads d_u without another handle call should call swept_check first.
 */
#ifndef SWEPT1D_H
#define SWEPT1D_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swept_ctx *swept_handle_t; /* opaque; owned by the library */

/* problem -- the per-problem stencil device functions (radius h, stages S, fields ncomp):
 *   SWEPT_HEAT   FTCS, Eq. (2) PAPER.md:54                                   h=1 S=1 ncomp=1
 *   SWEPT_KS     Kuramoto-Sivashinsky, Eq. (4),(15),(16) PAPER.md:64,291,295 h=2 S=2 ncomp=1
 *   SWEPT_EULER  MUSCL/minmod/Rusanov midpoint (BASELINE.json config 4)      h=2 S=2 ncomp=3   */
enum { SWEPT_HEAT = 0, SWEPT_KS = 1, SWEPT_EULER = 2 };
/* dtype -- the paper's compile-time REAL as a run-time choice */
enum { SWEPT_F32 = 0, SWEPT_F64 = 1 };
enum { SWEPT_OK = 0, SWEPT_EINVAL = -1, SWEPT_ENOMEM = -2, SWEPT_ECUDA = -3 };
/* boundary -- SWEPT_BC_PERIODIC: neighbours mod nx (every BASELINE.json config).
 *             SWEPT_BC_INSULATED (heat only): the paper's heat problem, a rod with insulated ends (Eq. 9
 *             PAPER.md:266-269): the ghost value beyond an end is the adjacent interior value, T_0 = T_1.  On the shifted
 *             half-cycles the tile that is "split across the spatial boundary" becomes two tiles, one per end,
 *             each evaluated on the mirror image of its half (WAVE kernels; the band schedule needs a periodic domain, so the
 *             launch-free sweep runs on the tile-flag kernel). */
enum { SWEPT_BC_PERIODIC = 0, SWEPT_BC_INSULATED = 1 };

/* Which swept kernels swept_run uses (SWEPT_OPT_KERNEL):
 *   SWEPT_KERNEL_SMEM  the paper's design (Fig. 5): one block per tile, one
 *                      thread per point, two-row shared-memory matrix, a block barrier per tier.
 *   SWEPT_KERNEL_WAVE  B200 design: one lane group per tile, tile values resident in registers,
 *                      tiers evaluated as a lane-skewed wavefront over the diamond's characteristic
 *                      lattice, halos by warp shuffle (generalises PAPER.md:183).  Default.      */
enum { SWEPT_KERNEL_SMEM = 0, SWEPT_KERNEL_WAVE = 1 };

/* swept_set_option keys */
enum {
    SWEPT_OPT_KERNEL = 0,         /* SWEPT_KERNEL_*                                              */
    SWEPT_OPT_NAIVE_GRAPH = 1,    /* 1: naive_run replays a CUDA graph of its launches (default 0:
                                     plain launches = the paper's classic program)               */
    SWEPT_OPT_BLOCKS_PER_SM = 2,  /* cap on resident blocks per SM for the swept kernels (the band kernel, which runs one
                                     block per SM, caps its warps at 4 x this), 0 = none / the tuner's choice        */
    SWEPT_OPT_WARPS_PER_BLOCK = 3,/* WAVE kernels: lane groups are packed this many warps a block   */
    SWEPT_OPT_SWEPT_GRAPH = 4,    /* 1: swept_run replays a CUDA graph of its half-cycle launches  */
    SWEPT_OPT_NAIVE_SHARE = 7,    /* Euler, classic path: 1 = a thread evaluates the faces between the 2 (fp64) / 4 (fp32) cells it updates
                                     once (3 / 5 face fluxes instead of 4 / 8): the same operations on the same operands, bit-identical.
                                     Default 0: every point through the per-point stencil function, the paper's naive kernel (Fig. 6).
                                     Ignored for heat and KS                                                            */
    SWEPT_OPT_INJECT_ABORT = 8,   /* fault injection for tests of the error path (value 1; waits for the handle's work): marks the
                                     handle as if a bounded wait of a launch-free kernel had given up.  The next sweep's waiting
                                     warps leave early, and the mark is reported as described under "Conventions"            */
    SWEPT_OPT_PACK = 6,           /* heat and KS fp32 on the streaming band kernel: 2 = every warp slot advances TWO bands (half a domain
                                     apart) in lock step on packed f32x2 arithmetic (FADD2 / FMUL2 / FFMA2: half the FP
                                     instructions, per-component IEEE rounding, so the result is bit-identical); 1 = one band
                                     per slot; 0 (default) = swept_tune's measurement for the tuned width, else (heat only) on
                                     when every SM gets at least sixteen bands.  Ignored for fp64 and for Euler      */
    SWEPT_OPT_CHAIN = 5           /* WAVE kernels, launch-free sweep (beyond the paper; removes PAPER.md:232's launch / wave
                                     costs): ONE persistent launch runs all half-cycles of a swept_run.
                                     3 (default) = streaming bands with a communication warp per block: as 2, but the edge
                                         exchange is staged by cp.async through shared-memory rings by a dedicated warp, so the
                                         computing warps never wait on global memory, and the remainder timesteps (nsteps mod
                                         L/S) run inside the same launch as a truncated closing cycle: swept_run is
                                         ONE launch for any nsteps.  Falls back to 2 where the width / schedule does not fit.
                                     2 = streaming bands: a warp keeps its tile's columns in registers from one
                                         half-cycle to the next (the upper-left edge of PAPER.md Fig. 2b never leaves the
                                         SM), only the upper-right edge travels through global memory, ordered by one
                                         progress counter per band; falls back to 1 when the schedule does not fit.
                                     1 = tiles handed out by an atomic counter, ordered by per-tile flags, both edges
                                         through global memory every half-cycle.
                                     0 = one launch per half-cycle as in the paper    */
};

/* Shared memory a block may opt in to on B200 (227 KB); swept_plan, which has no device, checks SMEM-kernel tile widths
 * against it (a handle checks against the device's own attribute). */
#define SWEPT_SMEM_LIMIT_B200 232448

/* One entry of the launch plan of swept_run (host driver):
 *   CLASSIC  `count` classic timesteps (count * S kernels)
 *   UP       upright triangles, tiles at `offset`                                  (Fig. 5)
 *   DIAMOND  `count` consecutive diamond launches, the first at `offset`, then alternating 0 <-> W/2
 *   DOWN     closing inverted triangles at `offset`
 *   CHAIN    `count` half-cycles (1 UP + (count-1) DIAMOND + 1 DOWN phases, offsets 0, W/2, 0, ...) in ONE launch
 *   BAND     `count` half-cycles AND `offset` remainder timesteps (a truncated closing cycle, as RING) in ONE launch of the
 *            streaming band kernel (SWEPT_OPT_CHAIN = 2; a handle whose device cannot hold the band schedule runs the same
 *            timesteps as the plan of SWEPT_OPT_CHAIN = 1)
 *   RING     `count` half-cycles AND `offset` remainder timesteps (offset < L/S; a truncated closing cycle) in ONE launch of
 *            the ring kernel (SWEPT_OPT_CHAIN = 3): the whole swept_run.  A handle whose device cannot hold the schedule runs
 *            the same timesteps as the plan of SWEPT_OPT_CHAIN = 2.                                                   */
enum { SWEPT_LAUNCH_CLASSIC = 0, SWEPT_LAUNCH_UP = 1, SWEPT_LAUNCH_DIAMOND = 2, SWEPT_LAUNCH_DOWN = 3, SWEPT_LAUNCH_CHAIN = 4, SWEPT_LAUNCH_BAND = 5,
       SWEPT_LAUNCH_RING = 6 };
typedef struct {
    int kind;           /* SWEPT_LAUNCH_*                         */
    int tile_width;     /* W of the entry (0 for CLASSIC)         */
    int64_t offset;     /* tile-grid shift of the (first) launch  */
    int64_t count;      /* see above                              */
} swept_launch_t;

typedef struct {
    int dtype;          /* SWEPT_F32 | SWEPT_F64                                               */
    double alpha;       /* heat: thermal diffusivity (Fo = alpha dt / dx^2)       */
    double gamma;       /* Euler: ratio of specific heats                                      */
    int max_tile_width; /* upper bound for the tuner's tile-width sweep, 0 = library default   */
    int boundary;       /* SWEPT_BC_PERIODIC (0, default) | SWEPT_BC_INSULATED (heat only)      */
} swept_params_t;

typedef struct {
    int problem, dtype, radius, stages, ncomp;
    int64_t nx;
    int64_t workspace_bytes;     /* device workspace owned by the handle (row R1 / classic's 2nd buffer) */
    int tuned_tile_width;        /* 0 until swept_tune ran                                      */
    int64_t launches_last_call;  /* kernels the last swept_run / naive_run enqueued              */
    int64_t launches_total;      /* kernels enqueued through this handle since creation          */
    int sm_count;                /* multiprocessors of the device the handle lives on            */
    int max_smem_per_block;      /* opt-in shared-memory limit per block (bytes)                 */
    int last_sweep_launch;       /* SWEPT_LAUNCH_* that ran the half-cycles of the last swept_run enqueued outside a
                                    graph (RING, BAND, CHAIN, or DIAMOND for per-half-cycle launches); -1 = none yet  */
    int boundary;                /* SWEPT_BC_*                                                    */
    int tuned_chain;             /* SWEPT_OPT_CHAIN value (1 | 2 | 3) swept_tune measured as fastest for tuned_tile_width
                                    under the default option 3; 0 = not tuned                                        */
    int tuned_blocks_per_sm;     /* resident-blocks cap swept_tune measured as fastest for tuned_tile_width when called with
                                    blocks_per_sm_cap = 0 (0 = none); used while SWEPT_OPT_BLOCKS_PER_SM is 0          */
    int tuned_pack;              /* SWEPT_OPT_PACK value (1 | 2) swept_tune measured as faster for the tuned width and kernel;
                                    0 = not measured (not heat / KS fp32 on the band kernel)                              */
    int tuned_kernel;            /* -1, or SWEPT_KERNEL_SMEM where swept_tune -- under the default options -- measured the
                                    paper-style shared-memory kernels as fastest: swept_run then runs the tuned width on them
                                    (tuned_chain = 0).  Small Euler grids.                                           */
} swept_info_t;

/* Create a solver for `problem` on nx periodic points with spacing dx and timestep dt (the paper's
 * statement of the problem: PAPER.md:48-66).  nx must be a power of two >= 8 (periodic neighbour
 * is `& (nx-1)`).  Computes the scheme constants once on the host in double (Fo,
 * 1-2Fo; 0.25/dx, 1/dx^2, 1/dx^4, dt, dt/2; gamma, gamma-1, dt/dx, dt/2dx -- stored reciprocals
 * instead of divisions), allocates ncomp*nx elements of device workspace on the
 * current device, and returns the handle in *out.  `p` may be NULL (= f64, alpha 1, gamma 1.4).
 * Errors: SWEPT_EINVAL (bad problem/dtype/nx, non-finite or non-positive dx/dt, NULL out),
 * SWEPT_ENOMEM / SWEPT_ECUDA (allocation or device errors). */
int swept_create(swept_handle_t *out, int problem, int64_t nx, double dx, double dt, const swept_params_t *p);

/* Advance the field at d_u by nsteps full timesteps IN PLACE with the swept rule:
 * with L = tile_width/(2h) tiers per half-cycle (L/S timesteps), q = nsteps div (L/S) half-cycles
 * are run as 1 upright triangle (Fig. 5) + (q-1) diamonds on tiles shifted by W/2 each
 * launch + 1 closing inverted triangle; the nsteps mod (L/S) remaining
 * timesteps are run as a truncated closing cycle inside the same launch (ring kernel, the default) or first, on narrower
 * tiles / the classic kernel (the other kernels; the paper can only output every n-th step; reading S3).  Edges are exchanged through d_u itself (even
 * tiers) and the handle's workspace (odd tiers) -- the paper's left/right arrays.
 * tile_width: power of two, >= 4h, <= nx, nx % tile_width == 0, L even; 0 = the tuned width, or, if swept_tune has
 * not run, the library default: the widest legal width <= 256 of the selected kernel family -- on grids narrower than the
 * narrowest register tile (nx < 64 h) the paper-style shared-memory kernels.  Result is bit-identical to naive_run.
 * d_u: device, [ncomp][nx], caller-owned.  Errors: SWEPT_EINVAL (NULL, nsteps < 0, illegal width
 * or a width whose tile does not fit the chosen kernel), SWEPT_ECUDA (launch error). */
int swept_run(swept_handle_t h, void *d_u, int64_t nsteps, int tile_width, void *cuda_stream);

/* Advance the field by nsteps timesteps with the classic decomposition (Fig. 6): one
 * kernel per sub-timestep over all nx points, neighbours through `& (nx-1)`, global memory in and
 * out (heat ping-pongs d_u and the workspace; two-stage schemes write the predictor to the
 * workspace and accumulate the final stage onto d_u, Fig. 6 `+=`).  Same argument rules as swept_run. */
int naive_run(swept_handle_t h, void *d_u, int64_t nsteps, void *cuda_stream);

/* The launch list swept_run(h, d_u, nsteps, tile_width) enqueues for a solver of (problem, dtype, nx) with the given
 * kernel family (SWEPT_KERNEL_*) and chain option: host logic only, needs neither a handle nor a device.  Writes up
 * to `cap` entries to out (may be NULL when cap == 0) and returns the number of entries of the full plan, or a negative
 * error code (illegal width, bad arguments).  Reading S3 of DESIGN.md: with nsteps = q*(L/S) + r, chain = 3 gives the single
 * entry RING(count = q, offset = r) where the ring kernel takes the width (at least 64 iterations per tile, two tiles); else the
 * r remainder timesteps come first -- one UP + DOWN pair on each narrower legal width of r's binary decomposition, then CLASSIC
 * for what is left -- followed by the q half-cycles of width tile_width. */
int64_t swept_plan(int problem, int dtype, int64_t nx, int64_t nsteps, int tile_width, int kernel, int chain,
                   swept_launch_t *out, int64_t cap);

/* Host logic of the streaming-band schedule (SWEPT_OPT_CHAIN = 2), no device needed.  A band is the chain of tiles that
 * stitch onto one another's upper-left edge from half-cycle to half-cycle (Fig. 2b); ntiles = nx / tile_width
 * bands exist.  swept_band_layout: the grid for `ntiles` bands on `sm_count` SMs with `warps_per_block` warps per block (at
 * most one block per SM).  swept_band_owner: the block, the warp of that block, and the position in that warp's band list
 * that own `band`: band n goes to sub-partition slot n mod slots, so every slot carries floor or ceil(ntiles / slots) bands. */
typedef struct {
    int blocks, warps_per_block, slots_per_block, warps_per_slot, slots, max_bands_per_warp, ntiles;
} swept_band_layout_t;
int swept_band_layout(int ntiles, int sm_count, int warps_per_block, swept_band_layout_t *out);
int swept_band_owner(const swept_band_layout_t *layout, int band, int *block, int *warp, int *index);

/* The paper's best-node-size sweep: time swept_run on d_u_scratch (device,
 * [ncomp][nx], contents destroyed) for every legal tile width (and kernel launch shape) up to
 * max_tile_width with at most blocks_per_sm_cap resident blocks per SM (0 = no cap), keep the
 * fastest in the handle and return it in *best_tile_width (may be NULL).  Under the default SWEPT_OPT_CHAIN = 3 each
 * width is timed with the ring kernel, the streaming band kernel and the tile-flag kernel, and swept_run uses the fastest of
 * the three for the tuned width; with blocks_per_sm_cap = 0 the register-resident per-tile kernels are also timed at 4, 3 and 2 blocks
 * of 4 warps per SM (the paper's occupancy trade-off), and the paper-style shared-memory kernels compete as
 * well: where they win (small Euler grids) swept_run runs the tuned width on them (swept_info_t.tuned_kernel).  The returned width is
 * then legal for that family, not necessarily for SWEPT_KERNEL_WAVE.  SYNCHRONISES the stream. */
int swept_tune(swept_handle_t h, void *d_u_scratch, int blocks_per_sm_cap, int *best_tile_width, void *cuda_stream);

/* End-to-end convenience used for the `e2e` measurement: copy h_u (HOST, [ncomp][nx], ideally
 * pinned) to an internal device buffer, swept_run (use_swept != 0) or naive_run on it, copy the
 * result back into h_u, and synchronise the stream. */
int swept_run_host(swept_handle_t h, void *h_u, int64_t nsteps, int tile_width, int use_swept, void *cuda_stream);

/* The swept rule without a handle and without any allocation -- for callers that cannot call cudaMalloc.
 *
 * Who that is: a host program that gave the whole GPU to its own pool (a framework's caching allocator, a simulation code's
 * arena, a fixed per-tenant budget), where a cudaMalloc from inside a library fails or eats into somebody else's share; a
 * time-critical loop, where cudaMalloc / cudaFree stall the device for every stream; and code that runs where the CUDA
 * runtime does not accept allocation calls at all.  swept_create needs three allocations (the odd-tier edge row R1, the flag
 * area of the launch-free kernels, a pinned word), so none of these callers can have a handle.
 *
 * swept_run_static advances the caller's field d_u (DEVICE, [ncomp][nx], 16-byte aligned, caller-owned, updated in place) by
 * nsteps timesteps exactly as swept_run does with SWEPT_OPT_KERNEL = SWEPT_KERNEL_WAVE and SWEPT_OPT_CHAIN = 0: the
 * register-resident tile kernels, one launch per half-cycle -- upright triangle, diamonds on tiles
 * shifted by W/2, closing inverted triangle -- with the nsteps mod (L/S) remaining timesteps first, on narrower tiles and the
 * classic kernel (reading S3).  The result is bit-identical to swept_run and naive_run.  The odd-tier edges (the
 * paper's left / right arrays), for which a handle owns a workspace, go through a fixed array of
 * SWEPT_STATIC_SCRATCH_BYTES that is part of the library image: every GPU that loads the library holds these bytes until
 * the process ends, whether or not this function is ever called.
 *
 *   problem, nx, dx, dt, p   as for swept_create (p may be NULL = f64, alpha 1, gamma 1.4); periodic domains only
 *   tile_width               as for swept_run with the WAVE kernels; 0 = the widest legal width <= 256
 *   cuda_stream              the work is only enqueued, as by swept_run
 *
 * Limit: ncomp * nx * sizeof(dtype) <= SWEPT_STATIC_SCRATCH_BYTES (heat / KS: nx <= 2^20 in fp64, 2^21 in fp32; Euler:
 * nx <= 2^18 / 2^19); a larger field is refused with SWEPT_EINVAL before anything is enqueued.  Other errors as for swept_run.
 * The call makes no cudaMalloc, cudaFree or other allocating call, creates no stream, event or graph, and never synchronises.
 *
 * First call on a device: the library looks up the device address of the array (cudaGetSymbolAddress -- in host code the
 * array's own name is not a device pointer) and raises the shared-memory limits of the kernels for (problem, dtype); the
 * device that is current at the call is the one set up and used.  Make that first call for each (device, problem, dtype)
 * outside any stream capture.
 *
 * All calls on one device share the one array, and it keeps what the last call left there.  Nothing in it has to start
 * at zero: every phase writes each odd-tier edge value before a later phase of the same call reads it, so old contents are
 * never read.  But two calls whose kernels can overlap on the GPU (different streams, no ordering between them) race on the
 * array and corrupt each other's edges: order them, or give all but one a handle. */
#define SWEPT_STATIC_SCRATCH_BYTES (8 << 20)
int swept_run_static(int problem, int64_t nx, double dx, double dt, const swept_params_t *p, void *d_u, int64_t nsteps,
                     int tile_width, void *cuda_stream);

/* Set a SWEPT_OPT_* option.  SWEPT_EINVAL for unknown keys / values. */
int swept_set_option(swept_handle_t h, int key, int value);

/* Stencil radius h per sub-timestep, sub-timesteps S per timestep and fields per point of `problem` (any pointer may be
 * NULL): a half-cycle of tile width W advances W / (2 h S) timesteps.  Host logic, no device needed. */
int swept_problem_info(int problem, int *radius, int *stages, int *ncomp);

/* Fill *info (caller-owned). */
int swept_get_info(swept_handle_t h, swept_info_t *info);

/* 1 if swept_run accepts tile_width on this handle -- for the kernel family it would run that width on: the selected one, or, for the
 * tuned width, the family swept_tune chose (swept_info_t.tuned_kernel) -- else 0 (reason in swept_last_error). */
int swept_tile_width_ok(swept_handle_t h, int tile_width);

/* Measure the plain-ALU peak the swept kernels are bound by: a dependent-free FMA chain of the
 * given dtype on every SM; returns warp-level FP instructions x 32 lanes per second (thread-level
 * FP instr/s) in *instr_per_s and the elapsed milliseconds of the timed launch in *ms (may be
 * NULL).  SYNCHRONISES.  Used by bench.py for the "alu" roofline denominator. */
int swept_measure_alu_peak(int dtype, double *instr_per_s, double *ms, void *cuda_stream);

/* Measure the shared-memory read peak the paper-style kernels are bound by: conflict-free 16-byte loads by every thread of
 * every SM; returns bytes per second in *bytes_per_s (nominal: 128 B per clock per SM) and the milliseconds of the timed launch
 * in *ms (may be NULL).  SYNCHRONISES. */
int swept_measure_smem_peak(double *bytes_per_s, double *ms, void *cuda_stream);

/* Latency probes, in SM clock cycles per operation, one warp alone on its SM (cycles[0..4], a host array of 5 doubles):
 * [0] a dependent DFMA; [1] the heat update's chain DADD -> DFMA; [2] a dependent 64-bit warp shuffle; [3] a lock-step tier
 * (two 64-bit shuffles -> DADD -> DFMA); [4] a tier exchanged through shared memory with one block barrier, 256 threads.
 * They bound what any decomposition of a small grid can reach.  SYNCHRONISES. */
int swept_measure_latencies(double *cycles, void *cuda_stream);

/* Wait (on the host) for everything enqueued through this handle and report whether a bounded wait of a launch-free sweep gave up
 * since the last report: SWEPT_ECUDA once (the fields those sweeps ran on are invalid; the handle is usable again), else SWEPT_OK. */
int swept_check(swept_handle_t h);

/* Free the workspace and the handle.  The caller must have synchronised every stream it used. */
int swept_destroy(swept_handle_t h);

/* Message of the last error on this thread ("" if none).  Never NULL. */
const char *swept_last_error(void);

/* Library version string (static storage). */
const char *swept_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SWEPT1D_H */
