// api.cu -- the C ABI of libswept1d.so (include/swept1d.h): handle, host driver,
// tuner (row A8), options.  No CPU fallback: every compute entry point needs a CUDA device.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>

#include "internal.h"
#include "stencils.cuh"

using namespace swept;

struct swept_ctx {
    int problem, dtype, H, S, NC, bc;
    int64_t nx;
    double dx, dt, alpha, gamma;
    ConstBlock cb;
    void *work;            // row R1 of the staircase / the classic path's second buffer: NC*nx elements
    size_t field_bytes;    // NC*nx*sizeof(T)
    void *host_stage;      // device buffer for swept_run_host (allocated on first use)
    int device, sm_count, max_smem;
    int kernel, chain, naive_graph, naive_share, swept_graph, blocks_per_sm, warps_per_block, pack, tuned_pack;
    void *sync_base;       // SYNC_HEADER bytes (word 0: the abort word of the bounded waits, swept_wave.cuh) + the sync area
    void *sync;            // sync area = sync_base + SYNC_HEADER; chain kernel: work counter (8 bytes) + done[] flags; band kernel: prog[]
    unsigned *abort_seen;  // pinned host copy of the abort word, refreshed by an async copy behind every launch-free launch
    cudaEvent_t busy;      // recorded behind the work of every call; the next call's stream waits on it (calls on one handle
                           // from several streams are serialised on the device instead of corrupting the shared scratch)
    int max_tile_width, tuned_tile_width, tuned_chain, tuned_cap, tuned_kernel, last_sweep_launch;   // tuned_kernel: -1 = the option's family   // tuned_chain: 1 | 2 for tuned_tile_width, 0 = not tuned
    int64_t launches_last, launches_total;
    // cached CUDA graphs (one per path; rebuilt when the key changes)
    cudaGraphExec_t ngraph;  void *ngraph_u;  int64_t ngraph_steps, ngraph_launches;
    cudaGraphExec_t sgraph;  void *sgraph_u;  int64_t sgraph_steps;  int sgraph_W, sgraph_kernel, sgraph_chain, sgraph_cap, sgraph_wpb;
    int64_t sgraph_launches;
};

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...) __attribute__((format(printf, 2, 3)));
static int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
static int fail_cuda(cudaError_t e, const char *what) {
    cudaGetLastError();   // clear the sticky-less error state
    return fail(SWEPT_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

int swept::swept_fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

extern "C" const char *swept_last_error(void) { return g_err; }
extern "C" const char *swept_version(void) { return "swept1d-b200 0.1 (sm_100a)"; }

static bool is_pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }

// ---- row A0: scheme constants, computed once on the host in double, then cast to the run dtype ------------
template <class T> static void fill_consts(swept_ctx *h) {
    memset(h->cb.bytes, 0, sizeof h->cb.bytes);
    if (h->problem == SWEPT_HEAT) {
        typename Heat<T>::Consts c;
        const double Fo = h->alpha * h->dt / (h->dx * h->dx);
        c.Fo = (T)Fo;
        c.c0 = (T)(1.0 - 2.0 * Fo);
        memcpy(h->cb.bytes, &c, sizeof c);
    } else if (h->problem == SWEPT_KS) {
        typename KS<T>::Consts c;
        const double c2 = 1.0 / (h->dx * h->dx);                        // stored reciprocals
        c.c1 = (T)(0.25 / h->dx);
        c.c2 = (T)c2;
        c.c4 = (T)(c2 * c2);
        c.dt = (T)h->dt;
        c.dth = (T)(0.5 * h->dt);
        memcpy(h->cb.bytes, &c, sizeof c);
    } else {
        typename Euler<T>::Consts c;
        const double lam = h->dt / h->dx;
        c.gamma = (T)h->gamma;
        c.gm1 = (T)(h->gamma - 1.0);
        c.lam = (T)lam;
        c.lamh = (T)(0.5 * lam);
        memcpy(h->cb.bytes, &c, sizeof c);
    }
}

extern "C" int swept_create(swept_handle_t *out, int problem, int64_t nx, double dx, double dt, const swept_params_t *p) {
    g_err[0] = 0;
    if (!out) return fail(SWEPT_EINVAL, "swept_create: out is NULL");
    *out = nullptr;
    if (problem != SWEPT_HEAT && problem != SWEPT_KS && problem != SWEPT_EULER) return fail(SWEPT_EINVAL, "swept_create: unknown problem %d", problem);
    const int dtype = p ? p->dtype : SWEPT_F64;
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return fail(SWEPT_EINVAL, "swept_create: unknown dtype %d", dtype);
    if (!is_pow2(nx) || nx < 8) return fail(SWEPT_EINVAL, "swept_create: nx=%lld must be a power of two >= 8 (periodic index is & (nx-1))", (long long)nx);
    if (nx > ((int64_t)1 << 40)) return fail(SWEPT_EINVAL, "swept_create: nx too large");
    if (!isfinite(dx) || !isfinite(dt) || dx <= 0.0 || dt <= 0.0) return fail(SWEPT_EINVAL, "swept_create: dx and dt must be finite and positive");
    const double alpha = p ? p->alpha : 1.0, gamma = p ? p->gamma : 1.4;
    if (problem == SWEPT_HEAT && !(isfinite(alpha) && alpha > 0.0)) return fail(SWEPT_EINVAL, "swept_create: alpha must be finite and positive");
    if (problem == SWEPT_EULER && !(isfinite(gamma) && gamma > 1.0)) return fail(SWEPT_EINVAL, "swept_create: gamma must be finite and > 1");
    if (p && p->max_tile_width < 0) return fail(SWEPT_EINVAL, "swept_create: max_tile_width < 0");
    const int bc = p ? p->boundary : SWEPT_BC_PERIODIC;
    if (bc != SWEPT_BC_PERIODIC && bc != SWEPT_BC_INSULATED) return fail(SWEPT_EINVAL, "swept_create: unknown boundary %d", bc);
    if (bc == SWEPT_BC_INSULATED && problem != SWEPT_HEAT)
        return fail(SWEPT_EINVAL, "swept_create: insulated ends exist for the heat problem only (the paper's KS problem is periodic, PAPER.md:66)");

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "swept_create: no CUDA device (this library has no CPU fallback)");
    swept_ctx *h = new (std::nothrow) swept_ctx();
    if (!h) return fail(SWEPT_ENOMEM, "swept_create: out of host memory");
    memset(h, 0, sizeof *h);
    h->problem = problem; h->dtype = dtype;
    h->H = radius_of(problem); h->S = stages_of(problem); h->NC = ncomp_of(problem);
    h->nx = nx; h->dx = dx; h->dt = dt; h->alpha = alpha; h->gamma = gamma;
    h->bc = bc;
    h->device = dev;
    h->kernel = SWEPT_KERNEL_WAVE;
    h->chain = 3;
    h->last_sweep_launch = -1;
    h->tuned_kernel = -1;
    h->warps_per_block = 4;
    h->max_tile_width = p ? p->max_tile_width : 0;
    if (dtype == SWEPT_F64) fill_consts<double>(h); else fill_consts<float>(h);
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&h->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    h->field_bytes = (size_t)h->NC * (size_t)nx * elem_size(dtype);
    e = cudaMalloc(&h->work, h->field_bytes);
    if (e != cudaSuccess) {
        delete h;
        cudaGetLastError();
        return fail(e == cudaErrorMemoryAllocation ? SWEPT_ENOMEM : SWEPT_ECUDA, "swept_create: cudaMalloc workspace: %s", cudaGetErrorString(e));
    }
    e = cudaMalloc(&h->sync_base, SYNC_HEADER + 8 + sizeof(unsigned) * (size_t)(nx / 8 + 2));
    if (e != cudaSuccess) {
        cudaFree(h->work);
        delete h;
        cudaGetLastError();
        return fail(e == cudaErrorMemoryAllocation ? SWEPT_ENOMEM : SWEPT_ECUDA, "swept_create: cudaMalloc flags: %s", cudaGetErrorString(e));
    }
    h->sync = (char *)h->sync_base + SYNC_HEADER;
    e = cudaMemset(h->sync_base, 0, SYNC_HEADER);
    if (e == cudaSuccess) e = cudaHostAlloc((void **)&h->abort_seen, sizeof(unsigned), cudaHostAllocDefault);
    if (e == cudaSuccess) { *h->abort_seen = 0; e = cudaEventCreateWithFlags(&h->busy, cudaEventDisableTiming); }
    if (e == cudaSuccess) e = swept_smem_prepare(problem, dtype, (size_t)h->max_smem);
    if (e == cudaSuccess) e = swept_wave_prepare(problem, dtype);
    if (e != cudaSuccess) {
        cudaFree(h->work); cudaFree(h->sync_base);
        if (h->abort_seen) cudaFreeHost(h->abort_seen);
        if (h->busy) cudaEventDestroy(h->busy);
        delete h;
        return fail_cuda(e, "swept_create: scratch / kernel attribute setup");
    }
    *out = h;
    return SWEPT_OK;
}

static void drop_graphs(swept_ctx *h) {
    if (h->ngraph) { cudaGraphExecDestroy(h->ngraph); h->ngraph = nullptr; }
    if (h->sgraph) { cudaGraphExecDestroy(h->sgraph); h->sgraph = nullptr; }
}

extern "C" int swept_destroy(swept_handle_t h) {
    if (!h) return fail(SWEPT_EINVAL, "swept_destroy: NULL handle");
    drop_graphs(h);
    if (h->work) cudaFree(h->work);
    if (h->sync_base) cudaFree(h->sync_base);
    if (h->abort_seen) cudaFreeHost(h->abort_seen);
    if (h->busy) cudaEventDestroy(h->busy);
    if (h->host_stage) cudaFree(h->host_stage);
    delete h;
    return SWEPT_OK;
}

// ---- legality of a tile width (SURVEY.md section 8(a) "Legal tile widths") ------------------------------------
static const char *width_problem(int problem, int dtype, int64_t nx, int W, int kernel, int max_smem, char *buf, size_t nbuf) {
    const int H = radius_of(problem);
    if (W <= 0 || !is_pow2(W)) return "tile width must be a power of two";
    if (W < 4 * H) return "tile width must be >= 4h (L = W/(2h) even)";
    if ((int64_t)W > nx) return "tile width exceeds nx";
    if (kernel == SWEPT_KERNEL_SMEM) {
        const size_t need = swept_smem_bytes(problem, dtype, W);
        if (need > (size_t)max_smem) {
            snprintf(buf, nbuf, "tile needs %zu B of shared memory, limit %d B", need, max_smem);
            return buf;
        }
        return nullptr;
    }
    if (kernel == SWEPT_KERNEL_WAVE) return swept_wave_supports(problem, dtype, W) ? nullptr : "tile width not supported by the WAVE kernels for this problem/dtype";
    return "unknown kernel";
}

static int check_width(const swept_ctx *h, int W, int kernel, bool set_err) {
    char buf[160];
    if (h->bc && kernel == SWEPT_KERNEL_SMEM) {
        if (set_err) fail(SWEPT_EINVAL, "tile_width %d: insulated ends are implemented by the WAVE kernels only", W);
        return 0;
    }
    const char *why = width_problem(h->problem, h->dtype, h->nx, W, kernel, h->max_smem, buf, sizeof buf);
    if (why) {
        if (set_err) fail(SWEPT_EINVAL, "tile_width %d: %s", W, why);
        return 0;
    }
    return 1;
}

static int tuned_family(const swept_ctx *h, int W);

extern "C" int swept_tile_width_ok(swept_handle_t h, int tile_width) {
    if (!h) { fail(SWEPT_EINVAL, "swept_tile_width_ok: NULL handle"); return 0; }
    return check_width(h, tile_width, tuned_family(h, tile_width), true);    // the family swept_run would run this width on
}

// The kernel family swept_run uses for width W: the option's, except that under the default options (register kernels, launch-free
// sweep chosen by the tuner) the tuned width runs on the paper-style shared-memory kernels where swept_tune measured them faster
// (Euler on grids that give a lane-per-8-cells kernel too few warps: nx <= 2^16).
static int tuned_family(const swept_ctx *h, int W) {
    if (h->kernel == SWEPT_KERNEL_WAVE && h->chain == 3 && h->tuned_kernel >= 0 && W == h->tuned_tile_width) return h->tuned_kernel;
    return h->kernel;
}

// The width swept_run uses for tile_width = 0: the tuned one, else the largest legal width not above 256 (WAVE) / 512 (SMEM)
// and nx.  Grids too small for the narrowest register tile (32 lanes x 2h points) fall back to the paper-style shared-memory
// kernels, which take any power of two >= 4h: *kernel is the family to run.
static int default_width(const swept_ctx *h, int *kernel) {
    *kernel = h->kernel;
    if (h->tuned_tile_width) { *kernel = tuned_family(h, h->tuned_tile_width); return h->tuned_tile_width; }
    for (int W = h->kernel == SWEPT_KERNEL_WAVE ? 256 : 512; W >= 4 * h->H; W >>= 1)
        if (check_width(h, W, h->kernel, false)) return W;
    if (h->kernel == SWEPT_KERNEL_WAVE && !h->bc) {
        *kernel = SWEPT_KERNEL_SMEM;
        for (int W = 512; W >= 4 * h->H; W >>= 1)
            if (check_width(h, W, SWEPT_KERNEL_SMEM, false)) return W;
    }
    return 0;
}

// ---- entry / exit of every call that enqueues work on a handle ---------------------------------------------------
// The handle's device (the kernels' shared-memory opt-ins and the scratch are per device) must be current; a wait that gave up
// in an earlier launch-free sweep is reported once; the stream first waits for the handle's previous call (any stream).
// A bounded wait gave up (the pinned copy of the abort word is set): wait for everything the handle enqueued, clear the word on
// both sides so that the handle is usable again, and report once.
static int report_abort(swept_ctx *h, const char *who) {
    cudaEventSynchronize(h->busy);
    *h->abort_seen = 0;
    cudaMemset(h->sync_base, 0, SYNC_HEADER);
    return fail(SWEPT_ECUDA, "%s: an earlier launch-free sweep on this handle gave up waiting for a tile that never completed "
                             "(was the handle used from two host threads at once?); the field it ran on is invalid", who);
}

static int handle_enter(swept_ctx *h, cudaStream_t st, const char *who) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, who);
    if (dev != h->device) return fail(SWEPT_EINVAL, "%s: the handle was created on device %d but device %d is current", who, h->device, dev);
    if (*(volatile unsigned *)h->abort_seen) return report_abort(h, who);
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
    if (cs == cudaStreamCaptureStatusNone) {
        e = cudaStreamWaitEvent(st, h->busy, 0);
        if (e != cudaSuccess) return fail_cuda(e, who);
    }
    return SWEPT_OK;
}
static void handle_leave(swept_ctx *h, cudaStream_t st) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); return; }
    if (cs != cudaStreamCaptureStatusNone) return;     // the caller's own capture orders its nodes
    cudaMemcpyAsync(h->abort_seen, h->sync_base, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
    cudaEventRecord(h->busy, st);
}

// Every exit path of a call that passed handle_enter records the busy event, also the error returns: work that was enqueued before
// the error is then still ahead of whatever the next call (on any stream) enqueues.
struct LeaveGuard {
    swept_ctx *h;
    cudaStream_t st;
    ~LeaveGuard() { handle_leave(h, st); }
};

// ---- classic path (row A2) -----------------------------------------------------------------------------------
// Enqueue nsteps classic timesteps.  Heat ping-pongs u and work (and copies back after an odd count); two-stage
// schemes write the predictor to work and accumulate the final stage onto u (Fig. 6).
static cudaError_t enqueue_classic(swept_ctx *h, void *d_u, int64_t nsteps, cudaStream_t st, int64_t *launches) {
    cudaError_t e = cudaSuccess;
    if (h->S == 1) {
        void *a = d_u, *b = h->work;
        for (int64_t m = 0; m < nsteps; ++m) {
            e = launch_classic_stage(h->problem, h->dtype, 1, a, a, b, h->nx, h->cb, h->bc, h->naive_share, st);
            if (e != cudaSuccess) return e;
            void *t = a; a = b; b = t;
            ++*launches;
        }
        if (a != d_u) {
            e = cudaMemcpyAsync(d_u, a, h->field_bytes, cudaMemcpyDeviceToDevice, st);   // a copy, not a kernel: not counted
        }
    } else {
        for (int64_t m = 0; m < nsteps; ++m) {
            e = launch_classic_stage(h->problem, h->dtype, 1, d_u, d_u, h->work, h->nx, h->cb, h->bc, h->naive_share, st);
            if (e != cudaSuccess) return e;
            e = launch_classic_stage(h->problem, h->dtype, 0, h->work, d_u, d_u, h->nx, h->cb, h->bc, h->naive_share, st);
            if (e != cudaSuccess) return e;
            *launches += 2;
        }
    }
    return e;
}

static int run_args_ok(swept_ctx *h, void *d_u, int64_t nsteps, const char *who) {
    if (!h) return fail(SWEPT_EINVAL, "%s: NULL handle", who);
    if (!d_u) return fail(SWEPT_EINVAL, "%s: d_u is NULL", who);
    if (nsteps < 0) return fail(SWEPT_EINVAL, "%s: nsteps < 0", who);
    if (((uintptr_t)d_u & 15) != 0) return fail(SWEPT_EINVAL, "%s: d_u must be 16-byte aligned", who);
    return SWEPT_OK;
}

// Replay `steps` of a path through a cached CUDA graph (captured on first use with the same key).
template <class Enqueue>
static int run_graphed(cudaGraphExec_t *exec, bool reuse, cudaStream_t st, int64_t *launches, Enqueue &&enq, const char *who) {
    cudaError_t e;
    if (!reuse) {
        if (*exec) { cudaGraphExecDestroy(*exec); *exec = nullptr; }
        cudaStream_t cap;
        e = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking);
        if (e != cudaSuccess) return fail_cuda(e, who);
        e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
        if (e != cudaSuccess) { cudaStreamDestroy(cap); return fail_cuda(e, who); }
        *launches = 0;
        cudaError_t el = enq(cap, launches);
        cudaGraph_t g = nullptr;
        e = cudaStreamEndCapture(cap, &g);
        cudaStreamDestroy(cap);
        if (el != cudaSuccess) { if (g) cudaGraphDestroy(g); return fail_cuda(el, who); }
        if (e != cudaSuccess) return fail_cuda(e, who);
        e = cudaGraphInstantiate(exec, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) { *exec = nullptr; return fail_cuda(e, who); }
    }
    e = cudaGraphLaunch(*exec, st);
    if (e != cudaSuccess) return fail_cuda(e, who);
    return SWEPT_OK;
}

extern "C" int naive_run(swept_handle_t h, void *d_u, int64_t nsteps, void *cuda_stream) {
    int rc = run_args_ok(h, d_u, nsteps, "naive_run");
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = handle_enter(h, st, "naive_run"))) return rc;
    LeaveGuard leave{h, st};
    int64_t launches = 0;
    if (h->naive_graph && nsteps >= 2) {
        // a graph of `chunk` timesteps (even, so heat's ping-pong ends in d_u), replayed; the rest as plain launches
        int64_t chunk = nsteps < 1000 ? nsteps : 1000;
        chunk -= chunk & 1;
        const bool reuse = h->ngraph && h->ngraph_u == d_u && h->ngraph_steps == chunk;
        const int64_t reps = nsteps / chunk;
        for (int64_t i = 0; i < reps; ++i) {
            int64_t l = 0;
            rc = run_graphed(&h->ngraph, reuse || i > 0, st, &l, [&](cudaStream_t s, int64_t *n) { return enqueue_classic(h, d_u, chunk, s, n); }, "naive_run(graph)");
            if (rc) return rc;
            if (!reuse && i == 0) { h->ngraph_u = d_u; h->ngraph_steps = chunk; h->ngraph_launches = l; }
            launches += h->ngraph_launches;
        }
        cudaError_t e = enqueue_classic(h, d_u, nsteps % chunk, st, &launches);
        if (e != cudaSuccess) return fail_cuda(e, "naive_run");
    } else {
        cudaError_t e = enqueue_classic(h, d_u, nsteps, st, &launches);
        if (e != cudaSuccess) return fail_cuda(e, "naive_run");
    }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

// ---- swept path (row A7) ---------------------------------------------------------------------------------------
// The host driver is data: build_plan() turns (nsteps, W) into the launch list, enqueue_plan() executes it.
// nsteps = q*(L/S) + r.  The r remaining timesteps run first (reading S3): on successively narrower legal tiles (each
// one half-cycle: one upright + one closing triangle), and what no tile width divides on the classic kernel.  Then q
// half-cycles of width W: 1 upright triangle + (q-1) diamonds on tiles shifted by W/2 each launch + 1 closing inverted
// triangle; on a periodic domain either alignment may write out (reading S4).  With `chain` (WAVE
// kernels) the q half-cycles are ONE launch of the flag-ordered persistent kernel.
static int64_t build_plan(int problem, int dtype, int64_t nx, int64_t nsteps, int W, int kernel, int chain, int bc, int max_smem,
                          swept_launch_t *out, int64_t cap) {
    const int H = radius_of(problem), S = stages_of(problem);
    const int per = 2 * H * S;   // W / per = timesteps per half-cycle
    int64_t n = 0;
    auto push = [&](int kind, int w, int64_t offset, int64_t count) {
        if (out && n < cap) { out[n].kind = kind; out[n].tile_width = w; out[n].offset = offset; out[n].count = count; }
        ++n;
    };
    auto half_cycles = [&](int w, int64_t q, bool chained) {
        if (q <= 0) return;
        if (chained) { push(chain >= 2 ? SWEPT_LAUNCH_BAND : SWEPT_LAUNCH_CHAIN, w, 0, q); return; }
        push(SWEPT_LAUNCH_UP, w, 0, 1);
        if (q > 1) push(SWEPT_LAUNCH_DIAMOND, w, w / 2, q - 1);   // offsets W/2, 0, W/2, ...
        push(SWEPT_LAUNCH_DOWN, w, (q & 1) ? w / 2 : 0, 1);
    };
    const int64_t sph = W / per;
    const int64_t q = nsteps / sph;
    int64_t r = nsteps % sph;
    // ring kernel (chain = 3) and band kernel (chain = 2): the q half-cycles AND the remainder (as a truncated closing cycle) in one
    // launch; entry.offset = r.  (Both need tiles of at least 64 iterations and two tiles.)
    if (chain >= 2 && kernel == SWEPT_KERNEL_WAVE && !bc && nsteps > 0 && swept_ring_supports(problem, W) && nx / W >= 2) {
        push(chain == 3 ? SWEPT_LAUNCH_RING : SWEPT_LAUNCH_BAND, W, r, q);
        return n;
    }
    char buf[160];
    for (int w = W / 2; w >= 4 * H && r > 0; w >>= 1) {
        const int64_t s = w / per;
        if (s >= 1 && r >= s && !width_problem(problem, dtype, nx, w, kernel, max_smem, buf, sizeof buf)) {
            half_cycles(w, 1, false);
            r -= s;
        }
    }
    if (r > 0) push(SWEPT_LAUNCH_CLASSIC, 0, 0, r);
    half_cycles(W, q, chain && kernel == SWEPT_KERNEL_WAVE);
    return n;
}

extern "C" int64_t swept_plan(int problem, int dtype, int64_t nx, int64_t nsteps, int tile_width, int kernel, int chain,
                              swept_launch_t *out, int64_t cap) {
    if (problem != SWEPT_HEAT && problem != SWEPT_KS && problem != SWEPT_EULER) return fail(SWEPT_EINVAL, "swept_plan: unknown problem %d", problem);
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return fail(SWEPT_EINVAL, "swept_plan: unknown dtype %d", dtype);
    if (!is_pow2(nx) || nx < 8) return fail(SWEPT_EINVAL, "swept_plan: nx=%lld must be a power of two >= 8", (long long)nx);
    if (nsteps < 0) return fail(SWEPT_EINVAL, "swept_plan: nsteps < 0");
    if (cap < 0 || (cap > 0 && !out)) return fail(SWEPT_EINVAL, "swept_plan: bad output buffer");
    char buf[160];
    const char *why = width_problem(problem, dtype, nx, tile_width, kernel, SWEPT_SMEM_LIMIT_B200, buf, sizeof buf);
    if (why) return fail(SWEPT_EINVAL, "tile_width %d: %s", tile_width, why);
    if (chain < 0 || chain > 3) return fail(SWEPT_EINVAL, "swept_plan: chain takes 0..3");
    return build_plan(problem, dtype, nx, nsteps, tile_width, kernel, chain, SWEPT_BC_PERIODIC, SWEPT_SMEM_LIMIT_B200, out, cap);
}

static int effective_cap(const swept_ctx *h, int W);
static int effective_pack(const swept_ctx *h, int W);

static cudaError_t launch_phase(swept_ctx *h, int kernel, int mode, void *d_u, int W, int64_t offset, cudaStream_t st) {
    if (kernel == SWEPT_KERNEL_SMEM) return launch_swept_smem(h->problem, h->dtype, mode, d_u, h->work, h->nx, W, offset, h->cb, st);
    return launch_swept_wave(h->problem, h->dtype, mode, d_u, h->work, h->nx, W, offset, h->cb, h->warps_per_block, effective_cap(h, W), h->bc, st);
}

// The launch-free variant swept_run uses for width W: the option, except that with the default (2 = streaming bands) the
// tuner's measured choice between the band and the tile-flag kernel is honoured for the width it tuned.
static int effective_chain(const swept_ctx *h, int W) {
    if (h->chain == 3 && h->tuned_chain && W == h->tuned_tile_width) return h->tuned_chain;
    return h->chain;
}

// Resident-blocks cap for width W: the option if set, else the cap the tuner measured as fastest for the tuned width.
// Packed pairs of bands (heat fp32, band kernel): the option if set (1 = off, 2 = on); with 0 (auto) the tuner's measurement for the
// tuned width, else on where every SM gets at least sixteen bands (enough pairs to fill its warps).
static int effective_pack(const swept_ctx *h, int W) {
    if (h->problem == SWEPT_EULER || h->dtype != SWEPT_F32) return 0;
    if (h->pack) return h->pack == 2;
    if (h->tuned_pack && W == h->tuned_tile_width) return h->tuned_pack == 2;
    if (h->problem == SWEPT_KS) return 0;                            // KS: packed pairs only on request or by the tuner's measurement
    return h->nx / W >= (int64_t)16 * h->sm_count;
}

static int effective_cap(const swept_ctx *h, int W) {
    if (h->blocks_per_sm == 0 && h->tuned_cap && W == h->tuned_tile_width) return h->tuned_cap;
    return h->blocks_per_sm;
}

static cudaError_t enqueue_swept(swept_ctx *h, int kernel, void *d_u, int64_t nsteps, int W, cudaStream_t st, int64_t *launches, int chain_override = -1) {
    swept_launch_t plan[64];   // at most 3 entries per narrower width + 1 classic + 3
    const int chain = chain_override >= 0 ? chain_override : effective_chain(h, W);
    const int64_t n = build_plan(h->problem, h->dtype, h->nx, nsteps, W, kernel, chain, h->bc, h->max_smem, plan, 64);
    if (n > 64) return cudaErrorInvalidValue;
    cudaError_t e = cudaSuccess;
    for (int64_t i = 0; i < n && e == cudaSuccess; ++i) {
        const swept_launch_t &L = plan[i];
        switch (L.kind) {
            case SWEPT_LAUNCH_CLASSIC: e = enqueue_classic(h, d_u, L.count, st, launches); break;
            case SWEPT_LAUNCH_UP: e = launch_phase(h, kernel, MODE_UP, d_u, L.tile_width, L.offset, st); ++*launches; break;
            case SWEPT_LAUNCH_DOWN: e = launch_phase(h, kernel, MODE_DOWN, d_u, L.tile_width, L.offset, st); ++*launches; break;
            case SWEPT_LAUNCH_DIAMOND:
                h->last_sweep_launch = SWEPT_LAUNCH_DIAMOND;
                for (int64_t k = 0; k < L.count && e == cudaSuccess; ++k) {
                    const int64_t off = (k & 1) ? (L.offset ? 0 : L.tile_width / 2) : L.offset;
                    e = launch_phase(h, kernel, MODE_DIAMOND, d_u, L.tile_width, off, st);
                    ++*launches;
                }
                break;
            case SWEPT_LAUNCH_RING:
                e = launch_swept_ring(h->problem, h->dtype, d_u, h->work, h->nx, L.tile_width, L.count, (int)(L.offset * h->S), h->sync, h->cb, h->sm_count, h->max_smem,
                                      4 * effective_cap(h, L.tile_width), st);
                if (e != cudaErrorNotSupported && e != cudaErrorCooperativeLaunchTooLarge) { ++*launches; h->last_sweep_launch = SWEPT_LAUNCH_RING; break; }
                cudaGetLastError();
                // the ring schedule does not fit this device / size: the same timesteps as remainder launches + band / tile-flag kernel
                return enqueue_swept(h, kernel, d_u, nsteps, W, st, launches, 2);
            case SWEPT_LAUNCH_BAND:
                // bands wrap around the periodic domain; a rod with insulated ends runs on the tile-flag kernel
                e = h->bc ? cudaErrorNotSupported
                          : launch_swept_band(h->problem, h->dtype, d_u, h->work, h->nx, L.tile_width, L.count, (int)(L.offset * h->S), h->sync, h->cb, h->sm_count, h->max_smem, 4 * effective_cap(h, L.tile_width), effective_pack(h, L.tile_width), st);
                if (e != cudaErrorNotSupported && e != cudaErrorCooperativeLaunchTooLarge) { ++*launches; h->last_sweep_launch = SWEPT_LAUNCH_BAND; break; }
                cudaGetLastError();
                // the band schedule does not fit this device / size: with a truncated closing cycle, the same timesteps as remainder
                // launches + the tile-flag kernel; without, the same half-cycles through the tile-flag kernel
                if (L.offset > 0 || L.count == 0) return enqueue_swept(h, kernel, d_u, nsteps, W, st, launches, 1);
                /* fall through */
            case SWEPT_LAUNCH_CHAIN:
                e = launch_swept_chain(h->problem, h->dtype, d_u, h->work, h->nx, L.tile_width, L.count, h->sync, h->cb, h->warps_per_block,
                                       effective_cap(h, L.tile_width), h->sm_count, h->bc, st);
                h->last_sweep_launch = SWEPT_LAUNCH_CHAIN;
                ++*launches;
                break;
            default: e = cudaErrorInvalidValue;
        }
    }
    return e;
}

extern "C" int swept_run(swept_handle_t h, void *d_u, int64_t nsteps, int tile_width, void *cuda_stream) {
    int rc = run_args_ok(h, d_u, nsteps, "swept_run");
    if (rc) return rc;
    int W = tile_width, kernel = h->kernel;
    if (W == 0) {
        W = default_width(h, &kernel);
        if (W == 0) return fail(SWEPT_EINVAL, "swept_run: no legal tile width for nx=%lld with the selected kernel", (long long)h->nx);
    } else {
        kernel = tuned_family(h, W);                      // the tuned width runs on the family the tuner measured as fastest
        if (!check_width(h, W, kernel, true)) return SWEPT_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = handle_enter(h, st, "swept_run"))) return rc;
    LeaveGuard leave{h, st};
    int64_t launches = 0;
    if (h->swept_graph && nsteps > 0) {
        const int chain = effective_chain(h, W), cap = effective_cap(h, W);
        const bool reuse = h->sgraph && h->sgraph_u == d_u && h->sgraph_steps == nsteps && h->sgraph_W == W && h->sgraph_kernel == kernel && h->sgraph_chain == chain &&
                           h->sgraph_cap == cap && h->sgraph_wpb == h->warps_per_block;
        int64_t l = 0;
        rc = run_graphed(&h->sgraph, reuse, st, &l, [&](cudaStream_t s, int64_t *n) { return enqueue_swept(h, kernel, d_u, nsteps, W, s, n); }, "swept_run(graph)");
        if (rc) return rc;
        if (!reuse) { h->sgraph_u = d_u; h->sgraph_steps = nsteps; h->sgraph_W = W; h->sgraph_kernel = kernel; h->sgraph_chain = chain; h->sgraph_cap = cap; h->sgraph_wpb = h->warps_per_block; h->sgraph_launches = l; }
        launches = h->sgraph_launches;
    } else {
        cudaError_t e = enqueue_swept(h, kernel, d_u, nsteps, W, st, &launches);
        if (e != cudaSuccess) return fail_cuda(e, "swept_run");
    }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

// ---- tuner (row A8; "best node size") -----------------------------------------------------------
extern "C" int swept_tune(swept_handle_t h, void *d_u_scratch, int blocks_per_sm_cap, int *best_tile_width, void *cuda_stream) {
    int rc = run_args_ok(h, d_u_scratch, 0, "swept_tune");
    if (rc) return rc;
    if (blocks_per_sm_cap < 0) return fail(SWEPT_EINVAL, "swept_tune: blocks_per_sm_cap < 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = handle_enter(h, st, "swept_tune"))) return rc;
    LeaveGuard leave{h, st};
    const int saved_cap = h->blocks_per_sm, saved_graph = h->swept_graph;
    h->blocks_per_sm = blocks_per_sm_cap;
    h->swept_graph = 0;
    int wmax = h->max_tile_width ? h->max_tile_width : 4096;
    if ((int64_t)wmax > h->nx) wmax = (int)h->nx;
    int wtop = 0;
    for (int W = 4 * h->H; W <= wmax; W <<= 1) if (check_width(h, W, h->kernel, false)) wtop = W;
    if (!wtop) { h->blocks_per_sm = saved_cap; h->swept_graph = saved_graph; return fail(SWEPT_EINVAL, "swept_tune: no legal tile width"); }
    // every candidate advances the same number of timesteps: 24 half-cycles of the widest tile (long enough that the first and last
    // phase -- half a phase of work each -- and the one-off wavefront fill of the launch-free kernels do not decide the ranking:
    // with twelve, heat fp32 at nx = 2^22 was tuned to W = 512 although W = 1024 is 6 % faster over a 50 000-step run)
    const int64_t nsteps = 24 * (int64_t)(wtop / (2 * h->H * h->S));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    int best = 0, best_chain = 0, best_cap = 0, best_pack = 0;
    const int saved_pack = h->pack;
    h->tuned_pack = 0;
    float best_ms = 1e30f;
    cudaError_t e = cudaSuccess;
    const int saved_chain = h->chain;
    h->tuned_chain = 0;
    h->tuned_cap = 0;
    h->tuned_kernel = -1;
    const bool wave = h->kernel == SWEPT_KERNEL_WAVE;
    for (int W = 4 * h->H; W <= wtop && e == cudaSuccess; W <<= 1) {
        if (!check_width(h, W, h->kernel, false)) continue;
        // default option (ring kernel): also time the band kernel with in-warp exchange (one more computing warp per SM on the
        // largest grids) and the tile-flag kernel (wins where few warps fit an SM)
        for (int mode = saved_chain; mode >= (saved_chain == 3 && wave ? 1 : saved_chain) && e == cudaSuccess; --mode) {
            h->chain = mode;
            // resident warps per SM: with no cap given, the register-resident kernels are also tried at 4, 3 and 2 blocks of 4
            // warps per SM (the band kernel: 16, 12, 8 warps in its one block) -- fp32 and KS run faster below full occupancy
            static const int caps_auto[] = {0, 4, 3, 2};
            const int ncaps = (blocks_per_sm_cap == 0 && wave) ? (mode >= 2 ? 2 : 4) : 1;   // band / ring: none and 16 warps only (measured: fewer never wins)
            for (int ci = 0; ci < ncaps && e == cudaSuccess; ++ci) {
                const int cap = ncaps == 1 ? blocks_per_sm_cap : caps_auto[ci];
                h->blocks_per_sm = cap;
                // heat and KS fp32 on the band kernel: one band per warp slot, and packed pairs
                const int npack = (saved_pack == 0 && mode == 2 && wave && h->problem != SWEPT_EULER && h->dtype == SWEPT_F32) ? 2 : 1;
                for (int pi = 0; pi < npack && e == cudaSuccess; ++pi) {
                    if (npack == 2) h->pack = 1 + pi;
                    float ms_min = 1e30f;
                    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {   // rep 0 warms up
                        int64_t l = 0;
                        cudaEventRecord(e0, st);
                        e = enqueue_swept(h, h->kernel, d_u_scratch, nsteps, W, st, &l);
                        cudaEventRecord(e1, st);
                        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
                        float ms = 0;
                        if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
                        if (rep > 0 && ms < ms_min) ms_min = ms;
                        h->launches_total += l;
                    }
                    if (e == cudaSuccess && ms_min < best_ms) { best_ms = ms_min; best = W; best_chain = mode; best_cap = cap; best_pack = npack == 2 ? h->pack : 0; }
                }
                h->pack = saved_pack;
            }
        }
    }
    h->chain = saved_chain;
    // default options: the paper-style shared-memory kernels compete too (one thread per point: on small Euler grids they have 8 x
    // the parallelism of the register kernels' lane per 8 cells)
    int best_kernel = -1;
    // ... which can only matter while the grid gives the register kernels fewer than four warps per SM sub-partition at their
    // narrowest launch-free tile (64 x 2h points); on larger grids the candidates would only cost tuning time
    const bool few_warps = h->nx / (64 * 2 * h->H) < (int64_t)16 * h->sm_count;
    if (wave && saved_chain == 3 && blocks_per_sm_cap == 0 && !h->bc && few_warps && e == cudaSuccess) {
        h->blocks_per_sm = 0;
        for (int W = 32; W <= wmax && e == cudaSuccess; W <<= 1) {
            if (!check_width(h, W, SWEPT_KERNEL_SMEM, false)) continue;
            float ms_min = 1e30f;
            for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
                int64_t l = 0;
                cudaEventRecord(e0, st);
                e = enqueue_swept(h, SWEPT_KERNEL_SMEM, d_u_scratch, nsteps, W, st, &l);
                cudaEventRecord(e1, st);
                if (e == cudaSuccess) e = cudaEventSynchronize(e1);
                float ms = 0;
                if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
                if (rep > 0 && ms < ms_min) ms_min = ms;
                h->launches_total += l;
            }
            if (e == cudaSuccess && ms_min < best_ms) { best_ms = ms_min; best = W; best_chain = 0; best_cap = 0; best_pack = 0; best_kernel = SWEPT_KERNEL_SMEM; }
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    h->blocks_per_sm = saved_cap;
    h->swept_graph = saved_graph;
    if (e != cudaSuccess) return fail_cuda(e, "swept_tune");
    drop_graphs(h);                                      // a cached swept graph was captured with the pre-tune launch shape
    h->tuned_tile_width = best;
    h->tuned_chain = (saved_chain == 3 && h->kernel == SWEPT_KERNEL_WAVE) ? best_chain : 0;
    h->tuned_cap = blocks_per_sm_cap == 0 ? best_cap : 0;
    h->tuned_pack = best_pack;
    h->tuned_kernel = best_kernel;
    if (best_tile_width) *best_tile_width = best;
    return SWEPT_OK;
}

// ---- end-to-end convenience: host buffer in, host buffer out -------------------------------------------------
extern "C" int swept_run_host(swept_handle_t h, void *h_u, int64_t nsteps, int tile_width, int use_swept, void *cuda_stream) {
    if (!h) return fail(SWEPT_EINVAL, "swept_run_host: NULL handle");
    if (!h_u) return fail(SWEPT_EINVAL, "swept_run_host: h_u is NULL");
    if (nsteps < 0) return fail(SWEPT_EINVAL, "swept_run_host: nsteps < 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    int rc0 = handle_enter(h, st, "swept_run_host");
    if (rc0) return rc0;
    LeaveGuard leave{h, st};
    if (!h->host_stage) {
        e = cudaMalloc(&h->host_stage, h->field_bytes);
        if (e != cudaSuccess) { cudaGetLastError(); h->host_stage = nullptr; return fail(SWEPT_ENOMEM, "swept_run_host: cudaMalloc: %s", cudaGetErrorString(e)); }
    }
    e = cudaMemcpyAsync(h->host_stage, h_u, h->field_bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail_cuda(e, "swept_run_host: H2D");
    int rc = use_swept ? swept_run(h, h->host_stage, nsteps, tile_width, cuda_stream) : naive_run(h, h->host_stage, nsteps, cuda_stream);
    if (rc) return rc;
    e = cudaMemcpyAsync(h_u, h->host_stage, h->field_bytes, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return fail_cuda(e, "swept_run_host: D2H");
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(e, "swept_run_host: synchronize");
    if (*(volatile unsigned *)h->abort_seen) return report_abort(h, "swept_run_host");    // h_u holds garbage: say so now
    return SWEPT_OK;
}

extern "C" int swept_check(swept_handle_t h) {
    if (!h) return fail(SWEPT_EINVAL, "swept_check: NULL handle");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "swept_check");
    if (dev != h->device) return fail(SWEPT_EINVAL, "swept_check: the handle was created on device %d but device %d is current", h->device, dev);
    e = cudaEventSynchronize(h->busy);       // behind the last call's kernels and the copy of the abort word
    if (e != cudaSuccess) return fail_cuda(e, "swept_check");
    if (*(volatile unsigned *)h->abort_seen) return report_abort(h, "swept_check");
    return SWEPT_OK;
}

extern "C" int swept_set_option(swept_handle_t h, int key, int value) {
    if (!h) return fail(SWEPT_EINVAL, "swept_set_option: NULL handle");
    switch (key) {
        case SWEPT_OPT_KERNEL:
            if (value != SWEPT_KERNEL_SMEM && value != SWEPT_KERNEL_WAVE) return fail(SWEPT_EINVAL, "swept_set_option: unknown kernel %d", value);
            if (value != h->kernel) { h->tuned_tile_width = 0; h->tuned_chain = 0; h->tuned_cap = 0; h->tuned_kernel = -1; }
            h->kernel = value;
            return SWEPT_OK;
        case SWEPT_OPT_NAIVE_GRAPH:
            if (value != 0 && value != 1) return fail(SWEPT_EINVAL, "swept_set_option: NAIVE_GRAPH takes 0 or 1");
            h->naive_graph = value;
            return SWEPT_OK;
        case SWEPT_OPT_NAIVE_SHARE:
            if (value != 0 && value != 1) return fail(SWEPT_EINVAL, "swept_set_option: NAIVE_SHARE takes 0 or 1");
            if (value != h->naive_share) drop_graphs(h);
            h->naive_share = value;
            return SWEPT_OK;
        case SWEPT_OPT_SWEPT_GRAPH:
            if (value != 0 && value != 1) return fail(SWEPT_EINVAL, "swept_set_option: SWEPT_GRAPH takes 0 or 1");
            h->swept_graph = value;
            return SWEPT_OK;
        case SWEPT_OPT_CHAIN:
            if (value < 0 || value > 3) return fail(SWEPT_EINVAL, "swept_set_option: CHAIN takes 0, 1, 2 or 3");
            h->chain = value;
            return SWEPT_OK;
        case SWEPT_OPT_PACK:
            if (value < 0 || value > 2) return fail(SWEPT_EINVAL, "swept_set_option: PACK takes 0 (auto), 1 (off) or 2 (on)");
            h->pack = value;
            drop_graphs(h);
            return SWEPT_OK;
        case SWEPT_OPT_INJECT_ABORT: {
            if (value != 1) return fail(SWEPT_EINVAL, "swept_set_option: INJECT_ABORT takes 1");
            const unsigned one = 1;
            cudaError_t e = cudaEventSynchronize(h->busy);
            if (e == cudaSuccess) e = cudaMemcpy(h->sync_base, &one, sizeof one, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) return fail_cuda(e, "swept_set_option(INJECT_ABORT)");
            return SWEPT_OK;
        }
        case SWEPT_OPT_BLOCKS_PER_SM:
            if (value < 0 || value > 32) return fail(SWEPT_EINVAL, "swept_set_option: BLOCKS_PER_SM takes 0..32");
            h->blocks_per_sm = value;
            drop_graphs(h);
            return SWEPT_OK;
        case SWEPT_OPT_WARPS_PER_BLOCK:
            if (value != 1 && value != 2 && value != 4 && value != 8 && value != 16) return fail(SWEPT_EINVAL, "swept_set_option: WARPS_PER_BLOCK takes 1, 2, 4, 8 or 16");
            h->warps_per_block = value;
            drop_graphs(h);
            return SWEPT_OK;
        default:
            return fail(SWEPT_EINVAL, "swept_set_option: unknown key %d", key);
    }
}

extern "C" int swept_get_info(swept_handle_t h, swept_info_t *info) {
    if (!h || !info) return fail(SWEPT_EINVAL, "swept_get_info: NULL argument");
    info->problem = h->problem; info->dtype = h->dtype;
    info->radius = h->H; info->stages = h->S; info->ncomp = h->NC;
    info->nx = h->nx;
    info->workspace_bytes = (int64_t)h->field_bytes;
    info->tuned_tile_width = h->tuned_tile_width;
    info->launches_last_call = h->launches_last;
    info->launches_total = h->launches_total;
    info->sm_count = h->sm_count;
    info->max_smem_per_block = h->max_smem;
    info->last_sweep_launch = h->last_sweep_launch;
    info->boundary = h->bc;
    info->tuned_chain = h->tuned_chain;
    info->tuned_blocks_per_sm = h->tuned_cap;
    info->tuned_pack = h->tuned_pack;
    info->tuned_kernel = h->tuned_kernel;
    return SWEPT_OK;
}

// ---- streaming-band schedule, host logic only (no device needed) ------------------------------------------------
extern "C" int swept_band_layout(int ntiles, int sm_count, int warps_per_block, swept_band_layout_t *out) {
    if (!out) return fail(SWEPT_EINVAL, "swept_band_layout: out is NULL");
    if (ntiles < 1 || sm_count < 1) return fail(SWEPT_EINVAL, "swept_band_layout: ntiles and sm_count must be positive");
    if (warps_per_block < 1 || warps_per_block > 32 || (warps_per_block > 4 && warps_per_block % 4 != 0))
        return fail(SWEPT_EINVAL, "swept_band_layout: warps_per_block must be 1, 2, 3, 4 or a multiple of 4 up to 32");
    const BandGrid g = band_layout(ntiles, sm_count, warps_per_block);
    out->blocks = g.nblocks; out->warps_per_block = g.wpb; out->slots_per_block = g.SL; out->warps_per_slot = g.wps;
    out->slots = g.G; out->max_bands_per_warp = g.kmax; out->ntiles = ntiles;
    return SWEPT_OK;
}

extern "C" int swept_band_owner(const swept_band_layout_t *lay, int band, int *block, int *warp, int *index) {
    if (!lay || !block || !warp || !index) return fail(SWEPT_EINVAL, "swept_band_owner: NULL argument");
    if (band < 0 || band >= lay->ntiles) return fail(SWEPT_EINVAL, "swept_band_owner: band %d outside [0, %d)", band, lay->ntiles);
    BandGrid g;
    g.nblocks = lay->blocks; g.wpb = lay->warps_per_block; g.SL = lay->slots_per_block; g.wps = lay->warps_per_slot;
    g.G = lay->slots; g.kmax = lay->max_bands_per_warp;
    band_owner(g, band, block, warp, index);
    return SWEPT_OK;
}

extern "C" int swept_problem_info(int problem, int *radius, int *stages, int *ncomp) {
    if (problem != SWEPT_HEAT && problem != SWEPT_KS && problem != SWEPT_EULER) return fail(SWEPT_EINVAL, "swept_problem_info: unknown problem %d", problem);
    if (radius) *radius = radius_of(problem);
    if (stages) *stages = stages_of(problem);
    if (ncomp) *ncomp = ncomp_of(problem);
    return SWEPT_OK;
}

extern "C" int swept_measure_alu_peak(int dtype, double *instr_per_s, double *ms, void *cuda_stream) {
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return fail(SWEPT_EINVAL, "swept_measure_alu_peak: unknown dtype %d", dtype);
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "swept_measure_alu_peak: no CUDA device");
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    e = run_alu_peak(dtype, sms, instr_per_s, ms, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(e, "swept_measure_alu_peak");
    return SWEPT_OK;
}

extern "C" int swept_measure_latencies(double *cycles, void *cuda_stream) {
    if (!cycles) return fail(SWEPT_EINVAL, "swept_measure_latencies: cycles is NULL");
    const cudaError_t e = run_latency_probes(cycles, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(e, "swept_measure_latencies");
    return SWEPT_OK;
}

extern "C" int swept_measure_smem_peak(double *bytes_per_s, double *ms, void *cuda_stream) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "swept_measure_smem_peak: no CUDA device");
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    e = run_smem_peak(sms, bytes_per_s, ms, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(e, "swept_measure_smem_peak");
    return SWEPT_OK;
}

// ---- swept_run_static: the swept rule for callers that must not allocate (include/swept1d.h) ------------------------
// Row R1 of the staircase (the handle's `work`) lives in this file-scope array instead of a cudaMalloc'ed buffer.  Every
// device that loads the library carries the array until the process exits.
static __device__ __align__(256) unsigned char g_static_r1[SWEPT_STATIC_SCRATCH_BYTES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDevice {
    void *r1;                    // DEVICE address of g_static_r1 on this device; nullptr until the set-up ran
    unsigned char prepared[3][2];// kernel attributes set for (problem, dtype)
    int sm_count, max_smem;
};
StaticDevice g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mutex;
}  // namespace

// Once per device, with that device current.  In host code `g_static_r1` names a host-side shadow of the symbol, not device
// memory: the address a kernel may use has to be asked for.
static int static_setup(int dev, int problem, int dtype, StaticDevice **out) {
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(SWEPT_EINVAL, "swept_run_static: device ordinal %d outside [0, %d)", dev, STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice *d = &g_static_dev[dev];
    if (!d->r1) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_r1);
        if (e != cudaSuccess) return fail_cuda(e, "swept_run_static: cudaGetSymbolAddress(static scratch)");
        if (!p || ((uintptr_t)p & 255) != 0) return fail(SWEPT_ECUDA, "swept_run_static: static scratch address %p is not 256-byte aligned", p);
        e = cudaDeviceGetAttribute(&d->sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&d->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return fail_cuda(e, "swept_run_static: device attributes");
        d->r1 = p;
    }
    if (!d->prepared[problem][dtype]) {
        const cudaError_t e = swept_wave_prepare(problem, dtype);    // cudaFuncSetAttribute only
        if (e != cudaSuccess) return fail_cuda(e, "swept_run_static: kernel attribute setup");
        d->prepared[problem][dtype] = 1;
    }
    *out = d;
    return SWEPT_OK;
}

extern "C" int swept_run_static(int problem, int64_t nx, double dx, double dt, const swept_params_t *p, void *d_u, int64_t nsteps,
                                int tile_width, void *cuda_stream) {
    g_err[0] = 0;
    if (problem != SWEPT_HEAT && problem != SWEPT_KS && problem != SWEPT_EULER) return fail(SWEPT_EINVAL, "swept_run_static: unknown problem %d", problem);
    const int dtype = p ? p->dtype : SWEPT_F64;
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return fail(SWEPT_EINVAL, "swept_run_static: unknown dtype %d", dtype);
    if (!is_pow2(nx) || nx < 8) return fail(SWEPT_EINVAL, "swept_run_static: nx=%lld must be a power of two >= 8", (long long)nx);
    if (!isfinite(dx) || !isfinite(dt) || dx <= 0.0 || dt <= 0.0) return fail(SWEPT_EINVAL, "swept_run_static: dx and dt must be finite and positive");
    const double alpha = p ? p->alpha : 1.0, gamma = p ? p->gamma : 1.4;
    if (problem == SWEPT_HEAT && !(isfinite(alpha) && alpha > 0.0)) return fail(SWEPT_EINVAL, "swept_run_static: alpha must be finite and positive");
    if (problem == SWEPT_EULER && !(isfinite(gamma) && gamma > 1.0)) return fail(SWEPT_EINVAL, "swept_run_static: gamma must be finite and > 1");
    if (p && p->boundary != SWEPT_BC_PERIODIC) return fail(SWEPT_EINVAL, "swept_run_static: periodic domains only");
    // the size limit comes before anything touches the device
    const int NC = ncomp_of(problem);
    if (nx > (int64_t)(SWEPT_STATIC_SCRATCH_BYTES / (NC * elem_size(dtype))))
        return fail(SWEPT_EINVAL, "swept_run_static: the field has %lld x %d elements of %zu bytes, the static scratch holds %d bytes "
                                  "(SWEPT_STATIC_SCRATCH_BYTES); larger grids need a handle (swept_create)",
                    (long long)nx, NC, elem_size(dtype), (int)SWEPT_STATIC_SCRATCH_BYTES);

    // a handle on the stack whose workspace is the static array: the host driver below is the one swept_run uses
    swept_ctx ctx;
    memset(&ctx, 0, sizeof ctx);
    swept_ctx *h = &ctx;
    h->problem = problem; h->dtype = dtype;
    h->H = radius_of(problem); h->S = stages_of(problem); h->NC = NC;
    h->nx = nx; h->dx = dx; h->dt = dt; h->alpha = alpha; h->gamma = gamma;
    h->bc = SWEPT_BC_PERIODIC;
    h->kernel = SWEPT_KERNEL_WAVE;
    h->chain = 0;                          // one launch per half-cycle: needs no flags, no counters, no pinned abort word
    h->last_sweep_launch = -1;
    h->tuned_kernel = -1;
    h->warps_per_block = 4;
    h->field_bytes = (size_t)NC * (size_t)nx * elem_size(dtype);
    if (dtype == SWEPT_F64) fill_consts<double>(h); else fill_consts<float>(h);
    int rc = run_args_ok(h, d_u, nsteps, "swept_run_static");
    if (rc) return rc;

    int W = tile_width;
    if (W == 0) {
        for (int w = 256; w >= 4 * h->H && !W; w >>= 1)
            if ((int64_t)w <= nx && swept_wave_supports(problem, dtype, w)) W = w;
        if (!W) return fail(SWEPT_EINVAL, "swept_run_static: nx=%lld is narrower than the narrowest register-resident tile", (long long)nx);
    }
    char buf[160];
    const char *why = width_problem(problem, dtype, nx, W, SWEPT_KERNEL_WAVE, 0, buf, sizeof buf);
    if (why) return fail(SWEPT_EINVAL, "swept_run_static: tile_width %d: %s", W, why);

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "swept_run_static: no CUDA device (this library has no CPU fallback)");
    StaticDevice *sd = nullptr;
    if ((rc = static_setup(dev, problem, dtype, &sd))) return rc;
    h->device = dev; h->sm_count = sd->sm_count; h->max_smem = sd->max_smem;
    h->work = sd->r1;

    int64_t launches = 0;
    e = enqueue_swept(h, SWEPT_KERNEL_WAVE, d_u, nsteps, W, (cudaStream_t)cuda_stream, &launches, 0);
    if (e != cudaSuccess) return fail_cuda(e, "swept_run_static");
    return SWEPT_OK;
}
