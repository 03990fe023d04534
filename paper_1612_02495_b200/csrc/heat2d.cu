// heat2d.cu -- the 2-D swept rule for the heat equation (include/swept2d.h): kernels and C ABI.
//
// Block = tile of W x W points, thread = point, two shared-memory planes of (W + 2)^2 values: plane 0 holds the newest even
// tier of every point of the tile and its one-point halo, plane 1 the newest odd tier -- the 2-D form of the paper's two-row
// shared matrix.  A launch runs one REGION kind on every tile of its alignment: at local tier s the points
// of rect_x(s) x rect_y(s) are updated from plane (s-1)&1 into plane s&1 (one block barrier per tier), where per direction
//     U (shrinking, the upright triangle of PAPER.md:82):   [s, W - s)
//     D (expanding, the inverted triangle of PAPER.md:98):  [W/2 - s, W/2 + s)
// and tiers s > L of an octahedron continue as U with s - L.  Afterwards every thread stores what it updated: plane p of its point
// if it wrote plane p -- nothing else, so tiles of one launch never write what another reads (tests/test_geometry2d.py runs the same
// plan on a plain-Python model).  The point update is Heat2D<T>::point of stencils.cuh, shared with the classic kernel.
#include <math.h>
#include <string.h>

#include <new>

#include "../../include/swept2d.h"
#include "internal.h"
#include "stencils.cuh"

using namespace swept;

struct swept2d_ctx {
    int dtype, device;
    int64_t nx, ny;
    double dx, dt, alpha;
    ConstBlock cb;
    void *work;
    size_t field_bytes;
    int64_t launches_last, launches_total;
};

namespace {

enum { R_PYRAMID = 0, R_BRIDGES = 1, R_INVERTED = 2, R_OCTAHEDRON = 3 };

template <class T>
__global__ void __launch_bounds__(256) classic2d_kernel(const T *__restrict__ src, T *__restrict__ dst, int64_t nx, int64_t ny, typename Heat2D<T>::Consts c) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, j = (int64_t)blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= nx || j >= ny) return;
    const int64_t ie = (i + 1) & (nx - 1), iw = (i - 1) & (nx - 1), jn = (j + 1) & (ny - 1), js = (j - 1) & (ny - 1);
    dst[j * nx + i] = Heat2D<T>::point(c, src[j * nx + i], src[j * nx + ie], src[j * nx + iw], src[jn * nx + i], src[js * nx + i]);
}

// One region kind on the tiles whose origin is (ox, oy) + (tile index) * W.  REGION = R_BRIDGES: blockIdx.z = 0 runs the x-bridges
// (expanding in x, shrinking in y) at origin (ox, oy), blockIdx.z = 1 the y-bridges at origin (oy, ox).
template <class T, int W, int REGION>
__global__ void __launch_bounds__(W *W) swept2d_kernel(T *__restrict__ p0, T *__restrict__ p1, int64_t nx, int64_t ny, int ox, int oy, typename Heat2D<T>::Consts c) {
    constexpr int L = W / 2, C = W / 2, PS = W + 2;       // PS: plane stride (one halo point on every side)
    __shared__ T pl[2][PS * PS];
    const int x = (int)threadIdx.x, y = (int)threadIdx.y;
    const bool ybridge = REGION == R_BRIDGES && blockIdx.z == 1;
    const int64_t gx0 = (int64_t)blockIdx.x * W + (ybridge ? oy : ox), gy0 = (int64_t)blockIdx.y * W + (ybridge ? ox : oy);
    const int64_t mx = nx - 1, my = ny - 1;
    auto gidx = [&](int lx, int ly) -> int64_t { return ((gy0 + ly) & my) * nx + ((gx0 + lx) & mx); };
    // ---- load both planes: own point, and the halo ring by the first 4 W threads
    {
        const int64_t g = gidx(x, y);
        pl[0][(y + 1) * PS + x + 1] = p0[g];
        if (REGION != R_PYRAMID) pl[1][(y + 1) * PS + x + 1] = p1[g];
        const int t = y * W + x;
        if (t < 4 * W) {
            const int side = t / W, k = t % W;
            const int lx = side == 0 ? -1 : (side == 1 ? W : k), ly = side == 2 ? -1 : (side == 3 ? W : k);
            const int64_t gh = gidx(lx, ly);
            pl[0][(ly + 1) * PS + lx + 1] = p0[gh];
            if (REGION != R_PYRAMID) pl[1][(ly + 1) * PS + lx + 1] = p1[gh];
        }
    }
    __syncthreads();
    // ---- tiers
    constexpr int S0 = 1, S1 = REGION == R_PYRAMID ? L - 1 : (REGION == R_OCTAHEDRON ? 2 * L - 1 : L);
    int s_lo = 0, s_hi = 0;                               // tiers this thread updated: [s_lo, s_hi] (0 = none)
    const int me = (y + 1) * PS + x + 1;
#pragma unroll 1
    for (int s = S0; s <= S1; ++s) {
        int xa, xb, ya, yb;
        if (REGION == R_PYRAMID) { xa = ya = s; xb = yb = W - s; }
        else if (REGION == R_BRIDGES) {
            const int ea = C - s, eb = C + s, sa = s, sb = W - s;           // expanding / shrinking interval
            xa = ybridge ? sa : ea; xb = ybridge ? sb : eb;
            ya = ybridge ? ea : sa; yb = ybridge ? eb : sb;
        } else if (s <= L) { xa = ya = C - s; xb = yb = C + s; }
        else { xa = ya = s - L; xb = yb = W - (s - L); }
        if (x >= xa && x < xb && y >= ya && y < yb) {
            const T *src = pl[(s - 1) & 1];
            pl[s & 1][me] = Heat2D<T>::point(c, src[me], src[me + 1], src[me - 1], src[me + PS], src[me - PS]);
            if (s_lo == 0) s_lo = s;
            s_hi = s;
        }
        __syncthreads();
    }
    // ---- store what this thread updated
    if (s_hi > 0) {
        const int64_t g = gidx(x, y);
        T *newest = (s_hi & 1) ? p1 : p0, *other = (s_hi & 1) ? p0 : p1;
        newest[g] = pl[s_hi & 1][me];
        if (s_hi > s_lo) other[g] = pl[(s_hi - 1) & 1][me];
    }
}

template <class T> typename Heat2D<T>::Consts consts_of(const swept2d_ctx *h) { return *reinterpret_cast<const typename Heat2D<T>::Consts *>(h->cb.bytes); }

template <class T> cudaError_t classic2d(swept2d_ctx *h, void *d_u, int64_t nsteps, cudaStream_t st, int64_t *launches) {
    T *a = (T *)d_u, *b = (T *)h->work;
    const dim3 block(32, 8), grid((unsigned)((h->nx + 31) / 32), (unsigned)((h->ny + 7) / 8));
    for (int64_t m = 0; m < nsteps; ++m) {
        classic2d_kernel<T><<<grid, block, 0, st>>>(a, b, h->nx, h->ny, consts_of<T>(h));
        T *t = a; a = b; b = t;
        ++*launches;
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && a != (T *)d_u) e = cudaMemcpyAsync(d_u, a, h->field_bytes, cudaMemcpyDeviceToDevice, st);
    return e;
}

template <class T, int W> cudaError_t sweep2d(swept2d_ctx *h, void *d_u, int64_t K, cudaStream_t st, int64_t *launches) {
    if (K <= 0) return cudaSuccess;
    T *p0 = (T *)d_u, *p1 = (T *)h->work;
    const dim3 block(W, W), grid((unsigned)(h->nx / W), (unsigned)(h->ny / W), 1), grid2(grid.x, grid.y, 2);
    const typename Heat2D<T>::Consts c = consts_of<T>(h);
    swept2d_kernel<T, W, R_PYRAMID><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, 0, 0, c);
    ++*launches;
    for (int64_t k = 0; k < K; ++k) {
        const int a = (int)(k & 1) * (W / 2), b = W / 2 - a;      // a: the alignment that shrinks in this half-cycle
        swept2d_kernel<T, W, R_BRIDGES><<<grid2, block, 0, st>>>(p0, p1, h->nx, h->ny, b, a, c);
        if (k == K - 1) swept2d_kernel<T, W, R_INVERTED><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, c);
        else swept2d_kernel<T, W, R_OCTAHEDRON><<<grid, block, 0, st>>>(p0, p1, h->nx, h->ny, b, b, c);
        *launches += 2;
    }
    return cudaGetLastError();
}

template <class T> cudaError_t sweep2d_w(swept2d_ctx *h, void *d_u, int W, int64_t K, cudaStream_t st, int64_t *launches) {
    switch (W) {
        case 8: return sweep2d<T, 8>(h, d_u, K, st, launches);
        case 16: return sweep2d<T, 16>(h, d_u, K, st, launches);
        case 32: return sweep2d<T, 32>(h, d_u, K, st, launches);
        default: return cudaErrorInvalidValue;
    }
}

bool pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }

}  // namespace

extern "C" int swept2d_create(swept2d_handle_t *out, int64_t nx, int64_t ny, double dx, double dt, const swept2d_params_t *p) {
    if (!out) return swept_fail(SWEPT_EINVAL, "swept2d_create: out is NULL");
    *out = nullptr;
    const int dtype = p ? p->dtype : SWEPT_F64;
    const double alpha = p ? p->alpha : 1.0;
    if (dtype != SWEPT_F32 && dtype != SWEPT_F64) return swept_fail(SWEPT_EINVAL, "swept2d_create: unknown dtype %d", dtype);
    if (!pow2(nx) || !pow2(ny) || nx < 8 || ny < 8 || nx > ((int64_t)1 << 20) || ny > ((int64_t)1 << 20))
        return swept_fail(SWEPT_EINVAL, "swept2d_create: nx=%lld, ny=%lld must be powers of two in [8, 2^20]", (long long)nx, (long long)ny);
    if (!isfinite(dx) || !isfinite(dt) || dx <= 0.0 || dt <= 0.0 || !(isfinite(alpha) && alpha > 0.0))
        return swept_fail(SWEPT_EINVAL, "swept2d_create: dx, dt and alpha must be finite and positive");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_create: no CUDA device (this library has no CPU fallback): %s", cudaGetErrorString(e)); }
    swept2d_ctx *h = new (std::nothrow) swept2d_ctx();
    if (!h) return swept_fail(SWEPT_ENOMEM, "swept2d_create: out of host memory");
    h->dtype = dtype; h->device = dev; h->nx = nx; h->ny = ny; h->dx = dx; h->dt = dt; h->alpha = alpha;
    h->launches_last = h->launches_total = 0;
    const double Fo = alpha * dt / (dx * dx);                     // row A0: constants on the host in double, cast once
    memset(h->cb.bytes, 0, sizeof h->cb.bytes);
    if (dtype == SWEPT_F64) { Heat2D<double>::Consts c{Fo, 1.0 - 4.0 * Fo}; memcpy(h->cb.bytes, &c, sizeof c); }
    else { Heat2D<float>::Consts c{(float)Fo, (float)(1.0 - 4.0 * Fo)}; memcpy(h->cb.bytes, &c, sizeof c); }
    h->field_bytes = (size_t)nx * (size_t)ny * elem_size(dtype);
    e = cudaMalloc(&h->work, h->field_bytes);
    if (e != cudaSuccess) {
        delete h;
        cudaGetLastError();
        return swept_fail(e == cudaErrorMemoryAllocation ? SWEPT_ENOMEM : SWEPT_ECUDA, "swept2d_create: cudaMalloc workspace: %s", cudaGetErrorString(e));
    }
    *out = h;
    return SWEPT_OK;
}

static int args2d_ok(swept2d_ctx *h, void *d_u, int64_t nsteps, const char *who) {
    if (!h) return swept_fail(SWEPT_EINVAL, "%s: NULL handle", who);
    if (!d_u) return swept_fail(SWEPT_EINVAL, "%s: d_u is NULL", who);
    if (nsteps < 0) return swept_fail(SWEPT_EINVAL, "%s: nsteps < 0", who);
    if (((uintptr_t)d_u & 15) != 0) return swept_fail(SWEPT_EINVAL, "%s: d_u must be 16-byte aligned", who);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) { cudaGetLastError(); return swept_fail(SWEPT_EINVAL, "%s: the handle was created on device %d but device %d is current", who, h->device, dev); }
    return SWEPT_OK;
}

extern "C" int naive2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, void *cuda_stream) {
    int rc = args2d_ok(h, d_u, nsteps, "naive2d_run");
    if (rc) return rc;
    int64_t launches = 0;
    const cudaError_t e = h->dtype == SWEPT_F64 ? classic2d<double>(h, d_u, nsteps, (cudaStream_t)cuda_stream, &launches)
                                                : classic2d<float>(h, d_u, nsteps, (cudaStream_t)cuda_stream, &launches);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "naive2d_run: %s", cudaGetErrorString(e)); }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

extern "C" int swept2d_run(swept2d_handle_t h, void *d_u, int64_t nsteps, int tile_width, void *cuda_stream) {
    int rc = args2d_ok(h, d_u, nsteps, "swept2d_run");
    if (rc) return rc;
    int W = tile_width;
    if (W == 0) for (W = 32; W > 8 && (W > h->nx || W > h->ny); W >>= 1) {}
    if ((W != 8 && W != 16 && W != 32) || W > h->nx || W > h->ny)
        return swept_fail(SWEPT_EINVAL, "swept2d_run: tile_width %d: must be 8, 16 or 32 and at most nx, ny", tile_width);
    const int64_t L = W / 2, K = nsteps / L, r = nsteps % L;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int64_t launches = 0;
    cudaError_t e = h->dtype == SWEPT_F64 ? classic2d<double>(h, d_u, r, st, &launches) : classic2d<float>(h, d_u, r, st, &launches);
    if (e == cudaSuccess) e = h->dtype == SWEPT_F64 ? sweep2d_w<double>(h, d_u, W, K, st, &launches) : sweep2d_w<float>(h, d_u, W, K, st, &launches);
    if (e != cudaSuccess) { cudaGetLastError(); return swept_fail(SWEPT_ECUDA, "swept2d_run: %s", cudaGetErrorString(e)); }
    h->launches_last = launches;
    h->launches_total += launches;
    return SWEPT_OK;
}

extern "C" int swept2d_get_info(swept2d_handle_t h, swept2d_info_t *info) {
    if (!h || !info) return swept_fail(SWEPT_EINVAL, "swept2d_get_info: NULL argument");
    info->dtype = h->dtype; info->nx = h->nx; info->ny = h->ny;
    info->workspace_bytes = (int64_t)h->field_bytes;
    info->launches_last_call = h->launches_last; info->launches_total = h->launches_total;
    return SWEPT_OK;
}

extern "C" int swept2d_destroy(swept2d_handle_t h) {
    if (!h) return swept_fail(SWEPT_EINVAL, "swept2d_destroy: NULL handle");
    if (h->work) cudaFree(h->work);
    delete h;
    return SWEPT_OK;
}
