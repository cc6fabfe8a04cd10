// Overlap pruning's neighbour search (§4.3): "eliminating Gaussians whose average distance of its three nearest
// neighbors falls below a pre-defined distance threshold d_OP^(l) ... set as half of the scale constraint s_min^(l)".
// SURVEY §8(f)4.  A training-side kernel: it runs on caller-owned device arrays and needs no scene.
//
// The decision mean(d1, d2, d3) < d_OP only ever involves neighbours closer than R = 3 d_OP (d1 + d2 + d3 < 3 d_OP makes
// every d_i < 3 d_OP), so a uniform grid of cell size h = R (1 + 2^-20) is searched over the 27 cells around a point:
//   k_knn_count   cell of every point (fp64 quotient, so that rounding cannot move a point across a cell), one counter per
//                 hash bucket;
//   k_knn_scan    one CTA: exclusive scan of the bucket counters;
//   k_knn_fill    point indices into their bucket's segment (any order: only distances are used);
//   k_knn_query   one thread per point: the k = min(3, n - 1) smallest squared distances among the points of the 27 cells
//                 (a bucket may hold other cells' points too: only members of the cell being visited count).  If the
//                 k-th smallest is within h no point outside the 27 cells can be nearer, and the mean is exact; otherwise
//                 all that is known is mean >= d_OP, and +inf is reported.
// Canonical arithmetic (the oracle's): d^2 = (dx dx + dy dy) + dz dz in fp32, one rounding per operation; mean =
// ((sqrt(a) + sqrt(b)) + sqrt(c)) / k with a <= b <= c, fp32; remove iff mean < 0.5f * s_min.
#include <math.h>

#include <mutex>

#include "flod_internal.cuh"

namespace flod {

struct KnnGrid { double lo[3]; double inv_h; unsigned int mask; };

__device__ __forceinline__ int3 knn_cell(const KnnGrid &g, float x, float y, float z)
{
    return make_int3((int)floor(((double)x - g.lo[0]) * g.inv_h), (int)floor(((double)y - g.lo[1]) * g.inv_h),
                     (int)floor(((double)z - g.lo[2]) * g.inv_h));
}
__device__ __forceinline__ unsigned int knn_hash(const KnnGrid &g, int3 c)
{
    return (((unsigned int)c.x * 73856093u) ^ ((unsigned int)c.y * 19349663u) ^ ((unsigned int)c.z * 83492791u)) & g.mask;
}

__global__ void k_knn_count(const float *__restrict__ mean, long long n, const __grid_constant__ KnnGrid g, int3 *__restrict__ cell,
                            unsigned int *__restrict__ count)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int3 c = knn_cell(g, mean[3 * i], mean[3 * i + 1], mean[3 * i + 2]);
    cell[i] = c;
    atomicAdd(count + knn_hash(g, c), 1u);
}

// count[0 .. m) -> exclusive offsets in start[0 .. m], cursors zeroed; one CTA of 1024 threads
__global__ void __launch_bounds__(1024) k_knn_scan(unsigned int *__restrict__ count, unsigned int *__restrict__ start, unsigned int m)
{
    __shared__ unsigned int s_w[32];
    const unsigned int tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const unsigned int per = (m + 1023u) / 1024u;
    const unsigned int b0 = min(tid * per, m), b1 = min(b0 + per, m);
    unsigned int sum = 0;
    for (unsigned int b = b0; b < b1; ++b) sum += count[b];
    unsigned int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    unsigned int run = incl - sum;
    for (unsigned int w = 0; w < warp; ++w) run += s_w[w];
    for (unsigned int b = b0; b < b1; ++b) {
        const unsigned int c = count[b];
        start[b] = run;
        count[b] = 0;                                   // becomes the fill cursor
        run += c;
    }
    if (tid == 1023) start[m] = run;
}

__global__ void k_knn_fill(long long n, const __grid_constant__ KnnGrid g, const int3 *__restrict__ cell, const unsigned int *__restrict__ start,
                           unsigned int *__restrict__ cursor, unsigned int *__restrict__ items)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned int b = knn_hash(g, cell[i]);
    items[start[b] + atomicAdd(cursor + b, 1u)] = (unsigned int)i;
}

__global__ void __launch_bounds__(128)
k_knn_query(const float *__restrict__ mean, long long n, const __grid_constant__ KnnGrid g, float h2, float d_op, const int3 *__restrict__ cell,
            const unsigned int *__restrict__ start, const unsigned int *__restrict__ items, float *__restrict__ out_mean,
            unsigned char *__restrict__ out_remove)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x = mean[3 * i], y = mean[3 * i + 1], z = mean[3 * i + 2];
    const int3 c = cell[i];
    const float INF = __int_as_float(0x7f800000);
    float a = INF, b = INF, cc = INF;                   // the three smallest squared distances, a <= b <= cc
    for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                const int3 q = make_int3(c.x + dx, c.y + dy, c.z + dz);
                const unsigned int bk = knn_hash(g, q);
                const unsigned int e = start[bk + 1];
                for (unsigned int t = start[bk]; t < e; ++t) {
                    const unsigned int j = items[t];
                    const int3 cj = cell[j];
                    if (cj.x != q.x || cj.y != q.y || cj.z != q.z || (long long)j == i) continue;   // another cell of the bucket / itself
                    const float ex = __fsub_rn(mean[3 * (size_t)j], x), ey = __fsub_rn(mean[3 * (size_t)j + 1], y), ez = __fsub_rn(mean[3 * (size_t)j + 2], z);
                    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(ex, ex), __fmul_rn(ey, ey)), __fmul_rn(ez, ez));
                    if (d2 < cc) {
                        if (d2 < b) { cc = b; if (d2 < a) { b = a; a = d2; } else b = d2; }
                        else cc = d2;
                    }
                }
            }
    const int k = n - 1 < 3 ? (int)(n - 1) : 3;
    const float kth = k == 3 ? cc : (k == 2 ? b : a);
    float m = INF;
    if (k >= 1 && kth <= h2) {
        float s = __fsqrt_rn(a);
        if (k >= 2) s = __fadd_rn(s, __fsqrt_rn(b));
        if (k >= 3) s = __fadd_rn(s, __fsqrt_rn(cc));
        m = __fdiv_rn(s, (float)k);
    }
    if (out_mean) out_mean[i] = m;
    out_remove[i] = (k >= 1 && m < d_op) ? 1 : 0;
}

}  // namespace flod

using namespace flod;

namespace {
unsigned int knn_table_size(long long n)
{
    unsigned int m = 1024;
    while ((long long)m < 2 * n && m < (1u << 30)) m <<= 1;
    return m;
}
size_t knn_align(size_t v) { return (v + 255) / 256 * 256; }
}  // namespace

extern "C" {

size_t flod_overlap_prune_workspace_bytes(int64_t n)
{
    if (n < 0 || n >= (1ll << 31)) return 0;
    const size_t m = knn_table_size(n), nn = (size_t)(n > 0 ? n : 1);
    return knn_align(nn * sizeof(int3)) + knn_align((m + 1) * 4) + knn_align((m + 1) * 4) + knn_align(nn * 4);
}

int flod_overlap_prune(const float *mean_dev, int64_t n, float s_min, const float bbox_lo[3], unsigned char *remove_dev,
                       float *mean_dist_dev, void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (n < 0 || n >= (1ll << 31) || !(s_min > 0.0f) || !isfinite(s_min) || !bbox_lo) return FLOD_E_INVALID_ARG;
    if (n == 0) return FLOD_OK;
    if (!mean_dev || !remove_dev || !workspace_dev || (uintptr_t)workspace_dev % 256) return FLOD_E_INVALID_ARG;
    if (workspace_bytes < flod_overlap_prune_workspace_bytes(n)) return FLOD_E_ARENA_TOO_SMALL;
    for (int k = 0; k < 3; ++k) if (!isfinite(bbox_lo[k])) return FLOD_E_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const float d_op = 0.5f * s_min;                                  // d_OP = s_min / 2
    const double h = 3.0 * (double)d_op * (1.0 + 9.5367431640625e-7);
    KnnGrid g;
    for (int k = 0; k < 3; ++k) g.lo[k] = (double)bbox_lo[k];
    g.inv_h = 1.0 / h;
    const unsigned int m = knn_table_size(n);
    g.mask = m - 1;
    unsigned char *base = (unsigned char *)workspace_dev;
    int3 *cell = (int3 *)base;                  base += knn_align((size_t)n * sizeof(int3));
    unsigned int *count = (unsigned int *)base; base += knn_align(((size_t)m + 1) * 4);
    unsigned int *start = (unsigned int *)base; base += knn_align(((size_t)m + 1) * 4);
    unsigned int *items = (unsigned int *)base;
    if (cudaMemsetAsync(count, 0, ((size_t)m + 1) * 4, s) != cudaSuccess) return FLOD_E_CUDA;
    const unsigned int grid = (unsigned int)((n + 255) / 256);
    k_knn_count<<<grid, 256, 0, s>>>(mean_dev, n, g, cell, count);
    k_knn_scan<<<1, 1024, 0, s>>>(count, start, m);
    k_knn_fill<<<grid, 256, 0, s>>>(n, g, cell, start, count, items);
    const float h2 = (float)(h * h) * 0.99999f;                       // (rounded down: "within h" must not be claimed too early)
    k_knn_query<<<(unsigned int)((n + 127) / 128), 128, 0, s>>>(mean_dev, n, g, h2, d_op, cell, start, items, mean_dist_dev, remove_dev);
    return cudaGetLastError() == cudaSuccess ? FLOD_OK : FLOD_E_CUDA;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ no-allocation variant
// flod_overlap_prune_static: the same four kernels on a scratch area that lives in the library's own device image, for
// callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The array below is
// held by every GPU that loads libflod.so until the process exits (8.0 MiB: the workspace of kKnnStaticMaxN points).
// In host code `g_knn_scratch` is a host-side stand-in for the symbol, NOT a device address: the address the kernels get
// comes from cudaGetSymbolAddress, asked once per device with that device current (knn_static_setup).
namespace {
constexpr long long kKnnStaticMaxN = 1ll << 18;                                   // 262 144 points
constexpr size_t knn_align_c(size_t v) { return (v + 255) / 256 * 256; }
constexpr size_t kKnnStaticTable = 2 * (size_t)kKnnStaticMaxN;                    // knn_table_size(kKnnStaticMaxN)
constexpr size_t kKnnStaticBytes = knn_align_c((size_t)kKnnStaticMaxN * sizeof(int3)) + 2 * knn_align_c((kKnnStaticTable + 1) * 4) +
                                   knn_align_c((size_t)kKnnStaticMaxN * 4);
static __device__ __align__(256) unsigned char g_knn_scratch[kKnnStaticBytes];

constexpr int kKnnMaxDevices = 64;
void *g_knn_scratch_ptr[kKnnMaxDevices];            // per device: the array's DEVICE address (null until set up)
std::mutex g_knn_setup_mutex;

// the device address of the scratch array on the CURRENT device; asked from the runtime once per device
int knn_static_setup(void **ptr_out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return FLOD_E_CUDA;
    if (dev < 0 || dev >= kKnnMaxDevices) return FLOD_E_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_knn_setup_mutex);
    if (!g_knn_scratch_ptr[dev]) {
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_knn_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return FLOD_E_CUDA; }
        g_knn_scratch_ptr[dev] = ptr;
    }
    *ptr_out = g_knn_scratch_ptr[dev];
    return FLOD_OK;
}
}  // namespace

extern "C" {

int64_t flod_overlap_prune_static_max_n(void) { return kKnnStaticMaxN; }

int flod_overlap_prune_static_setup(void)
{
    void *ptr = nullptr;
    return knn_static_setup(&ptr);
}

int flod_overlap_prune_static(const float *mean_dev, int64_t n, float s_min, const float bbox_lo[3], unsigned char *remove_dev,
                              float *mean_dist_dev, void *stream)
{
    if (n < 0 || !(s_min > 0.0f) || !isfinite(s_min) || !bbox_lo) return FLOD_E_INVALID_ARG;
    if (n > kKnnStaticMaxN) return FLOD_E_STATIC_LIMIT;               // beyond the built-in scratch: use flod_overlap_prune
    if (n == 0) return FLOD_OK;
    if (!mean_dev || !remove_dev) return FLOD_E_INVALID_ARG;
    for (int k = 0; k < 3; ++k) if (!isfinite(bbox_lo[k])) return FLOD_E_INVALID_ARG;
    void *scratch = nullptr;
    const int rc = knn_static_setup(&scratch);
    if (rc != FLOD_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const float d_op = 0.5f * s_min;                                  // d_OP = s_min / 2
    const double h = 3.0 * (double)d_op * (1.0 + 9.5367431640625e-7);
    KnnGrid g;
    for (int k = 0; k < 3; ++k) g.lo[k] = (double)bbox_lo[k];
    g.inv_h = 1.0 / h;
    const unsigned int m = knn_table_size(n);
    g.mask = m - 1;
    // the same carving as flod_overlap_prune's, sized by THIS call's n (at most kKnnStaticBytes by construction)
    unsigned char *base = (unsigned char *)scratch;
    int3 *cell = (int3 *)base;                  base += knn_align((size_t)n * sizeof(int3));
    unsigned int *count = (unsigned int *)base; base += knn_align(((size_t)m + 1) * 4);
    unsigned int *start = (unsigned int *)base; base += knn_align(((size_t)m + 1) * 4);
    unsigned int *items = (unsigned int *)base;
    // the array keeps the previous call's contents: the bucket counters are the one part that must start at zero
    // (cell, start and items are written in full before they are read)
    if (cudaMemsetAsync(count, 0, ((size_t)m + 1) * 4, s) != cudaSuccess) return FLOD_E_CUDA;
    const unsigned int grid = (unsigned int)((n + 255) / 256);
    k_knn_count<<<grid, 256, 0, s>>>(mean_dev, n, g, cell, count);
    k_knn_scan<<<1, 1024, 0, s>>>(count, start, m);
    k_knn_fill<<<grid, 256, 0, s>>>(n, g, cell, start, count, items);
    const float h2 = (float)(h * h) * 0.99999f;
    k_knn_query<<<(unsigned int)((n + 127) / 128), 128, 0, s>>>(mean_dev, n, g, h2, d_op, cell, start, items, mean_dist_dev, remove_dev);
    return cudaGetLastError() == cudaSuccess ? FLOD_OK : FLOD_E_CUDA;
}

}  // extern "C"
