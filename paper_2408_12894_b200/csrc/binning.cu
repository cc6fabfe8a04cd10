// Steps a5-a8: from per-Gaussian tile rects to per-tile lists in (depth, gid) order.
//
// No global sort runs.  The (tile | depth) order of the pairs (R15) is produced by binning + local sorts:
//   k_tile_scan   a5/a8  2-D prefix sum of the difference grid written by k_geometry = pairs per tile; exclusive
//                        scan over the tiles = [start, end) of every tile's list (the ranges of step a8);
//   k_duplicate   a6     every (visible Gaussian, tile of its rect) pair takes the next free slot of ITS TILE's list
//                        (one integer atomic) and stores the 64-bit key (depth bits << 32) | position;
//   k_tile_sort   a7     (tile_sort.cu) one CTA per tile sorts its list by that key.  The key is unique, so the
//                        result does not depend on the order in which the atomics were served.
#include "flod_internal.cuh"

namespace flod {

// ------------------------------------------------------------------------------------------------ a5 / a8
// One block.  grid = (TX+1) x (TY+1) ints, in shared memory when it fits, else in global memory (ws.tile_cnt).
__global__ void __launch_bounds__(1024)
k_tile_scan(const WorkspaceDev ws, int TX, int TY, unsigned int max_pairs, int use_smem)
{
    extern __shared__ int s_grid[];
    __shared__ unsigned long long s_part[1024];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int gw = TX + 1, gh = TY + 1, gn = gw * gh;
    int *grid = use_smem ? s_grid : ws.tile_cnt;
    for (int i = tid; i < gn; i += nthr) grid[i] = ws.tile_diff[(size_t)i * kCtrStride];
    __syncthreads();
    for (int y = tid; y < gh; y += nthr) {           // prefix along x
        int run = 0;
        int *row = grid + y * gw;
        for (int x = 0; x < gw; ++x) { run += row[x]; row[x] = run; }
    }
    __syncthreads();
    for (int x = tid; x < gw; x += nthr) {           // prefix along y: grid[y][x] = pairs of tile (x, y)
        int run = 0;
        for (int y = 0; y < gh; ++y) { run += grid[y * gw + x]; grid[y * gw + x] = run; }
    }
    __syncthreads();
    // exclusive scan over the tiles in row-major order; a thread owns a contiguous chunk
    const int T_n = TX * TY;
    const int per = (T_n + nthr - 1) / nthr;
    const int t0 = min(tid * per, T_n), t1 = min(t0 + per, T_n);
    unsigned long long sum = 0;
    for (int t = t0; t < t1; ++t) sum += (unsigned int)grid[(t / TX) * gw + (t % TX)];
    s_part[tid] = sum;
    __syncthreads();
    for (int o = 1; o < nthr; o <<= 1) {             // Hillis-Steele inclusive scan of the partials
        unsigned long long v = tid >= o ? s_part[tid - o] : 0ull;
        __syncthreads();
        s_part[tid] += v;
        __syncthreads();
    }
    unsigned long long run = s_part[tid] - sum;
    for (int t = t0; t < t1; ++t) {
        const unsigned int c = (unsigned int)grid[(t / TX) * gw + (t % TX)];
        const unsigned int a = (unsigned int)min(run, (unsigned long long)max_pairs);
        const unsigned int b = (unsigned int)min(run + c, (unsigned long long)max_pairs);
        ws.ranges[t] = make_uint2(a, b);
        ws.cursor[(size_t)t * kCtrStride] = a;
        run += c;
    }
    if (tid == nthr - 1) {
        const unsigned long long total = s_part[tid];
        ws.hdr->n_pairs_clamped = (unsigned int)min(total, (unsigned long long)max_pairs);
        ws.hdr->overflow = total > max_pairs ? 1u : 0u;
    }
}

int launch_tile_scan(const Context &c, const FrameParams &p, cudaStream_t s)
{
    const size_t bytes = (size_t)(p.TX + 1) * (p.TY + 1) * sizeof(int);
    const bool use_smem = bytes <= 200 * 1024;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_tile_scan, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        attr_set = true;
    }
    k_tile_scan<<<1, 1024, use_smem ? bytes : 0, s>>>(c.ws, p.TX, p.TY, p.max_pairs, use_smem ? 1 : 0);
    return 1;
}

// ------------------------------------------------------------------------------------------------ a6
// One block per segment of k_geometry (up to kGeoBlock visible Gaussians, four per thread).  A block scan of the rect
// areas lets the block expand its rects cooperatively, one pair per thread per step, whatever the individual sizes.
constexpr int kDupPer = kGeoBlock / kPreBlock;

__global__ void __launch_bounds__(kPreBlock)
k_duplicate(const WorkspaceDev ws, int TX, unsigned int max_pairs)
{
    __shared__ unsigned int s_warp_tot[kPreBlock / 32];
    __shared__ unsigned int s_incl[kGeoBlock];      // inclusive pair scan of the segment
    __shared__ unsigned int s_rect[kGeoBlock];      // tx0 | ty0 << 16
    __shared__ unsigned int s_wd[kGeoBlock];        // rect width
    __shared__ unsigned int s_depth[kGeoBlock];     // depth bits

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int seg = blockIdx.x;
    const unsigned int n_here = ws.seg_count[seg];
    if (n_here == 0) return;
    const unsigned int p0 = seg * kGeoBlock;
    // thread t owns entries kDupPer t .. kDupPer t + kDupPer - 1 (consecutive, so that the scan is a plain block scan)
    unsigned int nt[kDupPer], mine = 0;
#pragma unroll
    for (int k = 0; k < kDupPer; ++k) {
        const unsigned int j = tid * kDupPer + k;
        nt[k] = 0;
        if (j < n_here) {
            const ushort4 rc = ws.rect[p0 + j];
            const unsigned int w = (unsigned int)rc.z - rc.x;
            nt[k] = w * ((unsigned int)rc.w - rc.y);
            s_depth[j] = ws.depth[p0 + j];
            s_rect[j] = (unsigned int)rc.x | ((unsigned int)rc.y << 16);
            s_wd[j] = w;
        }
        mine += nt[k];
    }
    unsigned int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    if (lane == 31) s_warp_tot[warp] = incl;
    __syncthreads();
    unsigned int run = incl - mine, block_pairs = 0;
#pragma unroll
    for (int w = 0; w < kPreBlock / 32; ++w) {
        const unsigned int t = s_warp_tot[w];
        if (w < warp) run += t;
        block_pairs += t;
    }
#pragma unroll
    for (int k = 0; k < kDupPer; ++k) {
        run += nt[k];
        const unsigned int j = tid * kDupPer + k;
        if (j < n_here) s_incl[j] = run;
    }
    __syncthreads();
    for (unsigned int q = tid; q < block_pairs; q += kPreBlock) {
        int lo = 0, hi = (int)n_here - 1;              // first entry with s_incl[entry] > q
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (s_incl[mid] > q) hi = mid; else lo = mid + 1;
        }
        const unsigned int r = (unsigned int)lo;
        const unsigned int k = q - (r ? s_incl[r - 1] : 0u);
        const unsigned int w = s_wd[r];
        const unsigned int ry = k / w, rx = k - ry * w;
        const unsigned int rc = s_rect[r];
        const unsigned int tile = ((rc >> 16) + ry) * (unsigned int)TX + ((rc & 0xffffu) + rx);
        const unsigned int pos = atomicAdd(ws.cursor + (size_t)tile * kCtrStride, 1u);
        if (pos < max_pairs) ws.pairs[pos] = ((unsigned long long)s_depth[r] << 32) | (p0 + r);
    }
}

int launch_duplicate(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    k_duplicate<<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.ws, p.TX, p.max_pairs);
    return 1;
}

}  // namespace flod
