// Steps a5-a8: from per-Gaussian tile rects to per-tile lists in (depth, gid) order.
//
// No global sort runs.  The (tile | depth) order of the pairs (R15) is produced by binning + local sorts:
//   k_tile_scan   a5/a8  2-D prefix sum of the difference grid written by k_geometry = pairs per tile; exclusive
//                        scan over the tiles = [start, end) of every tile's list (the ranges of step a8);
//   k_duplicate   a6     every (visible Gaussian, tile of its rect) pair takes the next free slot of ITS TILE's list
//                        (one integer atomic) and stores the 64-bit key (depth bits << 32) | scan index;
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
// Persistent blocks over the visible list, kPreBlock Gaussians per step.  A block scan of the rect areas lets the
// block expand its rects cooperatively, one pair per thread per step, whatever the individual rect sizes.
__global__ void __launch_bounds__(kPreBlock)
k_duplicate(const WorkspaceDev ws, int TX, unsigned int max_pairs)
{
    __shared__ unsigned int s_warp_tot[kPreBlock / 32];
    __shared__ unsigned int s_incl[kPreBlock];      // inclusive pair scan of the step
    __shared__ unsigned int s_rect[kPreBlock];      // tx0 | ty0 << 16
    __shared__ unsigned int s_wd[kPreBlock];        // rect width
    __shared__ unsigned int s_idx[kPreBlock];       // scan index
    __shared__ unsigned int s_depth[kPreBlock];     // depth bits

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int n_vis = ws.hdr->n_vis32;
    for (unsigned int base = blockIdx.x * kPreBlock; base < n_vis; base += gridDim.x * kPreBlock) {
        const unsigned int s = base + tid;
        unsigned int n_tiles = 0;
        if (s < n_vis) {
            const unsigned int i = ws.vis_list[s];
            const ushort4 rc = ws.rect[i];
            const unsigned int w = (unsigned int)rc.z - rc.x;
            n_tiles = w * ((unsigned int)rc.w - rc.y);
            s_idx[tid] = i;
            s_depth[tid] = ws.depth[i];
            s_rect[tid] = (unsigned int)rc.x | ((unsigned int)rc.y << 16);
            s_wd[tid] = w;
        }
        unsigned int incl = n_tiles;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int n = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += n;
        }
        if (lane == 31) s_warp_tot[warp] = incl;
        __syncthreads();
        unsigned int warp_off = 0, block_pairs = 0;
#pragma unroll
        for (int w = 0; w < kPreBlock / 32; ++w) {
            const unsigned int t = s_warp_tot[w];
            if (w < warp) warp_off += t;
            block_pairs += t;
        }
        s_incl[tid] = incl + warp_off;
        __syncthreads();
        const int n_here = (int)min((unsigned int)kPreBlock, n_vis - base);
        for (unsigned int q = tid; q < block_pairs; q += kPreBlock) {
            int lo = 0, hi = n_here - 1;               // first position with s_incl[pos] > q
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
            if (pos < max_pairs) ws.pairs[pos] = ((unsigned long long)s_depth[r] << 32) | s_idx[r];
        }
        __syncthreads();
    }
}

int launch_duplicate(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    const int grid = min(p.n_pre_blocks, c.sm_count * 8);
    k_duplicate<<<grid, kPreBlock, 0, s>>>(c.ws, p.TX, p.max_pairs);
    return 1;
}

}  // namespace flod
