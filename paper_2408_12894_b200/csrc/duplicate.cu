// Steps a5-a6: exclusive scan of the tile counts and tile-keyed duplication, IN DEPTH ORDER.
//
// Input: the visible Gaussians sorted by (depth, gid) (sort.cu, depth passes).  One thread per sorted position
// reads its Gaussian's tile rect; a block scan plus a decoupled look-back over blocks (ordered by an atomic ticket)
// gives every block its pair base; the block then expands its rects cooperatively, one pair per thread per step
// with perfectly coalesced stores: key = tile id (row-major inside the rect), value = compact Gaussian index.
// Because pairs leave in (depth, gid) order, a STABLE sort by tile id alone yields the (tile, depth, gid) order.
#include "flod_internal.cuh"

namespace flod {

constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagIncl = 2ull << 62, kFlagMask = 3ull << 62;

template <typename KeyT>
__global__ void __launch_bounds__(kPreBlock)
k_duplicate(const WorkspaceDev ws, int depth_buf, int TX, unsigned int max_pairs)
{
    __shared__ unsigned int s_vb;
    __shared__ unsigned int s_warp_tot[kPreBlock / 32];
    __shared__ unsigned long long s_base;
    __shared__ unsigned int s_incl[kPreBlock];      // inclusive pair scan of the block
    __shared__ unsigned int s_rect[kPreBlock];      // tx0 | ty0 << 16
    __shared__ unsigned int s_wd[kPreBlock];        // rect width
    __shared__ unsigned int s_ci[kPreBlock];        // compact index

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_vb = atomicAdd(&ws.hdr->dup_ticket, 1u);
    __syncthreads();
    const unsigned int vb = s_vb;
    const unsigned int n_vis = ws.hdr->n_vis32;
    if (vb * kPreBlock >= n_vis) return;
    const unsigned int s = vb * kPreBlock + tid;

    unsigned int n_tiles = 0;
    if (s < n_vis) {
        const unsigned int ci = ws.dvals[depth_buf][s];
        const ushort4 rc = ws.rect[ci];
        const unsigned int w = (unsigned int)rc.z - rc.x;
        n_tiles = w * ((unsigned int)rc.w - rc.y);
        s_ci[tid] = ci;
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

    // ---- decoupled look-back over the blocks before this one (warp 0); words [2 b + 1] of scan_status
    if (warp == 0) {
        unsigned long long *status = ws.scan_status + 1;
        const unsigned long long agg = block_pairs;
        unsigned long long excl = 0;
        if (vb == 0) {
            if (lane == 0) atomicExch(status, kFlagIncl | agg);
        } else {
            if (lane == 0) atomicExch(status + 2 * (size_t)vb, kFlagAgg | agg);
            long long j = (long long)vb - 1;
            while (true) {
                const long long idx = j - lane;
                unsigned long long st = kFlagIncl;
                if (idx >= 0) {
                    volatile unsigned long long *ptr = status + 2 * (size_t)idx;
                    do { st = *ptr; } while ((st & kFlagMask) == 0);
                }
                const unsigned int incl_mask = __ballot_sync(0xffffffffu, (st & kFlagMask) == kFlagIncl);
                const unsigned long long val = st & ~kFlagMask;
                const int first = incl_mask ? (__ffs(incl_mask) - 1) : 31;
                unsigned long long contrib = (lane <= first) ? val : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
                excl += contrib;
                if (incl_mask) break;
                j -= 32;
            }
            if (lane == 0) atomicExch(status + 2 * (size_t)vb, kFlagIncl | (excl + agg));
        }
        if (lane == 0) s_base = excl;
    }
    __syncthreads();
    const unsigned long long pair_base = s_base;
    const int n_here = (int)min((unsigned int)kPreBlock, n_vis - vb * kPreBlock);

    // ---- a6: block-cooperative expansion, one pair per thread per step, coalesced stores
    KeyT *__restrict__ keys = reinterpret_cast<KeyT *>(ws.tkeys[0]);
    uint32_t *__restrict__ vals = ws.vals[0];
    for (unsigned int q = tid; q < block_pairs; q += kPreBlock) {
        int lo = 0, hi = n_here - 1;                   // first position with s_incl[pos] > q
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (s_incl[mid] > q) hi = mid; else lo = mid + 1;
        }
        const unsigned int r = (unsigned int)lo;
        const unsigned int start = r ? s_incl[r - 1] : 0u;
        const unsigned int k = q - start;
        const unsigned int w = s_wd[r];
        const unsigned int ry = k / w, rx = k - ry * w;
        const unsigned int rc = s_rect[r];
        const unsigned int tile = ((rc >> 16) + ry) * (unsigned int)TX + ((rc & 0xffffu) + rx);
        const unsigned long long dst = pair_base + q;
        if (dst < max_pairs) {
            keys[dst] = (KeyT)tile;
            vals[dst] = s_ci[r];
        }
    }
}

int launch_duplicate(const Context &c, const FrameParams &p, int depth_buf, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    if (tile_sort_plan(p.n_tiles).wide)
        k_duplicate<uint32_t><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.ws, depth_buf, p.TX, p.max_pairs);
    else
        k_duplicate<uint16_t><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.ws, depth_buf, p.TX, p.max_pairs);
    return 1;
}

}  // namespace flod
