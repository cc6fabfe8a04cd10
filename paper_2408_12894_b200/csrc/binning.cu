// Steps a5-a8: from per-Gaussian tile rects to per-tile lists in (depth, gid) order.
//
// No global sort runs.  The (tile | depth) order of the pairs (R15) is produced by binning + local sorts:
//   (tile scan)   a5/a8  tile_scan.cuh, run by block 0 of k_colour: pairs per tile and every tile's [start, end);
//   k_duplicate   a6     every (visible Gaussian, tile of its rect) pair takes the next free slot of ITS TILE's list
//                        (one float4 atomic per 2x2 group of tiles) and stores the 64-bit key (depth bits << 32) | position;
//   k_tile_sort   a7     (tile_sort.cu) one CTA per tile sorts its list by that key.  The key is unique, so the
//                        result does not depend on the order in which the atomics were served.
#include "flod_internal.cuh"

namespace flod {

// ------------------------------------------------------------------------------------------------ a6
// One block per segment of k_geometry (up to kGeoBlock visible Gaussians, four per thread).  The kernel is bound by the
// throughput of value-returning global atomics on scattered addresses (about 5 cycles per lane and SM, measured:
// profiles/r1h_launches.md), so it issues as few as possible: the append counters of a 2x2 GROUP of tiles are one float4
// and one ATOMG.ADD.F32x4 reserves a slot in each of the (up to four) tiles of the group that the rect covers.  The
// counters are relative to the tile's range start and exact as floats below 2^24 (k_colour's tile scan raises the
// capacity flag for a longer list).  A block scan of the per-Gaussian group counts lets the block expand its rects
// cooperatively, one group per thread per step, whatever the individual rect sizes.
constexpr int kDupPer = kGeoBlock / kPreBlock;

__global__ void __launch_bounds__(kPreBlock)
k_duplicate(const WorkspaceDev ws, int TX, int GX, unsigned int max_pairs)
{
    __shared__ unsigned int s_warp_tot[kPreBlock / 32];
    __shared__ unsigned int s_incl[kGeoBlock];      // inclusive group scan of the segment
    __shared__ uint2 s_rect[kGeoBlock];             // tx0 | ty0 << 16, tx1 | ty1 << 16
    __shared__ unsigned int s_depth[kGeoBlock];     // depth bits

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int seg = blockIdx.x;
    const unsigned int n_here = ws.seg_count[seg];
    if (n_here == 0) return;
    const unsigned int p0 = seg * kGeoBlock;
    // thread t owns entries kDupPer t .. kDupPer t + kDupPer - 1 (consecutive, so that the scan is a plain block scan)
    unsigned int ng[kDupPer], mine = 0;
#pragma unroll
    for (int k = 0; k < kDupPer; ++k) {
        const unsigned int j = tid * kDupPer + k;
        ng[k] = 0;
        if (j < n_here) {
            const ushort4 rc = ws.rect[p0 + j];
            ng[k] = ((((unsigned int)rc.z + 1u) >> 1) - ((unsigned int)rc.x >> 1)) *
                    ((((unsigned int)rc.w + 1u) >> 1) - ((unsigned int)rc.y >> 1));
            s_depth[j] = ws.depth[p0 + j];
            s_rect[j] = make_uint2((unsigned int)rc.x | ((unsigned int)rc.y << 16), (unsigned int)rc.z | ((unsigned int)rc.w << 16));
        }
        mine += ng[k];
    }
    unsigned int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    if (lane == 31) s_warp_tot[warp] = incl;
    __syncthreads();
    unsigned int run = incl - mine, block_groups = 0;
#pragma unroll
    for (int w = 0; w < kPreBlock / 32; ++w) {
        const unsigned int t = s_warp_tot[w];
        if (w < warp) run += t;
        block_groups += t;
    }
#pragma unroll
    for (int k = 0; k < kDupPer; ++k) {
        run += ng[k];
        const unsigned int j = tid * kDupPer + k;
        if (j < n_here) s_incl[j] = run;
    }
    __syncthreads();
    for (unsigned int q = tid; q < block_groups; q += kPreBlock) {
        int lo = 0, hi = (int)n_here - 1;              // first entry with s_incl[entry] > q
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (s_incl[mid] > q) hi = mid; else lo = mid + 1;
        }
        const unsigned int r = (unsigned int)lo;
        const unsigned int k = q - (r ? s_incl[r - 1] : 0u);
        const uint2 rc = s_rect[r];
        const unsigned int tx0 = rc.x & 0xffffu, ty0 = rc.x >> 16, tx1 = rc.y & 0xffffu, ty1 = rc.y >> 16;
        const unsigned int gx0 = tx0 >> 1, gw = ((tx1 + 1u) >> 1) - gx0;
        const unsigned int gy = (ty0 >> 1) + k / gw, gx = gx0 + k % gw;
        const unsigned int x = 2u * gx, y = 2u * gy;
        const bool cx0 = x >= tx0, cx1 = x + 1u < tx1, cy0 = y >= ty0, cy1 = y + 1u < ty1;   // x < tx1 and y < ty1 always hold
        const float4 add = make_float4(cx0 && cy0 ? 1.0f : 0.0f, cx1 && cy0 ? 1.0f : 0.0f,
                                       cx0 && cy1 ? 1.0f : 0.0f, cx1 && cy1 ? 1.0f : 0.0f);
        const float4 old = atomicAdd(reinterpret_cast<float4 *>(ws.cursor4 + (size_t)(gy * (unsigned int)GX + gx) * kCtrStride), add);
        const unsigned long long key = ((unsigned long long)s_depth[r] << 32) | (p0 + r);
        const unsigned int t00 = y * (unsigned int)TX + x;
        if (cx0 && cy0) { const unsigned int pos = ws.ranges[t00].x + (unsigned int)old.x; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (cx1 && cy0) { const unsigned int pos = ws.ranges[t00 + 1].x + (unsigned int)old.y; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (cx0 && cy1) { const unsigned int pos = ws.ranges[t00 + TX].x + (unsigned int)old.z; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (cx1 && cy1) { const unsigned int pos = ws.ranges[t00 + TX + 1].x + (unsigned int)old.w; if (pos < max_pairs) ws.pairs[pos] = key; }
    }
}

int launch_duplicate(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    k_duplicate<<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.ws, p.TX, (p.TX + 1) / 2, p.max_pairs);
    return 1;
}

}  // namespace flod
