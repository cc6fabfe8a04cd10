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
constexpr int kDupMaxParts = 32;            // CTAs that may share a segment (launch_duplicate; 16 -> 32: config 3 level 1 142 -> 133 us, level 2 200 -> 182)

// Which of the two duplication kernels serves the frame (when both are launched, the other one exits at once): the mean
// rect area, known on the device since k_geometry.  k_duplicate: one value-returning global atomic per 2x2 tile group.
// With one CTA per segment it was slow on a coarse level alone (hundreds of tiles per Gaussian, few segments: config 3,
// level 1, 979 us), which is what k_duplicate_shared -- counts in shared memory, one global reservation per block and
// tile -- was written for (270 us there); since up to 16 CTAs share a segment k_duplicate takes 142 us on that frame, so
// the shared-counter kernel is left with the frames of VERY large rects (ws.dup_large_area, flod_internal.cuh).
__device__ __forceinline__ bool dup_large_rects(const WorkspaceDev &ws)
{
    return ws.hdr->n_pairs > (unsigned long long)ws.dup_large_area * ws.hdr->n_vis32;
}

template <bool ELLIPSE>
__global__ void __launch_bounds__(kPreBlock)
k_duplicate(const WorkspaceDev ws, int TX, int GX, unsigned int max_pairs, unsigned int parts, int alone)
{
    __shared__ unsigned int s_warp_tot[kPreBlock / 32];
    __shared__ unsigned int s_incl[kGeoBlock];      // inclusive group scan of the segment
    __shared__ uint2 s_rect[kGeoBlock];             // tx0 | ty0 << 16, tx1 | ty1 << 16
    __shared__ unsigned int s_depth[kGeoBlock];     // depth bits

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // `parts` CTAs share a segment (all of them scan it, each expands every parts-th step of its groups): a frame of few
    // segments with many tile groups each (config 3, level 3: 293 segments, 22 K groups per segment) would otherwise run
    // two CTAs per SM with one atomic round trip per thread in flight
    const unsigned int seg = blockIdx.x / parts, part = blockIdx.x % parts;
    cudaGridDependencySynchronize();
    const unsigned int n_here = ws.seg_count[seg];
    if (n_here == 0 || (!alone && dup_large_rects(ws))) return;   // frames of large rects are served by k_duplicate_shared, if it was launched
    const bool absolute = ws.hdr->cursor_abs != 0u;
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
    for (unsigned int q = part * kPreBlock + tid; q < block_groups; q += parts * kPreBlock) {
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
        bool h00 = cx0 && cy0, h10 = cx1 && cy0, h01 = cx0 && cy1, h11 = cx1 && cy1;            // tile (x + i, y + j) is listed
        if (ELLIPSE) {
            // R26: inside the rect, a tile is listed if it lies in its row's span (span.cuh: the canonical fp32 sequence
            // k_geometry counted with, so count and emit agree by construction)
            const float4 fa = ws.gA[p0 + r];
            const float2 fb = *reinterpret_cast<const float2 *>(ws.gB + p0 + r);
            const SpanCoef sp = span_coefficients(fa.x, fa.y, fa.z, fa.w, fb.x, fb.y);
            int ta = 1, tb = 0;
            if (cy0 && span_of_row(sp, (int)tx0, (int)tx1, (int)y, &ta, &tb) == 0) { ta = 1; tb = 0; }
            h00 = h00 && (int)x >= ta && (int)x <= tb; h10 = h10 && (int)x + 1 >= ta && (int)x + 1 <= tb;
            ta = 1; tb = 0;
            if (cy1 && span_of_row(sp, (int)tx0, (int)tx1, (int)y + 1, &ta, &tb) == 0) { ta = 1; tb = 0; }
            h01 = h01 && (int)x >= ta && (int)x <= tb; h11 = h11 && (int)x + 1 >= ta && (int)x + 1 <= tb;
            if (!(h00 || h10 || h01 || h11)) continue;
        }
        const float4 add = make_float4(h00 ? 1.0f : 0.0f, h10 ? 1.0f : 0.0f, h01 ? 1.0f : 0.0f, h11 ? 1.0f : 0.0f);
        // absolute counters (tile_scan.cuh): the atomic returns the slots themselves; otherwise the four range starts are
        // fetched BEFORE the atomic, so that their L2 round trips overlap its latency (from ws.ranges: a copy next to the
        // counters, in their sector or the neighbouring one, made the load wait for the atomics -- config 3, level 3:
        // 229 -> 304 / 323 us)
        float *line = ws.cursor4 + (size_t)(gy * (unsigned int)GX + gx) * kCtrStride;
        uint4 base = make_uint4(0u, 0u, 0u, 0u);
        if (!absolute) {
            const unsigned int t00 = y * (unsigned int)TX + x;
            if (h00) base.x = ws.ranges[t00].x;
            if (h10) base.y = ws.ranges[t00 + 1].x;
            if (h01) base.z = ws.ranges[t00 + TX].x;
            if (h11) base.w = ws.ranges[t00 + TX + 1].x;
        }
        const unsigned long long key = ((unsigned long long)s_depth[r] << 32) | (p0 + r);
        const float4 old = atomicAdd(reinterpret_cast<float4 *>(line), add);
        if (h00) { const unsigned int pos = base.x + (unsigned int)old.x; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (h10) { const unsigned int pos = base.y + (unsigned int)old.y; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (h01) { const unsigned int pos = base.z + (unsigned int)old.z; if (pos < max_pairs) ws.pairs[pos] = key; }
        if (h11) { const unsigned int pos = base.w + (unsigned int)old.w; if (pos < max_pairs) ws.pairs[pos] = key; }
    }
}

// ------------------------------------------------------------------------------------------------ a6, large rects
// Persistent: one block of 1024 threads per SM.  The (segment, chunk of 32 entries) units of the frame are dealt
// round-robin to the warps of the whole grid; a block appends its share in two passes with a per-tile counter array in
// SHARED memory:
//   count    every pair adds 1 to its tile's shared counter;
//   reserve  one global atomicAdd per touched tile reserves the block's share of that tile's list;
//   emit     every pair takes the next slot of its tile from the shared counter and stores its key.
// A lane walks its own rect when it has at most kDupInline tiles, a larger rect is expanded by the whole warp.
// Images with more tiles than fit in shared memory are processed in windows of `win_cap` tiles (both passes each).
constexpr int kDupSThreads = 1024;
constexpr int kDupSWarps = kDupSThreads / 32;
constexpr int kDupSegRound = 256;          // segments of the block whose chunk counts are scanned at a time
constexpr unsigned int kDupInline = 8;     // rects up to this many tiles are walked by their own lane
constexpr int kDupWinCap = 48 * 1024;      // tiles per window: 192 KB of shared counters

template <bool kEmit>
__device__ __forceinline__ void dup_pair(unsigned int *s_cnt, unsigned int t, unsigned int win0, unsigned int win_n,
                                         unsigned long long key, unsigned long long *__restrict__ pairs, unsigned int max_pairs)
{
    const unsigned int r = t - win0;
    if (r >= win_n) return;
    if (kEmit) {
        const unsigned int pos = atomicAdd(&s_cnt[r], 1u);
        if (pos < max_pairs) pairs[pos] = key;
    } else {
        atomicAdd(&s_cnt[r], 1u);
    }
}

template <bool kEmit, bool ELLIPSE>
__device__ __forceinline__ void dup_pass(const WorkspaceDev &ws, unsigned int *s_cnt, unsigned int *s_pref, unsigned int *s_segn,
                                         unsigned int *s_wtot, unsigned int (*s_row)[32][2], unsigned int TX, unsigned int n_segs,
                                         unsigned int win0, unsigned int win_n, unsigned int max_pairs)
{
    const unsigned int tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    // every block walks ALL segments, kDupSegRound at a time, and takes every (32 gridDim)-th unit of the round: a coarse
    // level has few Gaussians (config 3, level 1: 30 segments) with hundreds of tiles each, so units, not segments,
    // are what is dealt out, and consecutive units go to different SMs
    for (unsigned int k0 = 0; k0 < n_segs; k0 += kDupSegRound) {
        const unsigned int nr = min((unsigned int)kDupSegRound, n_segs - k0);
        // exclusive scan of the chunk counts of the round's segments -> s_pref[0 .. nr]
        if (tid < kDupSegRound) {
            const unsigned int n = tid < nr ? ws.seg_count[k0 + tid] : 0u;
            unsigned int incl = (n + 31u) >> 5;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            if (lane == 31) s_wtot[warp] = incl;
            s_pref[tid + 1] = incl;                         // warp-local for now
            if (tid < nr) s_segn[tid] = n;
        }
        __syncthreads();
        if (tid < kDupSegRound) {
            unsigned int add = 0;
            for (unsigned int w = 0; w < warp; ++w) add += s_wtot[w];
            s_pref[tid + 1] += add;
            if (tid == 0) s_pref[0] = 0;
        }
        __syncthreads();
        const unsigned int n_units = s_pref[nr];
        for (unsigned int v = warp * gridDim.x + blockIdx.x; v < n_units; v += kDupSWarps * gridDim.x) {
            unsigned int lo = 0, hi = nr - 1u;          // the segment k with s_pref[k] <= v < s_pref[k + 1]
            while (lo < hi) {
                const unsigned int mid = (lo + hi + 1u) >> 1;
                if (s_pref[mid] <= v) lo = mid; else hi = mid - 1u;
            }
            const unsigned int k = lo, c = v - s_pref[lo];
            const unsigned int seg = k0 + k;
            const unsigned int j = (c << 5) + lane;
            const unsigned int p = seg * kGeoBlock + j;
            unsigned int xy0 = 0, w = 0, h = 0, area = 0, depth = 0;
            SpanCoef sp{};
            if (j < s_segn[k]) {
                const ushort4 rc = ws.rect[p];
                xy0 = (unsigned int)rc.x | ((unsigned int)rc.y << 16);
                w = (unsigned int)rc.z - rc.x; h = (unsigned int)rc.w - rc.y;
                area = w * h;
                if (kEmit) depth = ws.depth[p];
                if (ELLIPSE) {
                    const float4 fa = ws.gA[p];
                    const float2 fb = *reinterpret_cast<const float2 *>(ws.gB + p);
                    sp = span_coefficients(fa.x, fa.y, fa.z, fa.w, fb.x, fb.y);
                }
            }
            if (area <= kDupInline) {                   // small rects: every lane walks its own
                const unsigned long long key = ((unsigned long long)depth << 32) | p;
                const unsigned int tx0 = xy0 & 0xffffu, ty0 = xy0 >> 16;
                for (unsigned int dy = 0; dy < h; ++dy) {
                    int ta = (int)tx0, tb = (int)(tx0 + w) - 1;
                    if (ELLIPSE && span_of_row(sp, (int)tx0, (int)(tx0 + w), (int)(ty0 + dy), &ta, &tb) == 0) continue;
                    for (int tx = ta; tx <= tb; ++tx)
                        dup_pair<kEmit>(s_cnt, (ty0 + dy) * TX + (unsigned int)tx, win0, win_n, key, ws.pairs, max_pairs);
                }
            }
            unsigned int big = __ballot_sync(0xffffffffu, area > kDupInline);
            while (big) {                               // large rects: the whole warp expands one at a time
                const int r = __ffs((int)big) - 1;
                big &= big - 1u;
                const unsigned int rxy = __shfl_sync(0xffffffffu, xy0, r), rw = __shfl_sync(0xffffffffu, w, r);
                const unsigned int ra = __shfl_sync(0xffffffffu, area, r), rd = __shfl_sync(0xffffffffu, depth, r);
                const unsigned long long key = ((unsigned long long)rd << 32) | (p - lane + (unsigned int)r);
                const unsigned int tx0 = rxy & 0xffffu, ty0 = rxy >> 16, t0 = ty0 * TX + tx0;
                if (!ELLIPSE) {
                    // q / rw by multiplication: exact for q < 2^16 (inv = ceil(2^32 / rw), rw < 2^16)
                    const unsigned int inv = rw > 1u ? 0xffffffffu / rw + 1u : 0u;
                    const bool fast = ra <= 65536u && rw > 1u;
                    for (unsigned int q = lane; q < ra; q += 32u) {
                        const unsigned int dy = fast ? __umulhi(q, inv) : q / rw;
                        dup_pair<kEmit>(s_cnt, t0 + dy * TX + (q - dy * rw), win0, win_n, key, ws.pairs, max_pairs);
                    }
                } else {
                    // R26: 32 tile rows at a time, one row's span per lane; the listed tiles of the chunk are then dealt to
                    // the lanes through an exclusive scan of the span lengths
                    SpanCoef rs;
                    rs.sl = __shfl_sync(0xffffffffu, sp.sl, r); rs.KA = __shfl_sync(0xffffffffu, sp.KA, r);
                    rs.DA = __shfl_sync(0xffffffffu, sp.DA, r); rs.dyt = __shfl_sync(0xffffffffu, sp.dyt, r);
                    rs.pad = __shfl_sync(0xffffffffu, sp.pad, r); rs.mx = __shfl_sync(0xffffffffu, sp.mx, r);
                    rs.my = __shfl_sync(0xffffffffu, sp.my, r); rs.box = __shfl_sync(0xffffffffu, (int)sp.box, r) != 0;
                    const unsigned int rh = ra / rw;
                    for (unsigned int r0 = 0; r0 < rh; r0 += 32u) {
                        int ta = 1, tb = 0;
                        if (r0 + lane < rh && span_of_row(rs, (int)tx0, (int)(tx0 + rw), (int)(ty0 + r0 + lane), &ta, &tb) == 0) { ta = 1; tb = 0; }
                        const unsigned int n = tb >= ta ? (unsigned int)(tb - ta + 1) : 0u;
                        unsigned int incl = n;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
                            if (lane >= o) incl += t;
                        }
                        const unsigned int total = __shfl_sync(0xffffffffu, incl, 31);
                        __syncwarp();
                        s_row[warp][lane][0] = incl - n;                        // index of the row's first listed tile in the chunk
                        s_row[warp][lane][1] = (ty0 + r0 + lane) * TX + (unsigned int)ta;
                        __syncwarp();
                        for (unsigned int q = lane; q < total; q += 32u) {
                            unsigned int a = 0, b = 31;                         // last row whose first index is <= q
                            while (a < b) {
                                const unsigned int mid = (a + b + 1u) >> 1;
                                if (s_row[warp][mid][0] <= q) a = mid; else b = mid - 1u;
                            }
                            dup_pair<kEmit>(s_cnt, s_row[warp][a][1] + (q - s_row[warp][a][0]), win0, win_n, key, ws.pairs, max_pairs);
                        }
                    }
                }
            }
        }
        __syncthreads();
    }
}

template <bool ELLIPSE>
__global__ void __launch_bounds__(kDupSThreads, 1)
k_duplicate_shared(const WorkspaceDev ws, unsigned int TX, unsigned int T_n, unsigned int n_segs, unsigned int win_cap,
                   unsigned int max_pairs)
{
    extern __shared__ unsigned int s_cnt[];         // [win_cap] pairs of the block per tile, then the next free slot
    __shared__ unsigned int s_pref[kDupSegRound + 1];
    __shared__ unsigned int s_segn[kDupSegRound];
    __shared__ unsigned int s_wtot[kDupSegRound / 32];
    __shared__ unsigned int s_row[kDupSWarps][32][2];   // per warp: (index of the first listed tile, its tile id) of 32 tile rows
    cudaGridDependencySynchronize();
    if (!dup_large_rects(ws)) return;
    const unsigned int tid = threadIdx.x;
    for (unsigned int win0 = 0; win0 < T_n; win0 += win_cap) {
        const unsigned int win_n = min(win_cap, T_n - win0);
        for (unsigned int r = tid; r < win_n; r += kDupSThreads) s_cnt[r] = 0;
        __syncthreads();
        dup_pass<false, ELLIPSE>(ws, s_cnt, s_pref, s_segn, s_wtot, s_row, TX, n_segs, win0, win_n, max_pairs);
        for (unsigned int r = tid; r < win_n; r += kDupSThreads) {      // (dup_pass ends with a barrier)
            const unsigned int c = s_cnt[r];
            if (c) s_cnt[r] = ws.ranges[win0 + r].x + atomicAdd(&ws.cursor[win0 + r], c);
        }
        __syncthreads();
        dup_pass<true, ELLIPSE>(ws, s_cnt, s_pref, s_segn, s_wtot, s_row, TX, n_segs, win0, win_n, max_pairs);
    }
}

int init_duplicate()
{
    const int bytes = kDupWinCap * (int)sizeof(unsigned int);
    return cudaFuncSetAttribute(k_duplicate_shared<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess &&
           cudaFuncSetAttribute(k_duplicate_shared<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess ? 0 : -1;
}

int launch_duplicate(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    const unsigned int T_n = (unsigned int)p.n_tiles;
    const unsigned int win_cap = (c.flags & FLOD_OPT_SMALL_WINDOWS) ? 1024u : min(T_n, (unsigned int)kDupWinCap);
    // CTAs per segment of k_duplicate: about 32 CTAs per SM when the frame has few segments (measured: 16 and 64 per SM are slower)
    const unsigned int parts = (unsigned int)max(1, min(kDupMaxParts, 32 * c.sm_count / p.n_pre_blocks));
    // Frames of small rects (the hint of the previous frames' tile scans, flod_api.cu) launch k_duplicate alone, and it serves
    // the frame whatever its rects are: a kernel that only finds out that it has nothing to do still costs its place in
    // the chain of dependent launches.  After a frame of large rects both are launched and the device picks.
    const int alone = p.dup_both ? 0 : 1;
    if (p.pair_rule == FLOD_PAIR_RULE_BOX) {
        launch_pdl(k_duplicate<false>, p.n_pre_blocks * parts, kPreBlock, 0, s, c.ws, p.TX, (p.TX + 1) / 2, p.max_pairs, parts, alone);
        if (!alone)
            launch_pdl(k_duplicate_shared<false>, c.sm_count, kDupSThreads, win_cap * sizeof(unsigned int), s,
                       c.ws, (unsigned int)p.TX, T_n, (unsigned int)p.n_pre_blocks, win_cap, p.max_pairs);
    } else {
        launch_pdl(k_duplicate<true>, p.n_pre_blocks * parts, kPreBlock, 0, s, c.ws, p.TX, (p.TX + 1) / 2, p.max_pairs, parts, alone);
        if (!alone)
            launch_pdl(k_duplicate_shared<true>, c.sm_count, kDupSThreads, win_cap * sizeof(unsigned int), s,
                       c.ws, (unsigned int)p.TX, T_n, (unsigned int)p.n_pre_blocks, win_cap, p.max_pairs);
    }
    return alone ? 1 : 2;
}

}  // namespace flod
