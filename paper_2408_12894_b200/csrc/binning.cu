// Steps a5-a8: from per-Gaussian tile rects to per-tile lists in (depth, gid) order.
//
// No global sort runs.  The (tile | depth) order of the pairs (R15) is produced by binning + local sorts:
//   k_tile_scan   a5/a8  2-D prefix sum of the difference grid written by k_geometry = pairs per tile; exclusive
//                        scan over the tiles = [start, end) of every tile's list (the ranges of step a8);
//   k_duplicate   a6     every (visible Gaussian, tile of its rect) pair takes the next free slot of ITS TILE's list
//                        (one integer atomic) and stores the 64-bit key (depth bits << 32) | scan index;
//   k_tile_sort   a7     one CTA per tile sorts its list by that key in shared memory (bitonic network).  The key is
//                        unique, so the result does not depend on the order in which the atomics were served.
// Lists longer than kSortCap keys are consumed in rounds: a 256-bin histogram (refined until it resolves) picks the
// largest key threshold below which at most kSortCap unsorted keys lie; those are gathered, sorted and written out.
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

// ------------------------------------------------------------------------------------------------ a7
constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortMaxBins = 512;
constexpr int kSortRounds = kSortCap / kSortThreads;      // ranking rounds of a warp: its keys / 32
static_assert(kSortCap % (kSortThreads * 1) == 0, "kSortCap must be a multiple of the block size");

struct SortSmem {
    unsigned long long keys[2][kSortCap];                 // ping-pong
    unsigned int whist[kSortWarps][kSortMaxBins];         // per-warp digit counters -> exclusive offsets across warps
    unsigned int binstart[kSortMaxBins];
    unsigned int hist[256];                               // long lists: selection histogram
    unsigned int wsum[kSortWarps];
    unsigned int red[2][kSortWarps];
    unsigned int count;
    unsigned int flag;
    unsigned long long bcast[2];
    unsigned long long red64[kSortWarps];
};

// Ascending bitonic sort of s[0, n_pad), n_pad a power of two >= 2, by the whole block (fallback path).
__device__ __forceinline__ void bitonic_sort(unsigned long long *s, unsigned int n_pad, int tid)
{
    for (unsigned int k = 2; k <= n_pad; k <<= 1) {
        for (unsigned int j = k >> 1; j > 0; j >>= 1) {
            for (unsigned int t = tid; t < (n_pad >> 1); t += kSortThreads) {
                const unsigned int ix = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const unsigned int iy = ix | j;
                const unsigned long long a = s[ix], b = s[iy];
                const bool up = (ix & k) == 0;
                if ((a > b) == up) { s[ix] = b; s[iy] = a; }
            }
            __syncthreads();
        }
    }
}

__device__ __forceinline__ unsigned int next_pow2(unsigned int v)
{
    return v <= 2 ? 2u : 1u << (32 - __clz(v - 1));
}

// Block-wide min / max of the depth words; every thread gets the result.  Ends with a barrier.
__device__ __forceinline__ void block_minmax(SortSmem &S, unsigned int &dmin, unsigned int &dmax, int lane, int warp)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dmin = min(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
        dmax = max(dmax, __shfl_xor_sync(0xffffffffu, dmax, o));
    }
    if (lane == 0) { S.red[0][warp] = dmin; S.red[1][warp] = dmax; }
    __syncthreads();
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) { dmin = min(dmin, S.red[0][w]); dmax = max(dmax, S.red[1][w]); }
    __syncthreads();
}

// Sorts the n <= kSortCap unique 64-bit keys (depth bits << 32 | index) held in S.keys[0][0, n) and returns the
// sorted array.  Stable LSD radix passes over the bits in which the depth words differ (8 or 9 bits per pass; a warp
// ranks a contiguous chunk with match_any, per-warp digit counters make it stable), then runs of equal depth, which
// the passes leave in arrival order, are put in index order (insertion by the run's first thread; runs are short --
// a list with a run longer than 32 falls back to a bitonic network on the whole 64-bit keys).
__device__ unsigned long long *block_sort(SortSmem &S, unsigned int n, unsigned int dmin, unsigned int dmax, int tid)
{
    const int lane = tid & 31, warp = tid >> 5;
    const int bits = 32 - __clz(dmax - dmin);                         // 0 when all depths are equal
    const int dbits = (bits > 24 && bits <= 27) ? 9 : 8;
    const int passes = (bits + dbits - 1) / dbits;
    const unsigned int bins = 1u << dbits, dmask = bins - 1;
    const int bpt = (int)(bins / kSortThreads);                       // bins per thread in the scan: 1 or 2
    const unsigned int per_warp = (n + kSortThreads - 1) / kSortThreads * 32;   // keys per warp, a multiple of 32
    int cur = 0;
    for (int pass = 0; pass < passes; ++pass) {
        const unsigned long long *src = S.keys[cur];
        unsigned long long *dst = S.keys[cur ^ 1];
        const int shift = pass * dbits;
        for (unsigned int i = tid; i < kSortWarps * bins; i += kSortThreads) S.whist[i / bins][i % bins] = 0;
        __syncthreads();
        // ---- rank inside the warp's chunk, stable
        unsigned long long key[kSortRounds];
        unsigned short rnk[kSortRounds];
        unsigned int *wh = S.whist[warp];
#pragma unroll
        for (int r = 0; r < kSortRounds; ++r) {
            if ((unsigned int)r * 32 < per_warp) {
                const unsigned int j = warp * per_warp + r * 32 + lane;
                const bool ok = j < n;
                const unsigned int vm = __ballot_sync(0xffffffffu, ok);
                if (ok) {
                    key[r] = src[j];
                    const unsigned int d = (((unsigned int)(key[r] >> 32) - dmin) >> shift) & dmask;
                    const unsigned int peers = __match_any_sync(vm, d);
                    const unsigned int leader = __ffs(peers) - 1;
                    unsigned int old = 0;
                    if (lane == leader) { old = wh[d]; wh[d] = old + __popc(peers); }
                    old = __shfl_sync(peers, old, leader);
                    rnk[r] = (unsigned short)(old + __popc(peers & ((1u << lane) - 1)));
                }
                __syncwarp();
            }
        }
        __syncthreads();
        // ---- per bin: exclusive scan across warps; then exclusive scan across bins
        {
            unsigned int tot[2] = {0, 0};
            for (int q = 0; q < bpt; ++q) {
                const unsigned int b = tid * bpt + q;
                unsigned int run = 0;
#pragma unroll
                for (int w = 0; w < kSortWarps; ++w) { const unsigned int t = S.whist[w][b]; S.whist[w][b] = run; run += t; }
                tot[q] = run;
            }
            const unsigned int mine = tot[0] + tot[1];
            unsigned int incl = mine;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += t;
            }
            if (lane == 31) S.wsum[warp] = incl;
            __syncthreads();
            unsigned int excl = incl - mine;
#pragma unroll
            for (int w = 0; w < kSortWarps; ++w) if (w < warp) excl += S.wsum[w];
            S.binstart[tid * bpt] = excl;
            if (bpt == 2) S.binstart[tid * bpt + 1] = excl + tot[0];
        }
        __syncthreads();
        // ---- scatter
#pragma unroll
        for (int r = 0; r < kSortRounds; ++r) {
            if ((unsigned int)r * 32 < per_warp) {
                const unsigned int j = warp * per_warp + r * 32 + lane;
                if (j < n) {
                    const unsigned int d = (((unsigned int)(key[r] >> 32) - dmin) >> shift) & dmask;
                    dst[S.binstart[d] + wh[d] + rnk[r]] = key[r];
                }
            }
        }
        __syncthreads();
        cur ^= 1;
    }
    // ---- equal-depth runs -> index order
    unsigned long long *arr = S.keys[cur];
    bool big = false;
    for (unsigned int j = tid; j + 1 < n; j += kSortThreads) {
        const unsigned int dj = (unsigned int)(arr[j] >> 32);
        if (dj == (unsigned int)(arr[j + 1] >> 32) && (j == 0 || (unsigned int)(arr[j - 1] >> 32) != dj)) {
            unsigned int e = j + 2;
            while (e < n && (unsigned int)(arr[e] >> 32) == dj && e - j <= 32) ++e;
            if (e - j > 32) { big = true; continue; }
            for (unsigned int a = j + 1; a < e; ++a) {          // insertion sort of arr[j, e)
                const unsigned long long k = arr[a];
                unsigned int b = a;
                while (b > j && arr[b - 1] > k) { arr[b] = arr[b - 1]; --b; }
                arr[b] = k;
            }
        }
    }
    if (__syncthreads_or(big)) {
        const unsigned int n_pad = next_pow2(n);
        for (unsigned int j = n + tid; j < n_pad; j += kSortThreads) arr[j] = ~0ull;
        __syncthreads();
        bitonic_sort(arr, n_pad, tid);
    }
    return arr;
}

__global__ void __launch_bounds__(kSortThreads)
k_tile_sort(const WorkspaceDev ws, int n_tiles)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem &S = *reinterpret_cast<SortSmem *>(smem_raw);

    const int tile = blockIdx.x;
    if (tile >= n_tiles) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint2 rg = ws.ranges[tile];
    const unsigned int L = rg.y - rg.x;
    if (L == 0 || ws.hdr->overflow) return;            // an overflowed frame is undefined (and its keys need not be unique)
    const unsigned long long *__restrict__ pairs = ws.pairs + rg.x;
    uint32_t *__restrict__ vals = ws.vals + rg.x;

    if (L <= kSortCap) {
        unsigned int dmin = 0xffffffffu, dmax = 0;
        for (unsigned int j = tid; j < L; j += kSortThreads) {
            const unsigned long long k = pairs[j];
            S.keys[0][j] = k;
            dmin = min(dmin, (unsigned int)(k >> 32)); dmax = max(dmax, (unsigned int)(k >> 32));
        }
        block_minmax(S, dmin, dmax, lane, warp);
        const unsigned long long *arr = block_sort(S, L, dmin, dmax, tid);
        for (unsigned int j = tid; j < L; j += kSortThreads) vals[j] = (uint32_t)arr[j];
        return;
    }

    // ---- long list: rounds of (select the next <= kSortCap smallest keys, gather, sort, write out)
    unsigned long long kmax = 0;
    for (unsigned int j = tid; j < L; j += kSortThreads) kmax = max(kmax, pairs[j]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    if (lane == 0) S.red64[warp] = kmax;
    __syncthreads();
    kmax = 0;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) kmax = max(kmax, S.red64[w]);

    unsigned long long lo = 0;                         // every key < lo has been written out
    unsigned int out = 0;
    while (out < L) {
        unsigned long long hi = kmax;                  // inclusive
        if (L - out > kSortCap) {
            // refine [a, b] with 256 power-of-two-wide bins until at least 3/4 of the budget is used or bins are
            // single keys; keys are unique, so a range of w keys holds at most w entries and the loop ends
            unsigned long long a = lo, b = kmax;
            unsigned int budget = kSortCap;
            while (true) {
                const unsigned long long width = b - a;                  // b - a + 1 keys; both < 2^63
                const int sh = max(0, 64 - __clzll(width) - 8);          // (b - a) >> sh < 256
                __syncthreads();
                S.hist[tid] = 0;
                __syncthreads();
                for (unsigned int j = tid; j < L; j += kSortThreads) {
                    const unsigned long long k = pairs[j];
                    if (k >= a && k <= b) atomicAdd(&S.hist[(unsigned int)((k - a) >> sh)], 1u);
                }
                __syncthreads();
                if (tid == 0) {
                    unsigned int cum = 0, m = 0;
                    while (m < 256 && cum + S.hist[m] <= budget) { cum += S.hist[m]; ++m; }
                    S.bcast[0] = m; S.bcast[1] = cum;
                }
                __syncthreads();
                const unsigned int m = (unsigned int)S.bcast[0], cum = (unsigned int)S.bcast[1];
                if (m == 256) { hi = b; break; }
                budget -= cum;
                const unsigned long long edge = a + ((unsigned long long)m << sh);   // first key of the bin that overflows
                if (sh == 0 || budget < kSortCap / 4) { hi = edge - 1; break; }      // edge > lo: see below
                a = edge;
                b = min(b, edge + ((1ull << sh) - 1));
            }
        }
        // (hi >= lo always: with sh == 0 a bin holds at most one key, so the first bin of [a, b] fits the budget
        //  unless the budget is 0, which only happens after a round of refinement accepted keys below `edge`.)
        if (tid == 0) S.count = 0;
        __syncthreads();
        unsigned int dmin = 0xffffffffu, dmax = 0;
        for (unsigned int j0 = 0; j0 < L; j0 += kSortThreads) {
            const unsigned int j = j0 + tid;
            const unsigned long long k = j < L ? pairs[j] : 0ull;
            const bool take = j < L && k >= lo && k <= hi;
            const unsigned int bal = __ballot_sync(0xffffffffu, take);
            unsigned int wbase = 0;
            if (lane == 0 && bal) wbase = atomicAdd(&S.count, __popc(bal));
            wbase = __shfl_sync(0xffffffffu, wbase, 0);
            if (take) {
                S.keys[0][wbase + __popc(bal & ((1u << lane) - 1))] = k;
                dmin = min(dmin, (unsigned int)(k >> 32)); dmax = max(dmax, (unsigned int)(k >> 32));
            }
        }
        block_minmax(S, dmin, dmax, lane, warp);
        const unsigned int n = S.count;
        if (n == 0) break;                             // cannot happen with unique keys; never spin
        const unsigned long long *arr = block_sort(S, n, dmin, dmax, tid);
        for (unsigned int j = tid; j < n; j += kSortThreads) vals[out + j] = (uint32_t)arr[j];
        out += n;
        lo = hi + 1;
        __syncthreads();
    }
}

int launch_tile_sort(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_tile_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem));
        attr_set = true;
    }
    k_tile_sort<<<p.n_tiles, kSortThreads, sizeof(SortSmem), s>>>(c.ws, p.n_tiles);
    return 1;
}

}  // namespace flod
