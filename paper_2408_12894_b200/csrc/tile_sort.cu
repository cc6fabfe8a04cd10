// Step a7: every tile's pair list into (depth, gid) order ("in depth order"; R15).
//
// One CTA per tile.  The list holds unique 64-bit keys (depth bits << 32) | compact index, in the arbitrary order in
// which k_duplicate's atomics were served.  It is sorted most-significant-digit first, without any stable ranking:
//   bin pass   min / max of the keys -> bins of power-of-two width over [kmin, kmax] (at most 2048, about one key
//              per bin) -> histogram with shared-memory atomics -> exclusive scan -> scatter with a second atomic.
//              Bins are now in key order, keys inside a bin are not.
//   rank pass  one thread per key counts the keys of its own bin that are smaller (a bin holds a few keys): that is
//              its final position.  The 32-bit compact index is written to ws.vals.
// A bin with more than kRankMax keys (a cluster of nearly equal depths) is binned once more over its own key range
// (level 2, through global memory); what is still oversized after that is ranked by the whole block.
// Lists of up to kSortCap keys are scattered into shared memory, longer ones into ws.pairs_tmp (global, L2).
// Because the keys are unique the result is the unique sorted sequence whatever the atomics did.
#include "flod_internal.cuh"

namespace flod {

constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSortBinsLog = 11;
constexpr int kSortBins = 1 << kSortBinsLog;
constexpr int kSortKeysPerBinLog = 1;                     // about two keys per bin
constexpr int kSortSliceLog = 10;                         // depth slices of long lists: 512-1024 keys
constexpr int kCoarseBinsLog = 8;
static_assert(kCoarseBins == 1 << kCoarseBinsLog, "slices per long list");
constexpr unsigned int kLazyFirst = 1024;                 // LAZY: keys of a long list that are sorted before the blend starts
constexpr unsigned int kRankMax = 64;                     // bins up to this size are finished by per-key rank counting

typedef unsigned long long u64;

struct SortSmem {
    u64 keys[kSortCap];                                   // level-1 scatter target of lists up to kSortCap keys
    unsigned int ends[2][kSortBins];                      // per level: bin cursors; after the scatter, bin ends
    u64 red_min[kSortWarps], red_max[kSortWarps];
    unsigned int red_u[kSortWarps];
    unsigned int wsum[kSortWarps];
    unsigned int any_big[2];                              // per level: some bin exceeded kRankMax (set by rank_small)
    unsigned int cends[kCoarseBins];                      // lists longer than kSortCap: ends of the coarse depth slices
};

struct BinMap { u64 kmin; int shift; unsigned int nb; };

__device__ __forceinline__ unsigned int bin_of(const BinMap &m, u64 k) { return (unsigned int)((k - m.kmin) >> m.shift); }

// Block-wide minimum of v (every thread gets it).  Two barriers.
__device__ __forceinline__ unsigned int block_min_u32(SortSmem &S, unsigned int v, int tid)
{
    v = __reduce_min_sync(0xffffffffu, v);
    if ((tid & 31) == 0) S.red_u[tid >> 5] = v;
    __syncthreads();
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) v = min(v, S.red_u[w]);
    __syncthreads();
    return v;
}

constexpr int kSortU = 6;                  // keys a thread holds in registers / loads in flight per step

// f(key) for src[from .. n) strided over the block, kSortU independent loads in flight per thread and step.
template <class F>
__device__ __forceinline__ void for_keys(const u64 *src, unsigned int from, unsigned int n, int tid, F f)
{
    for (unsigned int j0 = from + tid; j0 < n; j0 += kSortU * kSortThreads) {
        u64 k[kSortU];
#pragma unroll
        for (int i = 0; i < kSortU; ++i) { const unsigned int j = j0 + i * kSortThreads; k[i] = j < n ? src[j] : 0ull; }
#pragma unroll
        for (int i = 0; i < kSortU; ++i) if (j0 + i * kSortThreads < n) f(k[i]);
    }
}

// Distributes src[0, n) into dst[0, n) by bin (src and dst must not overlap).  On return ends[b] is the exclusive end
// of bin b in dst (its start is ends[b-1], 0 for b = 0), and all writes are visible to the block.
__device__ BinMap bin_pass(const u64 *src, u64 *dst, unsigned int n, unsigned int *ends, SortSmem &S, int tid,
                           int per_bin_log = kSortKeysPerBinLog, int min_bins_log = 6, int max_bins_log = kSortBinsLog)
{
    const int lane = tid & 31, warp = tid >> 5;
    // the first kSortU * kSortThreads keys (the whole list of an average tile) stay in registers over the three passes
    u64 r[kSortU];
#pragma unroll
    for (int i = 0; i < kSortU; ++i) { const unsigned int j = tid + i * kSortThreads; r[i] = j < n ? src[j] : 0ull; }
    auto each = [&](auto f) {
#pragma unroll
        for (int i = 0; i < kSortU; ++i) if (tid + i * kSortThreads < n) f(r[i]);
        for_keys(src, kSortU * kSortThreads, n, tid, f);
    };
    u64 kmin = ~0ull, kmax = 0ull;
    each([&](u64 k) { kmin = min(kmin, k); kmax = max(kmax, k); });
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
        kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    }
    if (lane == 0) { S.red_min[warp] = kmin; S.red_max[warp] = kmax; }
    __syncthreads();
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) { kmin = min(kmin, S.red_min[w]); kmax = max(kmax, S.red_max[w]); }
    BinMap m;
    m.kmin = kmin;
    const u64 range = kmax - kmin;
    const int bits = range ? 64 - __clzll(range) : 0;
    const int want = min(max_bins_log, max(min_bins_log, 32 - per_bin_log - __clz(max(n, 2u) - 1)));   // about 2^per_bin_log keys per bin
    m.shift = max(0, bits - want);
    m.nb = (unsigned int)(range >> m.shift) + 1u;                                  // <= 2^want
    for (unsigned int b = tid; b < m.nb; b += kSortThreads) ends[b] = 0;
    __syncthreads();
    each([&](u64 k) { atomicAdd(&ends[bin_of(m, k)], 1u); });
    __syncthreads();
    // exclusive scan of ends[0, nb): a thread owns ipt consecutive bins
    {
        const unsigned int ipt = (m.nb + kSortThreads - 1) / kSortThreads;
        const unsigned int b0 = min(tid * ipt, m.nb), b1 = min(b0 + ipt, m.nb);
        unsigned int sum = 0;
        for (unsigned int b = b0; b < b1; ++b) sum += ends[b];
        unsigned int incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) S.wsum[warp] = incl;
        __syncthreads();
        unsigned int run = incl - sum;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) if (w < warp) run += S.wsum[w];
        for (unsigned int b = b0; b < b1; ++b) { const unsigned int c = ends[b]; ends[b] = run; run += c; }
    }
    __syncthreads();
    // (keeping the arrival rank that a value-returning histogram atomic would give, to save this second atomic,
    // measured 9 us slower on config 1: it needs a rank array, two more barriers and a pass that turns bin starts into
    // bin ends, and with about five keys per thread the fixed cost per tile is what counts)
    each([&](u64 k) { dst[atomicAdd(&ends[bin_of(m, k)], 1u)] = k; });
    __syncthreads();
    return m;
}

// Final positions of the keys that sit in bins of at most kRankMax keys: position = bin start + number of smaller
// keys in the bin.  buf[0, n) is the output of bin_pass; the compact indices go to out[0, n).
__device__ __forceinline__ void rank_small(const u64 *buf, unsigned int n, const unsigned int *ends, const BinMap &m,
                                           uint32_t *__restrict__ out, unsigned int *any_big, int tid)
{
    for (unsigned int p = tid; p < n; p += kSortThreads) {
        const u64 k = buf[p];
        const unsigned int b = bin_of(m, k);
        const unsigned int lo = b ? ends[b - 1] : 0u, hi = ends[b];
        if (hi - lo > kRankMax) { *any_big = 1u; continue; }
        unsigned int cnt = 0;
        for (unsigned int q = lo; q < hi; ++q) cnt += buf[q] < k ? 1u : 0u;
        out[lo + cnt] = (uint32_t)k;
    }
}

// Smallest bin index >= from holding more than kRankMax keys, or ~0u.  Block-uniform result.
__device__ __forceinline__ unsigned int next_big_bin(const unsigned int *ends, unsigned int nb, unsigned int from,
                                                     SortSmem &S, int tid)
{
    unsigned int cand = 0xffffffffu;
    for (unsigned int b = from + tid; b < nb; b += kSortThreads) {
        const unsigned int lo = b ? ends[b - 1] : 0u;
        if (ends[b] - lo > kRankMax) { cand = b; break; }
    }
    return block_min_u32(S, cand, tid);
}

// Sorts buf[0, n) (output of a level-1 bin pass with map m / ends) into out[0, n).  scratch[0, n) is global memory the
// block may overwrite (level-2 scatter target).
__device__ void finish_sort(const u64 *buf, unsigned int n, const BinMap &m, u64 *scratch, uint32_t *__restrict__ out,
                            SortSmem &S, int tid)
{
    const unsigned int *ends = S.ends[0];
    rank_small(buf, n, ends, m, out, &S.any_big[0], tid);       // any_big was zeroed before the barriers of bin_pass
    __syncthreads();
    if (!S.any_big[0]) return;                                  // the usual case: no bin scan, no further barrier
    unsigned int from = 0;
    while (true) {
        const unsigned int b = next_big_bin(ends, m.nb, from, S, tid);
        if (b == 0xffffffffu) break;
        from = b + 1;
        const unsigned int lo = b ? ends[b - 1] : 0u, n2 = ends[b] - lo;
        // ---- level 2: the bin over its own key range
        u64 *buf2 = scratch + lo;
        if (tid == 0) S.any_big[1] = 0;                         // ordered by the barriers of bin_pass / next_big_bin
        const BinMap m2 = bin_pass(buf + lo, buf2, n2, S.ends[1], S, tid);
        const unsigned int *ends2 = S.ends[1];
        rank_small(buf2, n2, ends2, m2, out + lo, &S.any_big[1], tid);
        __syncthreads();
        unsigned int from2 = 0;
        while (S.any_big[1]) {
            const unsigned int b2 = next_big_bin(ends2, m2.nb, from2, S, tid);
            if (b2 == 0xffffffffu) break;
            from2 = b2 + 1;
            // ---- still oversized (nested clusters of nearly equal keys): rank counting by the whole block
            const unsigned int lo2 = b2 ? ends2[b2 - 1] : 0u, hi2 = ends2[b2];
            for (unsigned int p = lo2 + tid; p < hi2; p += kSortThreads) {
                const u64 k = buf2[p];
                unsigned int cnt = 0;
                for (unsigned int q = lo2; q < hi2; ++q) cnt += buf2[q] < k ? 1u : 0u;
                out[lo + lo2 + cnt] = (uint32_t)k;
            }
        }
    }
}

// Sorts slice b (keys tmp[lo, lo + n2), left there by the coarse pass) into vals[lo, lo + n2); pairs[lo, ...) is scratch.
__device__ __forceinline__ void sort_slice(u64 *pairs, u64 *tmp, uint32_t *vals, unsigned int lo, unsigned int n2, SortSmem &S, int tid)
{
    if (n2 == 0) return;
    if (n2 == 1) { if (tid == 0) vals[lo] = (uint32_t)tmp[lo]; return; }
    if (n2 <= (unsigned int)kSortCap) {
        const BinMap m = bin_pass(tmp + lo, S.keys, n2, S.ends[0], S, tid);
        finish_sort(S.keys, n2, m, pairs + lo, vals + lo, S, tid);
    } else {
        const BinMap m = bin_pass(tmp + lo, pairs + lo, n2, S.ends[0], S, tid);
        finish_sort(pairs + lo, n2, m, tmp + lo, vals + lo, S, tid);
    }
    __syncthreads();
    if (tid == 0) S.any_big[0] = 0;                      // ordered before its next readers by the barriers of bin_pass
}

// LAZY (blend-driven ordering): of a list longer than kSortCap only the nearest depth slices -- at least
// kLazyFirst keys -- are sorted here; the slice ends stay in ws.slice_ends, ws.lazy[tile] says how far the order goes.
// k_blend consumes that prefix, and only the tiles whose pixels are still alive at its end are finished by
// k_tile_sort_rest / k_blend<.., true>.  On a coarse level alone the blend reads 5-7 % of every list.
template <bool LAZY>
__global__ void __launch_bounds__(kSortThreads, 4)      // 4 CTAs per SM is what the 49 KB of shared memory allow
k_tile_sort(const WorkspaceDev ws, int tile0, int n_tiles)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem &S = *reinterpret_cast<SortSmem *>(smem_raw);

    const int tile = tile0 + blockIdx.x;               // the grid covers the frame's strip of tile rows
    if (tile >= n_tiles) return;
    const int tid = threadIdx.x;
    cudaGridDependencySynchronize();
    const uint2 rg = ws.ranges[tile];
    const unsigned int L = rg.y - rg.x;
    if (L == 0 || ws.hdr->overflow) return;            // an overflowed frame is undefined (and its keys need not be unique)
    u64 *pairs = ws.pairs + rg.x;
    uint32_t *vals = ws.vals + rg.x;
    if (L == 1) { if (tid == 0) vals[0] = (uint32_t)pairs[0]; return; }
    if (tid == 0) S.any_big[0] = 0;
    if (L <= (unsigned int)kSortCap) {
        const BinMap m = bin_pass(pairs, S.keys, L, S.ends[0], S, tid);
        finish_sort(S.keys, L, m, pairs, vals, S, tid);
        return;
    }
    // ---- a long list: cut it into depth slices of 512-1024 keys (one pass through global memory), then sort every
    // slice in shared memory like a short list: ranking a 30 000-key list straight from 2048 bins costs 15 L2 reads
    // per key, the slices cost one more scatter.  A slice that is still longer than kSortCap (a cluster of nearly
    // equal depths) goes through global memory.
    u64 *tmp = ws.pairs_tmp + rg.x;
    const BinMap mc = bin_pass(pairs, tmp, L, S.cends, S, tid, kSortSliceLog, 1, kCoarseBinsLog);
    unsigned int b = 0;
    for (; b < mc.nb; ++b) {
        const unsigned int lo = b ? S.cends[b - 1] : 0u;
        if (LAZY && lo >= kLazyFirst) break;             // enough for most tiles: the rest on demand
        sort_slice(pairs, tmp, vals, lo, S.cends[b] - lo, S, tid);
    }
    if (LAZY) {
        for (unsigned int i = tid; i < mc.nb; i += kSortThreads) ws.slice_ends[(size_t)tile * kCoarseBins + i] = S.cends[i];
        if (tid == 0) ws.lazy[tile] = make_uint4(b ? S.cends[b - 1] : 0u, b, mc.nb, 0u);   // sorted up to, next slice, slices, more wanted
    }
}

// The rest of the lists whose tiles k_blend left unfinished (ws.todo): slices next .. n of the coarse pass.  A small
// persistent grid walks the list of those tiles, so that a frame without any costs one short launch.
__global__ void __launch_bounds__(kSortThreads, 4)
k_tile_sort_rest(const WorkspaceDev ws)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem &S = *reinterpret_cast<SortSmem *>(smem_raw);
    cudaGridDependencySynchronize();
    const unsigned int n_todo = ws.hdr->n_todo;
    const int tid = threadIdx.x;
    for (unsigned int w = blockIdx.x; w < n_todo; w += gridDim.x) {
        const unsigned int tile = ws.todo[w];
        const uint2 rg = ws.ranges[tile];
        const uint4 lz = ws.lazy[tile];
        __syncthreads();                                  // the previous tile's S.cends is no longer read
        for (unsigned int i = tid; i < lz.z; i += kSortThreads) S.cends[i] = ws.slice_ends[(size_t)tile * kCoarseBins + i];
        if (tid == 0) S.any_big[0] = 0;
        __syncthreads();
        u64 *pairs = ws.pairs + rg.x, *tmp = ws.pairs_tmp + rg.x;
        uint32_t *vals = ws.vals + rg.x;
        for (unsigned int b = lz.y; b < lz.z; ++b) {
            const unsigned int lo = b ? S.cends[b - 1] : 0u;
            sort_slice(pairs, tmp, vals, lo, S.cends[b] - lo, S, tid);
        }
    }
}

// Once per device (flod_create, after cudaSetDevice): SortSmem exceeds the 48 KB default of dynamic shared memory, and
// the opt-in is a per-device attribute of the function.
int init_tile_sort()
{
    const int bytes = (int)sizeof(SortSmem);
    return cudaFuncSetAttribute(k_tile_sort<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess &&
           cudaFuncSetAttribute(k_tile_sort<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess &&
           cudaFuncSetAttribute(k_tile_sort_rest, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) == cudaSuccess ? 0 : -1;
}

int launch_tile_sort(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    const int tile0 = p.ty_begin * p.TX, n_tiles = p.ty_end * p.TX;
    if (n_tiles <= tile0) return 0;
    if (p.lazy_sort) launch_pdl(k_tile_sort<true>, n_tiles - tile0, kSortThreads, sizeof(SortSmem), s, c.ws, tile0, n_tiles);
    else launch_pdl(k_tile_sort<false>, n_tiles - tile0, kSortThreads, sizeof(SortSmem), s, c.ws, tile0, n_tiles);
    return 1;
}

int launch_tile_sort_rest(const Context &c, const FrameParams &p, cudaStream_t s)
{
    const int tile0 = p.ty_begin * p.TX, n_tiles = p.ty_end * p.TX;
    if (p.n_pre_blocks <= 0 || n_tiles <= tile0 || !p.lazy_sort) return 0;
    launch_pdl(k_tile_sort_rest, min(n_tiles - tile0, 2 * c.sm_count), kSortThreads, sizeof(SortSmem), s, c.ws);
    return 1;
}

}  // namespace flod
