// Step a7: the (tile | depth) order of the pairs, and step a8: per-tile range extraction.
//
// The (tile, depth, gid) order is produced by two stable LSD radix sorts instead of one sort of 64-bit pair keys:
//   1. the VISIBLE GAUSSIANS (N_vis of them, not the P pairs) are sorted by their 32 depth bits, 4 passes of 8 bits,
//      carrying the compact index (ascending gid, so stability gives the (depth, gid) order of DESIGN R15);
//   2. pairs are emitted in that order (duplicate.cu) with only a tile id as key (uint16 when T_n <= 65536) and are
//      sorted by tile id alone: ceil(tile_bits / 8) stable passes (2 passes of 6 bits at 1237x822).
// Sorted traffic per frame: 4 x 16 B x N_vis + 2 x 12 B x P  instead of  6 x 24 B x P.
//
// Every pass is ONE kernel ("onesweep"): a block ranks a tile of keys in shared memory (per-warp digit counters +
// match_any ranking: stable), publishes its digit counts, obtains its global offsets from the blocks before it by a
// decoupled look-back (blocks are ordered by an atomic ticket; status words carry an epoch tag so nothing has to be
// zeroed between passes) and scatters.  Element counts are read from device memory (FrameHeader): the host never
// waits for them.
#include "flod_internal.cuh"

namespace flod {

static int ceil_log2(unsigned v) { int b = 0; while ((1u << b) < v) ++b; return b; }

TileSortPlan tile_sort_plan(int n_tiles)
{
    TileSortPlan pl{};
    const int tile_bits = ceil_log2((unsigned)(n_tiles > 1 ? n_tiles : 1));
    pl.passes = (tile_bits + kRadixBits - 1) / kRadixBits;
    pl.bits = pl.passes ? (tile_bits + pl.passes - 1) / pl.passes : 0;
    pl.wide = n_tiles > 65536;
    return pl;
}

// ---- digit histograms of all passes of one sort in one read of the keys
template <typename KeyT>
__global__ void __launch_bounds__(512)
k_sort_hist(const KeyT *__restrict__ keys, const unsigned int *__restrict__ n_ptr, unsigned int *__restrict__ hist_out,
            int passes, int bits)
{
    __shared__ unsigned int s_hist[kDepthPasses * kRadix];
    for (int i = threadIdx.x; i < passes * kRadix; i += blockDim.x) s_hist[i] = 0;
    __syncthreads();
    const unsigned int n = *n_ptr;
    const unsigned int mask = (1u << bits) - 1;
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned int k = (unsigned int)keys[i];
        for (int p = 0; p < passes; ++p) atomicAdd(&s_hist[p * kRadix + ((k >> (p * bits)) & mask)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * kRadix; i += blockDim.x) {
        const unsigned int c = s_hist[i];
        if (c) atomicAdd(&hist_out[i], c);
    }
}

constexpr unsigned int kStAgg = 1u << 30, kStIncl = 2u << 30, kStFlagMask = 3u << 30, kStValMask = (1u << 30) - 1;

// One stable radix pass on digit (key >> shift) & (2^bits - 1).  IOTA: the values are the element indices (pass 0).
template <typename KeyT, int THREADS, int ITEMS, bool IOTA>
__global__ void __launch_bounds__(THREADS)
k_onesweep(const KeyT *__restrict__ kin, const uint32_t *__restrict__ vin, KeyT *__restrict__ kout,
           uint32_t *__restrict__ vout, const unsigned int *__restrict__ n_ptr, unsigned int *ticket,
           const unsigned int *__restrict__ hist, unsigned long long *status, int shift, int bits, unsigned int epoch)
{
    constexpr int TILE = THREADS * ITEMS;
    constexpr int kWarps = THREADS / 32;
    static_assert(THREADS >= kRadix, "one thread per digit");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t *s_vals = reinterpret_cast<uint32_t *>(smem_raw);                  // [TILE]
    unsigned int *s_whist = s_vals + TILE;                                       // [warps][kRadix]
    unsigned int *s_dstart = s_whist + kWarps * kRadix;                          // [kRadix] block-local start of a digit
    unsigned int *s_gbase = s_dstart + kRadix;                                   // [kRadix] global start of the block's run
    unsigned int *s_wsum = s_gbase + kRadix;                                     // [16]
    KeyT *s_keys = reinterpret_cast<KeyT *>(s_wsum + 16);                        // [TILE]
    __shared__ unsigned int s_vb;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int n = *n_ptr;
    const unsigned int n_blocks = (n + TILE - 1) / TILE;
    const unsigned int radix = 1u << bits, dmask = radix - 1;
    constexpr KeyT kPad = (KeyT) ~(KeyT)0;

    while (true) {
        __syncthreads();
        if (tid == 0) s_vb = atomicAdd(ticket, 1u);
        __syncthreads();
        const unsigned int vb = s_vb;
        if (vb >= n_blocks) return;
        const unsigned int tile_base = vb * TILE;
        const unsigned int tile_n = min((unsigned int)TILE, n - tile_base);

        for (int i = tid; i < kWarps * kRadix; i += THREADS) s_whist[i] = 0;
        __syncthreads();

        // ---- load (warp-contiguous chunks, striped inside the warp) and rank within the warp, stable
        KeyT key[ITEMS];
        uint32_t val[ITEMS];
        unsigned short rnk[ITEMS];
        const unsigned int wbase = warp * (32 * ITEMS);
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {
            const unsigned int li = wbase + r * 32 + lane;
            const bool ok = li < tile_n;
            key[r] = ok ? kin[tile_base + li] : kPad;
            if (IOTA) val[r] = tile_base + li;
            else val[r] = ok ? vin[tile_base + li] : 0u;
        }
        unsigned int *wh = s_whist + warp * kRadix;
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {
            const unsigned int d = ((unsigned int)key[r] >> shift) & dmask;
            const unsigned int peers = __match_any_sync(0xffffffffu, d);
            const unsigned int leader = __ffs(peers) - 1;
            const unsigned int before = __popc(peers & ((1u << lane) - 1));
            unsigned int old = 0;
            if (lane == leader) { old = wh[d]; wh[d] = old + __popc(peers); }
            old = __shfl_sync(0xffffffffu, old, leader);
            rnk[r] = (unsigned short)(old + before);
            __syncwarp();
        }
        __syncthreads();

        // ---- per digit (thread d < radix): exclusive scan across warps -> block count; warp-level scans across
        //      digits of (block counts) and of (the frame's digit histogram)
        unsigned int cnt = 0, cnt_excl = 0, h_excl = 0;
        if (tid < kRadix) {
            unsigned int h = 0;
            if ((unsigned int)tid < radix) {
                unsigned int run = 0;
#pragma unroll
                for (int w = 0; w < kWarps; ++w) {
                    const unsigned int t = s_whist[w * kRadix + tid];
                    s_whist[w * kRadix + tid] = run;
                    run += t;
                }
                cnt = run;
                h = hist[tid];
            }
            unsigned int inc = cnt, hinc = h;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
                const unsigned int u = __shfl_up_sync(0xffffffffu, hinc, o);
                if (lane >= o) { inc += t; hinc += u; }
            }
            if (lane == 31) { s_wsum[warp] = inc; s_wsum[8 + warp] = hinc; }
            cnt_excl = inc - cnt;
            h_excl = hinc - h;
        }
        __syncthreads();
        if ((unsigned int)tid < radix) {
#pragma unroll
            for (int w = 0; w < kRadix / 32; ++w)
                if (w < warp) { cnt_excl += s_wsum[w]; h_excl += s_wsum[8 + w]; }
            s_dstart[tid] = cnt_excl;                     // block-local start of digit tid
            // padding keys (all ones) of a partial last tile sit at the end of the top digit's run: not counted globally
            const unsigned int real_count = ((unsigned int)tid == dmask) ? cnt - (TILE - tile_n) : cnt;
            // ---- decoupled look-back for this digit over the blocks before this one
            unsigned long long *st = status + tid;
            const unsigned long long tag = (unsigned long long)epoch << 32;
            unsigned int excl = 0;
            if (vb == 0) {
                atomicExch(st, tag | kStIncl | real_count);
            } else {
                atomicExch(st + (size_t)vb * kRadix, tag | kStAgg | real_count);
                long long j = (long long)vb - 1;
                while (true) {
                    volatile unsigned long long *ptr = st + (size_t)j * kRadix;
                    unsigned long long sv;
                    do { sv = *ptr; } while ((unsigned int)(sv >> 32) != epoch || ((unsigned int)sv & kStFlagMask) == 0);
                    excl += (unsigned int)sv & kStValMask;
                    if (((unsigned int)sv & kStFlagMask) == kStIncl) break;
                    --j;
                }
                atomicExch(st + (size_t)vb * kRadix, tag | kStIncl | (excl + real_count));
            }
            s_gbase[tid] = h_excl + excl;                 // global start of this block's run of digit tid
        }
        __syncthreads();

        // ---- scatter into shared memory in block-sorted order
#pragma unroll
        for (int r = 0; r < ITEMS; ++r) {
            const unsigned int d = ((unsigned int)key[r] >> shift) & dmask;
            const unsigned int pos = s_dstart[d] + wh[d] + rnk[r];
            s_keys[pos] = key[r];
            s_vals[pos] = val[r];
        }
        __syncthreads();

        // ---- coalesced runs to global memory
#pragma unroll 4
        for (unsigned int i = tid; i < tile_n; i += THREADS) {
            const KeyT k = s_keys[i];
            const unsigned int d = ((unsigned int)k >> shift) & dmask;
            const unsigned int dst = s_gbase[d] + (i - s_dstart[d]);
            kout[dst] = k;
            vout[dst] = s_vals[i];
        }
    }
}

template <typename KeyT, int THREADS, int ITEMS>
constexpr size_t onesweep_smem()
{
    return (size_t)THREADS * ITEMS * (4 + sizeof(KeyT)) + (size_t)(THREADS / 32) * kRadix * 4 + 2 * kRadix * 4 + 16 * 4;
}

template <typename KeyT, int THREADS, int ITEMS, bool IOTA>
static void launch_onesweep(int grid, const KeyT *kin, const uint32_t *vin, KeyT *kout, uint32_t *vout,
                            const unsigned int *n_ptr, unsigned int *ticket, const unsigned int *hist,
                            unsigned long long *status, int shift, int bits, unsigned int epoch, cudaStream_t s)
{
    constexpr size_t smem = onesweep_smem<KeyT, THREADS, ITEMS>();
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_onesweep<KeyT, THREADS, ITEMS, IOTA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    k_onesweep<KeyT, THREADS, ITEMS, IOTA><<<grid, THREADS, smem, s>>>(kin, vin, kout, vout, n_ptr, ticket, hist, status,
                                                                       shift, bits, epoch);
}

static unsigned int next_epoch(Context &c)
{
    c.epoch += 1;
    if (c.epoch == 0) c.epoch = 1;
    return c.epoch;
}

constexpr int kDepthThreads = 256, kDepthItems = kDepthSortTile / kDepthThreads;
constexpr int kTileThreads = 512, kTileItems = kTileSortTile / kTileThreads;

// Depth sort of the visible Gaussians: keys ws.depth (by compact index), values = compact indices.
// Pass 0 reads ws.depth and writes buffer 1; passes 1-3 ping-pong 1 -> 0 -> 1 -> 0.  *final_buf = 0.
int launch_depth_sort(Context &c, int *final_buf, cudaStream_t s)
{
    const WorkspaceDev &ws = c.ws;
    FrameHeader *h = ws.hdr;
    k_sort_hist<uint32_t><<<c.sm_count * 2, 512, 0, s>>>(ws.depth, &h->n_vis32, &h->hist[0][0], kDepthPasses, kRadixBits);
    const int grid = c.sm_count * 4;
    launch_onesweep<uint32_t, kDepthThreads, kDepthItems, true>(grid, ws.depth, nullptr, ws.dkeys[1], ws.dvals[1], &h->n_vis32,
                                                                &h->sort_ticket[0], h->hist[0], ws.sort_status, 0, kRadixBits,
                                                                next_epoch(c), s);
    int src = 1;
    for (int p = 1; p < kDepthPasses; ++p) {
        launch_onesweep<uint32_t, kDepthThreads, kDepthItems, false>(grid, ws.dkeys[src], ws.dvals[src], ws.dkeys[src ^ 1],
                                                                     ws.dvals[src ^ 1], &h->n_vis32, &h->sort_ticket[p],
                                                                     h->hist[p], ws.sort_status, p * kRadixBits, kRadixBits,
                                                                     next_epoch(c), s);
        src ^= 1;
    }
    *final_buf = src;
    return 1 + kDepthPasses;
}

template <typename KeyT>
static int tile_sort_t(Context &c, const TileSortPlan &pl, int *final_buf, cudaStream_t s)
{
    const WorkspaceDev &ws = c.ws;
    FrameHeader *h = ws.hdr;
    if (pl.passes == 0) { *final_buf = 0; return 0; }
    k_sort_hist<KeyT><<<c.sm_count * 2, 512, 0, s>>>((const KeyT *)ws.tkeys[0], &h->n_pairs_clamped,
                                                     &h->hist[kDepthPasses][0], pl.passes, pl.bits);
    int src = 0;
    for (int p = 0; p < pl.passes; ++p) {
        launch_onesweep<KeyT, kTileThreads, kTileItems, false>(c.sm_count * 2, (const KeyT *)ws.tkeys[src], ws.vals[src],
                                                               (KeyT *)ws.tkeys[src ^ 1], ws.vals[src ^ 1], &h->n_pairs_clamped,
                                                               &h->sort_ticket[kDepthPasses + p], h->hist[kDepthPasses + p],
                                                               ws.sort_status, p * pl.bits, pl.bits, next_epoch(c), s);
        src ^= 1;
    }
    *final_buf = src;
    return 1 + pl.passes;
}

int launch_tile_sort(Context &c, const FrameParams &p, int *final_buf, cudaStream_t s)
{
    const TileSortPlan pl = tile_sort_plan(p.n_tiles);
    return pl.wide ? tile_sort_t<uint32_t>(c, pl, final_buf, s) : tile_sort_t<uint16_t>(c, pl, final_buf, s);
}

// ---- a8: [start, end) of every tile in the sorted tile ids (ranges were zeroed with the frame header)
template <typename KeyT>
__global__ void __launch_bounds__(256)
k_ranges(const KeyT *__restrict__ keys, const unsigned int *__restrict__ n_ptr, uint2 *__restrict__ ranges)
{
    const unsigned int n = *n_ptr;
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned int t = keys[i];
        if (i == 0 || (unsigned int)keys[i - 1] != t) ranges[t].x = i;
        if (i == n - 1 || (unsigned int)keys[i + 1] != t) ranges[t].y = i + 1;
    }
}

int launch_ranges(const Context &c, const FrameParams &p, int final_buf, cudaStream_t s)
{
    const WorkspaceDev &ws = c.ws;
    if (tile_sort_plan(p.n_tiles).wide)
        k_ranges<uint32_t><<<c.sm_count * 8, 256, 0, s>>>((const uint32_t *)ws.tkeys[final_buf], &ws.hdr->n_pairs_clamped, ws.ranges);
    else
        k_ranges<uint16_t><<<c.sm_count * 8, 256, 0, s>>>((const uint16_t *)ws.tkeys[final_buf], &ws.hdr->n_pairs_clamped, ws.ranges);
    return 1;
}

}  // namespace flod
