// Step a7: stable LSD radix sort of (tile << 32 | depth bits) keys carrying compact Gaussian indices, and
// step a8: per-tile range extraction.
//
// Only the low (32 + tile_bits) key bits are significant, so ceil((32 + tile_bits) / 8) passes of 8 bits run.
// Each pass is ONE kernel ("onesweep"): a block ranks a tile of 4096 keys in shared memory (per-warp digit
// counters + match_any ranking: stable), publishes its digit counts, obtains its global offsets from the blocks
// before it by a decoupled look-back (blocks are ordered by an atomic ticket; status words carry an epoch tag so
// nothing has to be zeroed between passes) and scatters.  The number of pairs is read from device memory
// (FrameHeader::n_pairs_clamped): the host never waits for it.  Stability + emission in ascending gid (a6) gives
// the (depth, gid) order of DESIGN R15 without putting the id in the key.
#include "flod_internal.cuh"

namespace flod {

int sort_passes_for(int tile_bits) { return (32 + tile_bits + kRadixBits - 1) / kRadixBits; }

// ---- digit histograms of all passes in one read of the keys
__global__ void __launch_bounds__(512)
k_sort_hist(const WorkspaceDev ws, int passes)
{
    __shared__ unsigned int s_hist[kMaxPasses * kRadix];
    for (int i = threadIdx.x; i < passes * kRadix; i += blockDim.x) s_hist[i] = 0;
    __syncthreads();
    const unsigned int n = ws.hdr->n_pairs_clamped;
    const unsigned long long *__restrict__ keys = ws.keys[0];
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        unsigned long long k = keys[i];
        for (int p = 0; p < passes; ++p)
            atomicAdd(&s_hist[p * kRadix + (unsigned int)((k >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * kRadix; i += blockDim.x) {
        unsigned int c = s_hist[i];
        if (c) atomicAdd(&ws.hdr->hist[i / kRadix][i % kRadix], c);
    }
}

constexpr unsigned int kStAgg = 1u << 30, kStIncl = 2u << 30, kStFlagMask = 3u << 30, kStValMask = (1u << 30) - 1;

__global__ void __launch_bounds__(kSortThreads)
k_onesweep(const WorkspaceDev ws, int pass, int src, unsigned int epoch)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned long long *s_keys = reinterpret_cast<unsigned long long *>(smem_raw);                  // [kSortTile]
    uint32_t *s_vals = reinterpret_cast<uint32_t *>(s_keys + kSortTile);                             // [kSortTile]
    unsigned int *s_whist = s_vals + kSortTile;                                                      // [warps][kRadix]
    unsigned int *s_dstart = s_whist + (kSortThreads / 32) * kRadix;                                 // [kRadix] block-local exclusive digit start
    unsigned int *s_gbase = s_dstart + kRadix;                                                       // [kRadix] global base of this block's digit run
    unsigned int *s_wsum = s_gbase + kRadix;                                                         // [16]
    __shared__ unsigned int s_vb;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int kWarps = kSortThreads / 32;
    const unsigned int n = ws.hdr->n_pairs_clamped;
    const unsigned int n_blocks = (n + kSortTile - 1) / kSortTile;
    const int shift = pass * kRadixBits;
    const unsigned long long *__restrict__ kin = (src ? ws.keys[1] : ws.keys[0]);
    const uint32_t *__restrict__ vin = (src ? ws.vals[1] : ws.vals[0]);
    unsigned long long *__restrict__ kout = (src ? ws.keys[0] : ws.keys[1]);
    uint32_t *__restrict__ vout = (src ? ws.vals[0] : ws.vals[1]);
    unsigned long long *status = ws.sort_status;   // shared by all passes: words are tagged with the pass epoch

    while (true) {
        __syncthreads();
        if (tid == 0) s_vb = atomicAdd(&ws.hdr->sort_ticket[pass], 1u);
        __syncthreads();
        const unsigned int vb = s_vb;
        if (vb >= n_blocks) return;
        const unsigned int tile_base = vb * kSortTile;
        const unsigned int tile_n = min((unsigned int)kSortTile, n - tile_base);

        for (int i = tid; i < kWarps * kRadix; i += kSortThreads) s_whist[i] = 0;
        __syncthreads();

        // ---- load (warp-contiguous chunks, striped inside the warp) and rank within the warp, stable
        unsigned long long key[kSortItems];
        uint32_t val[kSortItems];
        unsigned short rnk[kSortItems];
        const unsigned int wbase = warp * (32 * kSortItems);
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) {
            unsigned int li = wbase + r * 32 + lane;
            bool ok = li < tile_n;
            key[r] = ok ? kin[tile_base + li] : ~0ull;
            val[r] = ok ? vin[tile_base + li] : 0u;
        }
        unsigned int *wh = s_whist + warp * kRadix;
#pragma unroll
        for (int r = 0; r < kSortItems; ++r) {
            unsigned int d = (unsigned int)((key[r] >> shift) & (kRadix - 1));
            unsigned int peers = __match_any_sync(0xffffffffu, d);
            unsigned int leader = __ffs(peers) - 1;
            unsigned int before = __popc(peers & ((1u << lane) - 1));
            unsigned int old = 0;
            if (lane == leader) { old = wh[d]; wh[d] = old + __popc(peers); }
            old = __shfl_sync(0xffffffffu, old, leader);
            rnk[r] = (unsigned short)(old + before);
            __syncwarp();
        }
        __syncthreads();

        // ---- per digit (thread d < 256): exclusive scan across warps -> block count; warp-level scans across
        //      digits of (block counts) and of (the frame's digit histogram)
        unsigned int cnt = 0, cnt_excl = 0, h_excl = 0;
        if (tid < kRadix) {
            unsigned int run = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                unsigned int t = s_whist[w * kRadix + tid];
                s_whist[w * kRadix + tid] = run;
                run += t;
            }
            cnt = run;
            unsigned int h = ws.hdr->hist[pass][tid];
            unsigned int inc = cnt, hinc = h;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
                unsigned int u = __shfl_up_sync(0xffffffffu, hinc, o);
                if (lane >= o) { inc += t; hinc += u; }
            }
            if (lane == 31) { s_wsum[warp] = inc; s_wsum[8 + warp] = hinc; }
            cnt_excl = inc - cnt;
            h_excl = hinc - h;
        }
        __syncthreads();
        if (tid < kRadix) {
#pragma unroll
            for (int w = 0; w < kRadix / 32; ++w)
                if (w < warp) { cnt_excl += s_wsum[w]; h_excl += s_wsum[8 + w]; }
            s_dstart[tid] = cnt_excl;                     // block-local start of digit tid
            // padding keys (~0) of a partial last tile sit at the end of digit 255's run: not counted globally
            const unsigned int real_count = (tid == kRadix - 1) ? cnt - (kSortTile - tile_n) : cnt;
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
        for (int r = 0; r < kSortItems; ++r) {
            unsigned int d = (unsigned int)((key[r] >> shift) & (kRadix - 1));
            unsigned int pos = s_dstart[d] + wh[d] + rnk[r];
            s_keys[pos] = key[r];
            s_vals[pos] = val[r];
        }
        __syncthreads();

        // ---- coalesced runs to global memory
        for (unsigned int i = tid; i < tile_n; i += kSortThreads) {
            unsigned long long k = s_keys[i];
            unsigned int d = (unsigned int)((k >> shift) & (kRadix - 1));
            unsigned int dst = s_gbase[d] + (i - s_dstart[d]);
            kout[dst] = k;
            vout[dst] = s_vals[i];
        }
    }
}

// ---- a8: [start, end) of every tile in the sorted keys (ranges were zeroed with the frame header)
__global__ void __launch_bounds__(256)
k_ranges(const WorkspaceDev ws, int buf)
{
    const unsigned int n = ws.hdr->n_pairs_clamped;
    const unsigned long long *__restrict__ keys = (buf ? ws.keys[1] : ws.keys[0]);
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        unsigned int t = (unsigned int)(keys[i] >> 32);
        if (i == 0 || (unsigned int)(keys[i - 1] >> 32) != t) ws.ranges[t].x = i;
        if (i == n - 1 || (unsigned int)(keys[i + 1] >> 32) != t) ws.ranges[t].y = i + 1;
    }
}

static size_t onesweep_smem()
{
    return (size_t)kSortTile * 12 + (size_t)(kSortThreads / 32) * kRadix * 4 + 2 * kRadix * 4 + 16 * 4;
}

int launch_sort(Context &c, int tile_bits, int *final_buf, cudaStream_t s)
{
    const int passes = sort_passes_for(tile_bits);
    const int grid = c.sm_count * 2;
    k_sort_hist<<<grid, 512, 0, s>>>(c.ws, passes);
    static bool attr_set = false;
    const size_t smem = onesweep_smem();
    if (!attr_set) {
        cudaFuncSetAttribute(k_onesweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        attr_set = true;
    }
    int src = 0;
    for (int p = 0; p < passes; ++p) {
        c.epoch += 1;
        if (c.epoch == 0) c.epoch = 1;
        k_onesweep<<<c.sm_count * 3, kSortThreads, smem, s>>>(c.ws, p, src, c.epoch);
        src ^= 1;
    }
    *final_buf = src;
    return 1 + passes;
}

int launch_ranges(const Context &c, int final_buf, cudaStream_t s)
{
    k_ranges<<<c.sm_count * 8, 256, 0, s>>>(c.ws, final_buf);
    return 1;
}

}  // namespace flod
