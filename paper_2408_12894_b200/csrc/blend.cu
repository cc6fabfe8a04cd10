// Step a9: per-tile front-to-back alpha blending with early transmittance termination.
// Eq. 2: alpha = o exp(-1/2 d^T Sigma'^-1 d); "alpha blending the projected Gaussians in depth
// order"; clamp 0.99, skip below 1/255, stop after T < 1e-4 (R11, R12).
//
// One CTA of 128 threads owns one 16x16 tile; a thread owns two vertically adjacent pixels, a warp a 16x4 strip.
// The tile's sorted list is consumed in batches of 128: a thread fetches one position (coalesced) and gathers the 36 B
// of blend features of that Gaussian (L2-resident) into shared memory with cp.async, double-buffered.
// Each warp then FILTERS the batch against its own strip, 32 Gaussians per step (one per lane).  With the
// factorised exponent (DESIGN R25)
//     e(x, y) = log2(o) + a2 w^2 + d2 dy^2,   w = (mu'x - x) + k dy,   a2, d2 <= 0
// everything that depends on the row only is computed ONCE per (Gaussian, row) by the filtering lane:
//     c_r = mu'x + k dy_r,   e0_r = log2(o) + d2 dy_r^2        so that   e = a2 (c_r - x)^2 + e0_r,
// the maximum of e over the 16 pixels of the row is closed-form, and a Gaussian whose four row maxima are all below
// log2(1/255) is dropped.  The survivors are ballot-compacted, in order, into a per-warp buffer of 48-byte records
// (c_0..c_3, e0_0..e0_3, a2, r, g, b); the per-pixel loop reads those and spends three packed instructions on the
// exponent.  The filter bounds the very values the loop evaluates (same c_r, e0_r; rounding is monotone), so a
// dropped Gaussian has alpha < 1/255 on every pixel of the strip and the image is bit-identical to the unfiltered
// loop.  A warp whose 64 pixels have all terminated skips filter and loop; the CTA stops when every warp has.
#include <type_traits>

#include "flod_internal.cuh"

namespace flod {

constexpr int kBlendThreads = 128;
constexpr int kBatch = 128;             // Gaussians staged per step (a multiple of kBlendThreads)
constexpr int kBlendWarps = kBlendThreads / 32;
constexpr int kWarpBuf = 32;                         // survivors a warp collects before it evaluates them
constexpr int kFlush = kWarpBuf - 32;                // evaluate when more than this many survivors wait (<= kWarpBuf - 32)

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned int)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned int)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// alpha if alpha >= 1/255 and T >= 1e-4, else 0 (FSETP, FSETP.AND, FSEL)
__device__ __forceinline__ float keep_if_live(float alpha, float T)
{
    float r;
    asm("{\n\t.reg .pred p, q;\n\t"
        "setp.ge.f32 q, %2, 0f38D1B717;\n\t"            // 1e-4f
        "setp.ge.and.f32 p, %1, 0f3B808081, q;\n\t"     // (float)(1/255)
        "selp.f32 %0, %1, 0f00000000, p;\n\t}"
        : "=f"(r) : "f"(alpha), "f"(T));
    return r;
}

// 2^x on the MUFU unit (x <= 0 here; results below 2^-126 flush to 0, far under the 1/255 skip threshold)
__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

constexpr int kBlendUnroll = 4;
constexpr int kBlendMinBlocks = 8;                   // 64 registers per thread
// RESUME: the second round of blend-driven ordering.  In a lazy frame k_tile_sort orders only the nearest
// slices of a long list; the first round (RESUME = false) blends that prefix and, if pixels of the tile are still alive at
// its end, saves (T, r, g, b) of every pixel and asks for the rest; k_tile_sort_rest orders it, and this kernel
// (RESUME = true) takes the saved state up from where the first round stopped.  The per-pixel sequence of blends is the
// one of a fully sorted list, so the image is bit-identical.
template <bool COUNT, bool RESUME>
__device__ __forceinline__ void blend_tile(const WorkspaceDev &ws, float *__restrict__ out, int W, int H, int TX, int n_tiles,
                                           float bg0, float bg1, float bg2, int tile, int out_row0, int out_rows, int lazy)
{
    // staging, 36 bytes per Gaussian of the batch: A = (mu'x, mu'y, k, a2), B = (d2, log2 o, r, g), c = b
    __shared__ float4 s_A[2][kBatch], s_B[2][kBatch];           // double-buffered
    __shared__ float s_c[2][kBatch];
    // per warp, one 48-byte record per surviving Gaussian: (c_0, c_1, e0_0, e0_1 | c_2, c_3, e0_2, e0_3 | a2, r, g, b)
    __shared__ float4 s_buf[kBlendWarps][kWarpBuf * 3];
    __shared__ unsigned short s_idx[kBlendWarps][kWarpBuf];    // batch index of the survivor (counting variant only)

    if (tile >= n_tiles || ws.hdr->overflow) return;   // an overflowed frame is undefined: its lists were not sorted
    const int tx = tile % TX, ty = tile / TX;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // warp = rows 4w..4w+3 of the tile; lanes 0-15 rows (4w, 4w+1), lanes 16-31 rows (4w+2, 4w+3)
    const int half = lane >> 4;
    const int px = tx * kTile + (lane & 15);
    const int py0 = ty * kTile + warp * 4 + half * 2, py1 = py0 + 1;
    const bool in0 = px < W && py0 < H, in1 = px < W && py1 < H;
    const float x0c = (float)(tx * kTile) + 0.5f, y0c = (float)(ty * kTile) + 0.5f;   // centre of the tile's first pixel
    const float nlx = -(float)(lane & 15);              // minus the pixel's column inside the tile
    const float row0 = (float)(warp * 4);               // first row of the warp's strip inside the tile
    const float kThr = -7.994353436858858f - 1.0e-3f;   // log2(1/255) minus a safety margin

    uint2 rg = ws.ranges[tile];
    const unsigned int L_full = rg.y - rg.x;
    bool partial = false;                               // this round ends before the list does
    if (RESUME) {
        if (L_full <= (unsigned int)kSortCap) return;
        const uint4 lz = ws.lazy[tile];
        if (!lz.w) return;                              // the first round finished this tile
        rg.x += lz.x;                                   // go on behind the prefix it consumed
    } else if (lazy && L_full > (unsigned int)kSortCap) {
        const unsigned int upto = ws.lazy[tile].x;
        partial = upto < L_full;
        rg.y = rg.x + upto;
    }
    const uint32_t *__restrict__ vals = ws.vals;
    const float4 *__restrict__ gA = ws.gA;
    const float4 *__restrict__ gB = ws.gB;
    const float *__restrict__ cB = ws.cB;

    // two pixels per thread, packed as float2 (.x = row py0, .y = row py1): the per-pixel arithmetic runs on the
    // packed FP32 instructions of sm_100 (FADD2 / FMUL2 / FFMA2: one issue slot for both pixels)
    float2 T = make_float2(in0 ? 1.0f : 0.0f, in1 ? 1.0f : 0.0f), cr = make_float2(0.0f, 0.0f), cg = cr, cb2 = cr;
    if (RESUME) {
        const float4 s0 = ws.tile_state[(size_t)tile * 256 + 2 * tid], s1 = ws.tile_state[(size_t)tile * 256 + 2 * tid + 1];
        T = make_float2(s0.x, s1.x); cr = make_float2(s0.y, s1.y); cg = make_float2(s0.z, s1.z); cb2 = make_float2(s0.w, s1.w);
    }
    unsigned int n_eval = 0, n_blend = 0;
    float4 *my_buf = s_buf[warp];
    const float4 *my_half = my_buf + half;
    bool warp_done = __all_sync(0xffffffffu, T.x < 1e-4f && T.y < 1e-4f);   // (pixels outside the image start with T = 0)

    // evaluates my_buf[0, cnt) on the thread's two pixels.  a2 <= 0 and e0 <= log2 o (k_geometry clamps d2), so
    // q >= 0 holds by construction and alpha needs the 0.99 clamp only.  A pixel that is done or below 1/255 blends 0.
    // CLAMP = false: no survivor of the buffer has o > 0.99 - margin (log2 o <= -0.0146), so alpha <= o stays below the
    // 0.99 clamp and min(0.99, .) would return its argument: the same bits with two instructions less per entry.
    auto evaluate = [&](unsigned int cnt, unsigned int base_in_list, auto clamp_tag) {
        constexpr bool CLAMP = decltype(clamp_tag)::value;
#pragma unroll kBlendUnroll
        for (unsigned int t = 0; t < cnt; ++t) {
            const float4 hrec = my_half[3 * t];
            const float4 c = my_buf[3 * t + 2];
            const float2 w = __fadd2_rn(make_float2(hrec.x, hrec.y), make_float2(nlx, nlx));
            const float2 e = __ffma2_rn(make_float2(c.x, c.x), __fmul2_rn(w, w), make_float2(hrec.z, hrec.w));
            float al0 = ex2(e.x), al1 = ex2(e.y);
            if (CLAMP) { al0 = fminf(al0, 0.99f); al1 = fminf(al1, 0.99f); }
            // skip below 1/255 (R11); a pixel that has stopped (T < 1e-4 after an earlier blend, R12) or lies outside
            // the image (T = 0 from the start) blends nothing.  The test reads T directly, so the loop-carried chain is
            // T -> compare -> select -> multiply -> subtract; one predicate per pixel carries both conditions.
            al0 = keep_if_live(al0, T.x);
            al1 = keep_if_live(al1, T.y);
            const float2 wgt = __fmul2_rn(T, make_float2(al0, al1));
            cr = __ffma2_rn(wgt, make_float2(c.y, c.y), cr);
            cg = __ffma2_rn(wgt, make_float2(c.z, c.z), cg);
            cb2 = __ffma2_rn(wgt, make_float2(c.w, c.w), cb2);
            const float2 Tn = __fadd2_rn(T, make_float2(-wgt.x, -wgt.y));        // T (1 - alpha)
            if (COUNT) {
                n_blend += (al0 > 0.0f ? 1u : 0u) + (al1 > 0.0f ? 1u : 0u);
                const unsigned int visited = base_in_list + s_idx[warp][t] + 1;
                if (T.x >= 1e-4f && Tn.x < 1e-4f) n_eval += visited;               // the blend that stops the pixel
                if (T.y >= 1e-4f && Tn.y < 1e-4f) n_eval += visited;
            }
            T = Tn;
        }
    };

    // Software pipeline over the batches, one barrier per batch.  The features of batch b + 1 travel from L2 to the
    // other staging buffer with cp.async (no registers, no wait) while batch b is filtered and evaluated; the list
    // positions of batch b + 2 are loaded into a register at the same time, so that the dependent chain position ->
    // feature gather never stalls a warp.
    const unsigned int n_batches = (rg.y - rg.x + kBatch - 1) / kBatch;
    constexpr int kPer = kBatch / kBlendThreads;                  // Gaussians a thread stages per batch
    auto stage_batch = [&](unsigned int b, const uint32_t (&ci)[kPer]) {   // batch b -> staging buffer b & 1
#pragma unroll
        for (int h = 0; h < kPer; ++h) {
            const unsigned int j = tid + h * kBlendThreads;
            if (rg.x + b * kBatch + j < rg.y) {
                cp_async16(&s_A[b & 1][j], gA + ci[h]);
                cp_async16(&s_B[b & 1][j], gB + ci[h]);
                cp_async4(&s_c[b & 1][j], cB + ci[h]);
            }
        }
        cp_async_commit();
    };
    auto load_positions = [&](unsigned int b, uint32_t (&ci)[kPer]) {
#pragma unroll
        for (int h = 0; h < kPer; ++h) {
            const unsigned int i = rg.x + b * kBatch + tid + h * kBlendThreads;
            if (i < rg.y) ci[h] = vals[i];
        }
    };
    uint32_t ci_next[kPer] = {};                                    // positions of the batch to stage next
    load_positions(0, ci_next);
    if (n_batches) stage_batch(0, ci_next);
    load_positions(1, ci_next);
    for (unsigned int b = 0; b < n_batches; ++b) {
        cp_async_wait_all();
        // barrier: batch b is complete in staging buffer b & 1 for every thread, and every warp is through with batch b - 1
        if (__syncthreads_count(!warp_done) == 0) break;
        if (b + 1 < n_batches) {
            stage_batch(b + 1, ci_next);
            load_positions(b + 2, ci_next);
        }
        if (warp_done) continue;
        const unsigned int base = rg.x + b * kBatch;
        const unsigned int m = min((unsigned int)kBatch, rg.y - base);
        const float4 *recA = s_A[b & 1], *recB = s_B[b & 1];
        const float *recC = s_c[b & 1];

        unsigned int cnt = 0, clampy = 0;                       // clampy: a survivor waiting in the buffer may reach the 0.99 clamp
        for (unsigned int j0 = 0; j0 < m; j0 += 32) {
            // ---- filter: can Gaussian j0 + lane reach alpha >= 1/255 somewhere on this warp's strip
            // (a lane beyond the batch's end tests the last entry once more and drops it: no divergent region)
            const unsigned int j = min(j0 + lane, m - 1u);
            bool hit, near_one;
            float4 h0, h1, c;
            {
                float4 a = recA[j];
                const float4 b = recB[j];
                a.x -= x0c; a.y -= y0c;                              // relative to the tile's first pixel centre
                // the four rows as two packed pairs (FADD2 / FMUL2 / FFMA2: the kernel is bound by issue slots, and a
                // packed instruction is the same IEEE operation on both halves -- same bits as the scalar sequence)
                const float dy0 = a.y - row0;
                const float2 dyA = make_float2(dy0, dy0 - 1.0f), dyB = __fadd2_rn(make_float2(dy0, dy0), make_float2(-2.0f, -3.0f));
                const float2 kk = make_float2(a.z, a.z), ax = make_float2(a.x, a.x);
                const float2 cA = __ffma2_rn(kk, dyA, ax), cB2 = __ffma2_rn(kk, dyB, ax);
                const float2 dd = make_float2(b.x, b.x), lo = make_float2(b.y, b.y);
                const float2 eA = __ffma2_rn(dd, __fmul2_rn(dyA, dyA), lo), eB = __ffma2_rn(dd, __fmul2_rn(dyB, dyB), lo);
                h0 = make_float4(cA.x, cA.y, eA.x, eA.y);
                h1 = make_float4(cB2.x, cB2.y, eB.x, eB.y);
                // min over the row's 16 pixel columns x = 0..15 of |c_r - x|
                const float2 m15 = make_float2(-15.0f, -15.0f);
                const float2 tA = __fadd2_rn(cA, m15), tB = __fadd2_rn(cB2, m15);
                const float2 wA = make_float2(fmaxf(fmaxf(tA.x, -cA.x), 0.0f), fmaxf(fmaxf(tA.y, -cA.y), 0.0f));
                const float2 wB = make_float2(fmaxf(fmaxf(tB.x, -cB2.x), 0.0f), fmaxf(fmaxf(tB.y, -cB2.y), 0.0f));
                const float2 aa = make_float2(a.w, a.w);
                const float2 bA = __ffma2_rn(aa, __fmul2_rn(wA, wA), eA), bB = __ffma2_rn(aa, __fmul2_rn(wB, wB), eB);
                const float best = fmaxf(fmaxf(bA.x, bA.y), fmaxf(bB.x, bB.y));
                hit = best >= kThr && j0 + lane < m;
                near_one = b.y > -0.0146f;                           // log2(0.99) = -0.014500, ex2.approx is good to 2^-22
                c = make_float4(a.w, b.z, b.w, recC[j]);
            }
            const unsigned int bal = __ballot_sync(0xffffffffu, hit);
            if (hit) {
                const unsigned int slot = cnt + __popc(bal & ((1u << lane) - 1));
                my_buf[3 * slot] = h0; my_buf[3 * slot + 1] = h1; my_buf[3 * slot + 2] = c;
                if (COUNT) s_idx[warp][slot] = (unsigned short)j;
            }
            cnt += __popc(bal);
            clampy |= __ballot_sync(0xffffffffu, hit && near_one);
            // ---- evaluate when the next step might not fit (or at the end of the batch)
            if (cnt > kFlush || j0 + 32 >= m) {
                __syncwarp();
                if (clampy) evaluate(cnt, base - rg.x, std::true_type{});
                else evaluate(cnt, base - rg.x, std::false_type{});
                cnt = 0; clampy = 0;
                warp_done = __all_sync(0xffffffffu, T.x < 1e-4f && T.y < 1e-4f);
                if (warp_done) break;
                __syncwarp();
            }
        }
    }
    if (!RESUME && partial) {
        // the sorted prefix is used up: is any pixel of the tile still alive?  Then the rest of the list is wanted
        if (__syncthreads_or(!(T.x < 1e-4f && T.y < 1e-4f))) {
            ws.tile_state[(size_t)tile * 256 + 2 * tid] = make_float4(T.x, cr.x, cg.x, cb2.x);
            ws.tile_state[(size_t)tile * 256 + 2 * tid + 1] = make_float4(T.y, cr.y, cg.y, cb2.y);
            if (tid == 0) { ws.lazy[tile].w = 1u; ws.todo[atomicAdd(&ws.hdr->n_todo, 1u)] = (unsigned int)tile; }
            return;                                     // k_blend_rest writes the pixels
        }
    }
    const bool done0 = T.x < 1e-4f, done1 = T.y < 1e-4f;
    const float T0 = T.x, T1 = T.y, r0 = cr.x, r1 = cr.y, g0 = cg.x, g1 = cg.y, b0 = cb2.x, b1 = cb2.y;
    const size_t plane = (size_t)W * out_rows;          // out holds image rows [out_row0, out_row0 + out_rows) of every plane
    if (in0) {
        const size_t o = (size_t)(py0 - out_row0) * W + px;
        out[o] = fmaf(T0, bg0, r0); out[plane + o] = fmaf(T0, bg1, g0); out[2 * plane + o] = fmaf(T0, bg2, b0);
    }
    if (in1) {
        const size_t o = (size_t)(py1 - out_row0) * W + px;
        out[o] = fmaf(T1, bg0, r1); out[plane + o] = fmaf(T1, bg1, g1); out[2 * plane + o] = fmaf(T1, bg2, b1);
    }
    if (COUNT) {
        // E as the oracle defines it: list entries visited before the pixel terminated (filtered ones included)
        if (in0 && !done0) n_eval += rg.y - rg.x;
        if (in1 && !done1) n_eval += rg.y - rg.x;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            n_eval += __shfl_xor_sync(0xffffffffu, n_eval, o);
            n_blend += __shfl_xor_sync(0xffffffffu, n_blend, o);
        }
        if (lane == 0) {
            atomicAdd(&ws.hdr->evals, (unsigned long long)n_eval);
            atomicAdd(&ws.hdr->blends, (unsigned long long)n_blend);
        }
    }
}

template <bool COUNT>
__global__ void __launch_bounds__(kBlendThreads, kBlendMinBlocks)
k_blend(const WorkspaceDev ws, float *__restrict__ out, int W, int H, int TX, int n_tiles,
        float bg0, float bg1, float bg2, int tile0, int out_row0, int out_rows, int lazy)
{
    // the grid covers the frame's strip of tile rows
    cudaGridDependencySynchronize();
    // the NEXT frame's counters start at zero (this frame's header stays for flod_get_stats)
    if (blockIdx.x == 0 && threadIdx.x < sizeof(FrameHeader) / sizeof(unsigned int)) reinterpret_cast<unsigned int *>(ws.hdr_next)[threadIdx.x] = 0u;
    blend_tile<COUNT, false>(ws, out, W, H, TX, n_tiles, bg0, bg1, bg2, tile0 + (int)blockIdx.x, out_row0, out_rows, lazy);
}

// Second round of blend-driven ordering: a small persistent grid walks the tiles that asked for the rest of their list
// (ws.todo), so that a frame without any costs one short launch.
__global__ void __launch_bounds__(kBlendThreads, kBlendMinBlocks)
k_blend_rest(const WorkspaceDev ws, float *__restrict__ out, int W, int H, int TX, int n_tiles,
             float bg0, float bg1, float bg2, int out_row0, int out_rows)
{
    cudaGridDependencySynchronize();
    const unsigned int n_todo = ws.hdr->n_todo;
    for (unsigned int w = blockIdx.x; w < n_todo; w += gridDim.x) {
        blend_tile<false, true>(ws, out, W, H, TX, n_tiles, bg0, bg1, bg2, (int)ws.todo[w], out_row0, out_rows, 1);
        __syncthreads();                                // the staging buffers are reused by the next tile
    }
}

int launch_blend(const Context &c, const FrameParams &p, float *out_rgb, cudaStream_t s)
{
    const int tile0 = p.ty_begin * p.TX, n_tiles = p.ty_end * p.TX, grid = n_tiles - tile0;
    if (grid <= 0) return 0;
    if (c.flags & FLOD_OPT_COUNT)
        launch_pdl(k_blend<true>, grid, kBlendThreads, 0, s, c.ws, out_rgb, p.W, p.H, p.TX, n_tiles,
                   p.bg[0], p.bg[1], p.bg[2], tile0, p.out_row0, p.out_rows, 0);
    else
        launch_pdl(k_blend<false>, grid, kBlendThreads, 0, s, c.ws, out_rgb, p.W, p.H, p.TX, n_tiles,
                   p.bg[0], p.bg[1], p.bg[2], tile0, p.out_row0, p.out_rows, p.lazy_sort);
    return 1;
}

// second round of a lazy frame: the tiles the first round left unfinished (all other CTAs exit at once)
int launch_blend_rest(const Context &c, const FrameParams &p, float *out_rgb, cudaStream_t s)
{
    const int tile0 = p.ty_begin * p.TX, n_tiles = p.ty_end * p.TX, grid = n_tiles - tile0;
    if (grid <= 0 || !p.lazy_sort) return 0;
    launch_pdl(k_blend_rest, min(grid, 4 * c.sm_count), kBlendThreads, 0, s, c.ws, out_rgb, p.W, p.H, p.TX, n_tiles,
               p.bg[0], p.bg[1], p.bg[2], p.out_row0, p.out_rows);
    return 1;
}

}  // namespace flod
