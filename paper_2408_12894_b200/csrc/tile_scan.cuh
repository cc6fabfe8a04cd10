// Steps a5 + a8: the 2-D prefix sum of the difference grid written by k_geometry = pairs per tile; the
// exclusive scan over the tiles in row-major order = [start, end) of every tile's list (the ranges of step a8, known
// before any pair exists); the append counters of k_duplicate are initialised here too.
//
// Run by ONE block of k_colour (block 0, so that it starts first): 65 KB of traffic and a few microseconds of pure
// latency, hidden under the HBM-bound colour blocks instead of sitting on the critical path as a kernel of its own.
// Works in place on ws.tile_cnt (global memory, L2-resident), any grid size, any block size that is a multiple of 32.
#pragma once
#include "flod_internal.cuh"

namespace flod {

// rowwise: the grid holds one +1 / -1 pair per (Gaussian, tile row) (pair rule 2), so the prefix along x alone gives the
// counts; otherwise +1 -1 -1 +1 at the corners of every rect (pair rule 1) and the prefix runs along x, then y.
__device__ __forceinline__ void tile_scan_block(const WorkspaceDev &ws, int TX, int TY, unsigned int max_pairs, bool rowwise)
{
    __shared__ unsigned long long s_wtot[32];
    __shared__ unsigned int s_long;                            // pairs that sit in lists longer than kSortCap (saturating)
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
    const int gw = TX + 1, gh = TY + 1;
    if (tid == 0) s_long = 0;
    int *__restrict__ diff = ws.tile_diff;
    int *cnt = ws.tile_cnt;

    // ---- prefix along x: a warp owns a row, 32 cells per step, carry in a register
    for (int y = warp; y < gh; y += nwarp) {
        int carry = 0;
        for (int x0 = 0; x0 < gw; x0 += 32) {
            const int x = x0 + lane;
            int v = 0;
            if (x < gw) { v = diff[(size_t)(y * gw + x) * kCtrStride]; diff[(size_t)(y * gw + x) * kCtrStride] = 0; }   // read once: ready for the next frame
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, v, o);
                if (lane >= o) v += t;
            }
            v += carry;
            if (x < gw) cnt[y * gw + x] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
    }
    __syncthreads();
    // ---- prefix along y: a thread owns a column, eight independent loads in flight per step
    for (int x = tid; x < gw && !rowwise; x += nthr) {
        int run = 0;
        for (int y0 = 0; y0 < gh; y0 += 8) {
            int v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = y0 + k < gh ? cnt[(y0 + k) * gw + x] : 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                run += v[k];
                if (y0 + k < gh) cnt[(y0 + k) * gw + x] = run;        // = pairs of tile (x, y0 + k)
            }
        }
    }
    __syncthreads();
    // ---- plus the pairs of the small rects, which k_geometry counted per 2x2 tile group (read once: ready for the next frame)
    {
        const int GXs = (TX + 1) / 2, n_groups = GXs * ((TY + 1) / 2);
        for (int g = tid; g < n_groups; g += nthr) {
            float4 *line = reinterpret_cast<float4 *>(ws.cnt4 + (size_t)g * kCtrStride);
            const float4 c = *line;
            *line = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            const int x = 2 * (g % GXs), y = 2 * (g / GXs);
            cnt[y * gw + x] += (int)c.x;                       // (cells of the grid's last row / column hold 0: a rect ends inside the image)
            cnt[y * gw + x + 1] += (int)c.y;
            cnt[(y + 1) * gw + x] += (int)c.z;
            cnt[(y + 1) * gw + x + 1] += (int)c.w;
        }
    }
    __syncthreads();
    // ---- exclusive scan over the tiles; a thread owns a contiguous chunk
    const int T_n = TX * TY;
    const int per = (T_n + nthr - 1) / nthr;
    const int t0 = min(tid * per, T_n), t1 = min(t0 + per, T_n);
    unsigned long long sum = 0;
    for (int t = t0; t < t1; ++t) sum += (unsigned int)cnt[(t / TX) * gw + (t % TX)];
    unsigned long long incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_wtot[warp] = incl;
    __syncthreads();
    unsigned long long run = incl - sum, total = 0;
    for (int w = 0; w < nwarp; ++w) {
        const unsigned long long t = s_wtot[w];
        if (w < warp) run += t;
        total += t;
    }
    unsigned int too_long = 0;
    unsigned int in_long = 0;
    for (int t = t0; t < t1; ++t) {
        const unsigned int c = (unsigned int)cnt[(t / TX) * gw + (t % TX)];
        if (c > (unsigned int)kSortCap) in_long += min(c, 1u << 20);
        const unsigned int a = (unsigned int)min(run, (unsigned long long)max_pairs);
        const unsigned int b = (unsigned int)min(run + c, (unsigned long long)max_pairs);
        ws.ranges[t] = make_uint2(a, b);
        ws.cursor[t] = 0;                                      // k_duplicate_shared: entries appended so far
        if (c >= (1u << 24)) too_long = 1u;                    // k_geometry and k_duplicate count a tile's entries in a float
        run += c;
    }
    in_long = __reduce_add_sync(0xffffffffu, min(in_long, 1u << 26));
    if (lane == 0 && in_long) atomicAdd(&s_long, in_long);
    too_long = __syncthreads_or((int)too_long);
    // The append counters of the 2x2 tile groups (one float4, the target of k_duplicate's one atomic per group).  A frame
    // of at most 2^24 pairs counts in ABSOLUTE positions: the counters start at the tiles' range starts (exact as floats)
    // and the atomic returns the slot itself.  A larger frame counts from 0 and k_duplicate adds the range starts it reads
    // from ws.ranges.  (ws.ranges of the whole image are visible here: the barrier above.)
    const bool absolute = total <= (1ull << 24);
    const int GXs = (TX + 1) / 2, n_groups = GXs * ((TY + 1) / 2);
    for (int g = tid; g < n_groups; g += nthr) {
        const int x = 2 * (g % GXs), y = 2 * (g / GXs);
        const bool x1 = x + 1 < TX, y1 = y + 1 < TY;
        const unsigned int s00 = ws.ranges[y * TX + x].x, s10 = x1 ? ws.ranges[y * TX + x + 1].x : 0u;
        const unsigned int s01 = y1 ? ws.ranges[(y + 1) * TX + x].x : 0u, s11 = x1 && y1 ? ws.ranges[(y + 1) * TX + x + 1].x : 0u;
        float4 *line = reinterpret_cast<float4 *>(ws.cursor4 + (size_t)g * kCtrStride);
        line[0] = absolute ? make_float4((float)s00, (float)s10, (float)s01, (float)s11) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    }
    if (tid == 0) {
        // host memory, a hint for the next frame (flod_api.cu): blend-driven ordering pays when a good part of the pairs
        // sits in long lists (a coarse level alone), not for a few crowded tiles of a fine level
        // (written only when it changes: a store to host memory holds the kernel's completion back by microseconds)
        // (bit 1: the frame's mean rect exceeds ws.dup_large_area tiles -- the next frames launch k_duplicate_shared as well)
        const unsigned int hint = (((unsigned long long)s_long * 4ull >= total && s_long) ? 1u : 0u) |
                                  (total > (unsigned long long)ws.dup_large_area * ws.hdr->n_vis32 ? 2u : 0u);
        if (*ws.hint_state != (hint | 0x100u)) { *ws.hint_state = hint | 0x100u; *ws.long_hint = hint | 0x100u; }   // 0x100: a hint exists
        ws.hdr->n_pairs_clamped = (unsigned int)min(total, (unsigned long long)max_pairs);
        const unsigned int ovf = (total > max_pairs ? 1u : 0u) | (too_long ? 2u : 0u);
        ws.hdr->overflow = ovf;
        ws.hdr->cursor_abs = absolute ? 1u : 0u;
        *ws.ovf_out = ovf;                                     // read back with the image by flod_render_to_host*
    }
}

}  // namespace flod
