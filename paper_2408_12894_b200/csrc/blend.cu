// Step a9: per-tile front-to-back alpha blending with early transmittance termination.
// Eq. 2: alpha = o exp(-1/2 d^T Sigma'^-1 d); "alpha blending the projected Gaussians in depth
// order"; clamp 0.99, skip below 1/255, stop after T < 1e-4 (R11, R12).
//
// One CTA of 128 threads owns one 16x16 tile; a thread owns two vertically adjacent pixels, a warp a 16x4 strip.
// The tile's sorted list is consumed in batches of 256: threads fetch compact indices (coalesced) and gather the
// 36 B of blend features per Gaussian (L2-resident) into shared memory.  Each warp then FILTERS the batch against
// its own strip -- a lane tests 8 Gaussians with the exact row-segment bound of the factorised exponent
//     e(x, y) = log2(o) - a2 w^2 - d2 dy^2,   w = (mu'x - x) + k dy          (DESIGN R25)
// (min over x in the strip of |w| is closed-form) and the survivors are ballot-compacted, in order, into a
// per-warp index list.  Only those are evaluated per pixel.  A filtered-out Gaussian has alpha < 2^-0.001 / 255 on
// every pixel of the strip, so the image is bit-identical to the unfiltered loop.  A warp whose 64 pixels have
// all terminated skips filter and loop; the CTA stops when every warp has.
#include "flod_internal.cuh"

namespace flod {

constexpr int kBlendThreads = 128;
constexpr int kBatch = 256;
constexpr int kBlendWarps = kBlendThreads / 32;
constexpr float kTwo100 = 1.2676506002282294e30f;   // 2^100

// 2^x on the MUFU unit (x <= 0 here; results below 2^-126 flush to 0, far under the 1/255 skip threshold)
__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <bool COUNT>
__global__ void __launch_bounds__(kBlendThreads)
k_blend(const WorkspaceDev ws, float *__restrict__ out, int W, int H, int TX, int n_tiles,
        float bg0, float bg1, float bg2)
{
    // one 48-byte record per Gaussian of the batch: (mu'x, mu'y, k, a2 | d2, log2 o, r, g | b, -, -, -)
    __shared__ float4 s_rec[kBatch * 3];
    __shared__ unsigned short s_list[kBlendWarps][kBatch];   // per warp: byte offsets of the surviving records

    const int tile = blockIdx.x;
    if (tile >= n_tiles || ws.hdr->overflow) return;   // an overflowed frame is undefined: its lists were not sorted
    const int tx = tile % TX, ty = tile / TX;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // warp = rows 4w..4w+3 of the tile; lanes 0-15 rows (4w, 4w+1), lanes 16-31 rows (4w+2, 4w+3)
    const int px = tx * kTile + (lane & 15);
    const int py0 = ty * kTile + warp * 4 + (lane >> 4) * 2, py1 = py0 + 1;
    const bool in0 = px < W && py0 < H, in1 = px < W && py1 < H;
    const float pxc = (float)px + 0.5f, pyc0 = (float)py0 + 0.5f, pyc1 = (float)py1 + 0.5f;
    // the warp's strip, for the filter: pixel centres x in [sx0, sx1], rows sy + {0,1,2,3}
    const float sx0 = (float)(tx * kTile) + 0.5f, sx1 = sx0 + 15.0f;
    const float sy = (float)(ty * kTile + warp * 4) + 0.5f;
    const float kThr = -7.994353436858858f - 1.0e-3f;  // log2(1/255) minus a safety margin

    const uint2 rg = ws.ranges[tile];
    const uint32_t *__restrict__ vals = ws.vals;
    const float4 *__restrict__ gA = ws.gA;
    const float4 *__restrict__ gB = ws.gB;
    const float *__restrict__ cB = ws.cB;

    // two pixels per thread, packed as float2 (.x = row py0, .y = row py1): the per-pixel arithmetic runs on the
    // packed FP32 instructions of sm_100 (FADD2 / FMUL2 / FFMA2: one issue slot for both pixels)
    float2 T = make_float2(1.0f, 1.0f), cr = make_float2(0.0f, 0.0f), cg = cr, cb2 = cr;
    const float2 npyc = make_float2(-pyc0, -pyc1);
    bool done0 = !in0, done1 = !in1;
    unsigned int n_eval = 0, n_blend = 0;
    unsigned short *my_list = s_list[warp];
    const unsigned char *rec_bytes = reinterpret_cast<const unsigned char *>(s_rec);
    // done pixels: thr = +huge, so that no alpha passes the skip test (live pixels: thr = 1/255)
    float thr0 = in0 ? (1.0f / 255.0f) : 3.0e38f, thr1 = in1 ? (1.0f / 255.0f) : 3.0e38f;

    for (unsigned int base = rg.x; base < rg.y; base += kBatch) {
        const bool warp_done = __all_sync(0xffffffffu, done0 && done1);
        if (__syncthreads_count(!warp_done) == 0) break;
        const unsigned int m = min((unsigned int)kBatch, rg.y - base);
#pragma unroll
        for (int h = 0; h < kBatch / kBlendThreads; ++h) {
            const unsigned int j = tid + h * kBlendThreads;
            if (j < m) {
                const uint32_t ci = vals[base + j];
                s_rec[3 * j] = gA[ci];
                s_rec[3 * j + 1] = gB[ci];
                s_rec[3 * j + 2].x = cB[ci];
            }
        }
        __syncthreads();
        if (warp_done) continue;

        // ---- filter: which Gaussians of the batch can reach alpha >= 1/255 somewhere on this warp's strip
        unsigned int cnt = 0;
#pragma unroll
        for (int i = 0; i < kBatch / 32; ++i) {
            const unsigned int j = lane + 32 * i;
            bool hit = false;
            if (j < m) {
                const float4 a = s_rec[3 * j];
                const float4 b = s_rec[3 * j + 1];
                const float dxl = a.x - sx1, dxh = a.x - sx0;        // range of (mu'x - x) over the strip
                float best = -INFINITY;
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                    const float dy = a.y - (sy + (float)rr);
                    const float kd = a.z * dy;
                    const float wmin = fmaxf(fmaxf(dxl + kd, -(dxh + kd)), 0.0f);
                    const float e = fmaf(a.w, wmin * wmin, fmaf(b.x, dy * dy, b.y));
                    best = fmaxf(best, e);
                }
                hit = best >= kThr;
            }
            const unsigned int bal = __ballot_sync(0xffffffffu, hit);
            if (hit) my_list[cnt + __popc(bal & ((1u << lane) - 1))] = (unsigned short)(j * 48u);
            cnt += __popc(bal);
        }
        __syncwarp();

        // ---- evaluate the survivors.  a.w and b.x are <= 0 (k_geometry clamps them), so e <= log2 o: q >= 0 holds
        // by construction and alpha needs the 0.99 clamp only.  A pixel that is done or below 1/255 blends alpha = 0.
#pragma unroll 2
        for (unsigned int t = 0; t < cnt; ++t) {
            const unsigned int off = my_list[t];
            const float4 a = *reinterpret_cast<const float4 *>(rec_bytes + off);
            const float4 b = *reinterpret_cast<const float4 *>(rec_bytes + off + 16);
            const float cbj = *reinterpret_cast<const float *>(rec_bytes + off + 32);
            const float dx = a.x - pxc;
            const float2 dy = __fadd2_rn(make_float2(a.y, a.y), npyc);
            const float2 w = __ffma2_rn(make_float2(a.z, a.z), dy, make_float2(dx, dx));
            const float2 e = __ffma2_rn(make_float2(a.w, a.w), __fmul2_rn(w, w),
                                        __ffma2_rn(make_float2(b.x, b.x), __fmul2_rn(dy, dy), make_float2(b.y, b.y)));
            float al0 = fminf(ex2(e.x), 0.99f), al1 = fminf(ex2(e.y), 0.99f);
            al0 = al0 >= thr0 ? al0 : 0.0f;
            al1 = al1 >= thr1 ? al1 : 0.0f;
            const float2 wgt = __fmul2_rn(T, make_float2(al0, al1));
            cr = __ffma2_rn(wgt, make_float2(b.z, b.z), cr);
            cg = __ffma2_rn(wgt, make_float2(b.w, b.w), cg);
            cb2 = __ffma2_rn(wgt, make_float2(cbj, cbj), cb2);
            T = __fadd2_rn(T, make_float2(-wgt.x, -wgt.y));           // T (1 - alpha)
            if (COUNT) {
                n_blend += (al0 > 0.0f ? 1u : 0u) + (al1 > 0.0f ? 1u : 0u);
                if (thr0 < 1.0f && T.x < 1e-4f) n_eval += (base - rg.x) + off / 48u + 1;
                if (thr1 < 1.0f && T.y < 1e-4f) n_eval += (base - rg.x) + off / 48u + 1;
            }
            // blend, then stop (R12): (1e-4 - T) 2^100 is positive exactly when T < 1e-4 (the scaling by a power of
            // two and the difference of the two products are exact up to one rounding that keeps the sign), and
            // then at least 2^-37 2^100 > 0.99
            const float2 stop = __ffma2_rn(T, make_float2(-kTwo100, -kTwo100), make_float2(1e-4f * kTwo100, 1e-4f * kTwo100));
            thr0 = fmaxf(thr0, stop.x);
            thr1 = fmaxf(thr1, stop.y);
        }
        done0 = thr0 > 1.0f; done1 = thr1 > 1.0f;
    }
    const float T0 = T.x, T1 = T.y, r0 = cr.x, r1 = cr.y, g0 = cg.x, g1 = cg.y, b0 = cb2.x, b1 = cb2.y;
    const size_t plane = (size_t)W * H;
    if (in0) {
        const size_t o = (size_t)py0 * W + px;
        out[o] = fmaf(T0, bg0, r0); out[plane + o] = fmaf(T0, bg1, g0); out[2 * plane + o] = fmaf(T0, bg2, b0);
    }
    if (in1) {
        const size_t o = (size_t)py1 * W + px;
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

int launch_blend(const Context &c, const FrameParams &p, float *out_rgb, cudaStream_t s)
{
    const int n_tiles = p.TX * p.TY;
    if (c.flags & FLOD_OPT_COUNT)
        k_blend<true><<<n_tiles, kBlendThreads, 0, s>>>(c.ws, out_rgb, p.W, p.H, p.TX, n_tiles,
                                                        p.bg[0], p.bg[1], p.bg[2]);
    else
        k_blend<false><<<n_tiles, kBlendThreads, 0, s>>>(c.ws, out_rgb, p.W, p.H, p.TX, n_tiles,
                                                         p.bg[0], p.bg[1], p.bg[2]);
    return 1;
}

}  // namespace flod
