// Step a9: per-tile front-to-back alpha blending with early transmittance termination.
// Eq. 2: alpha = o exp(-1/2 d^T Sigma'^-1 d); "alpha blending the projected Gaussians in depth
// order"; clamp 0.99, skip below 1/255, stop after T < 1e-4 (R11, R12).
//
// One CTA of 256 threads owns one 16x16 tile (thread = pixel).  The tile's sorted list is consumed in batches
// of 256: each thread fetches one compact index (coalesced), gathers that Gaussian's 36 B of blend features
// (L2-resident: the compacted feature arrays of a frame are ~50 MB) into shared memory, then every pixel walks
// the batch from shared memory (broadcast reads).  The exponent is evaluated in the factorised base-2 form of
// DESIGN R25:   e = log2(o) - (a2 w^2 + d2 dy^2),  w = dx + k dy,  alpha = min(0.99, 2^min(e, log2 o)).
// A warp whose 32 pixels have all terminated stops issuing math; the CTA stops when every warp has.
#include "flod_internal.cuh"

namespace flod {

constexpr int kBlendThreads = 256;

// 2^x on the MUFU unit (x <= 0 here; results below 2^-126 flush to 0, far under the 1/255 skip threshold)
__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <bool COUNT>
__global__ void __launch_bounds__(kBlendThreads)
k_blend(const WorkspaceDev ws, int buf, float *__restrict__ out, int W, int H, int TX, int n_tiles,
        float bg0, float bg1, float bg2)
{
    __shared__ float4 s_a[kBlendThreads];
    __shared__ float4 s_b[kBlendThreads];
    __shared__ float s_c[kBlendThreads];

    const int tile = blockIdx.x;
    if (tile >= n_tiles) return;
    const int tx = tile % TX, ty = tile / TX;
    const int tid = threadIdx.x;
    const int px = tx * kTile + (tid & 15), py = ty * kTile + (tid >> 4);
    const bool inside = px < W && py < H;
    const float pxc = (float)px + 0.5f, pyc = (float)py + 0.5f;

    const uint2 rg = ws.ranges[tile];
    const uint32_t *__restrict__ vals = (buf ? ws.vals[1] : ws.vals[0]);
    const float4 *__restrict__ gA = ws.gA;
    const float4 *__restrict__ gB = ws.gB;
    const float *__restrict__ cB = ws.cB;

    float T = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    bool done = !inside;
    unsigned int n_eval = 0, n_blend = 0;

    for (unsigned int base = rg.x; base < rg.y; base += kBlendThreads) {
        if (__syncthreads_count(!done) == 0) break;
        const unsigned int m = min((unsigned int)kBlendThreads, rg.y - base);
        if ((unsigned int)tid < m) {
            const uint32_t ci = vals[base + tid];
            s_a[tid] = gA[ci];
            s_b[tid] = gB[ci];
            s_c[tid] = cB[ci];
        }
        __syncthreads();
        if (!__all_sync(0xffffffffu, done)) {
            for (unsigned int j = 0; j < m; ++j) {
                const float4 a = s_a[j];
                const float4 b = s_b[j];
                const float dx = a.x - pxc, dy = a.y - pyc;
                const float w = fmaf(a.z, dy, dx);
                float e = b.y - fmaf(a.w, w * w, b.x * (dy * dy));
                e = fminf(e, b.y);                                   // q >= 0 (oracle clamps q at 0)
                float alpha = fminf(ex2(e), 0.99f);
                if (COUNT && !done) ++n_eval;
                if (done || alpha < (1.0f / 255.0f)) continue;
                const float wgt = T * alpha;
                Cr = fmaf(wgt, b.z, Cr);
                Cg = fmaf(wgt, b.w, Cg);
                Cb = fmaf(wgt, s_c[j], Cb);
                T = T - wgt;                                         // T (1 - alpha)
                if (COUNT) ++n_blend;
                if (T < 1e-4f) done = true;                          // blend, then stop (R12)
            }
        }
    }
    if (inside) {
        const size_t o = (size_t)py * W + px, plane = (size_t)W * H;
        out[o] = fmaf(T, bg0, Cr);
        out[plane + o] = fmaf(T, bg1, Cg);
        out[2 * plane + o] = fmaf(T, bg2, Cb);
    }
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            n_eval += __shfl_xor_sync(0xffffffffu, n_eval, o);
            n_blend += __shfl_xor_sync(0xffffffffu, n_blend, o);
        }
        if ((tid & 31) == 0) {
            atomicAdd(&ws.hdr->evals, (unsigned long long)n_eval);
            atomicAdd(&ws.hdr->blends, (unsigned long long)n_blend);
        }
    }
}

int launch_blend(const Context &c, const FrameParams &p, int final_buf, float *out_rgb, cudaStream_t s)
{
    const int n_tiles = p.TX * p.TY;
    if (c.flags & FLOD_OPT_COUNT)
        k_blend<true><<<n_tiles, kBlendThreads, 0, s>>>(c.ws, final_buf, out_rgb, p.W, p.H, p.TX, n_tiles,
                                                        p.bg[0], p.bg[1], p.bg[2]);
    else
        k_blend<false><<<n_tiles, kBlendThreads, 0, s>>>(c.ws, final_buf, out_rgb, p.W, p.H, p.TX, n_tiles,
                                                         p.bg[0], p.bg[1], p.bg[2]);
    return 1;
}

}  // namespace flod
