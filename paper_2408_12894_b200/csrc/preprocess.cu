// Steps a1-a4 of the hot path:
//   k_geometry  a1 level selection (Eq. 6-7), a2 cull + view transform, a3 EWA projection, conic,
//               tile rect; every visible Gaussian adds its rect to a 2-D difference grid of the tile counts
//               (four integer atomics whatever the rect size) and appends its index to the unordered visible list;
//   k_colour    a4 SH -> RGB over the visible list.
// One thread per scanned Gaussian, no inter-block dependency: records are written in place at the scan index.
//
// The geometry (a1-a3 and the rect) is the canonical fp32 sequence of DESIGN §2: each operation is one IEEE
// round-to-nearest binary32 operation (the *_rn intrinsics are never contracted into FMAs), in the written order.
#include "flod_internal.cuh"

namespace flod {

__device__ __forceinline__ float fmul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fadd(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float fsub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdiv_rn(a, b); }

// real SH constants of DESIGN R16
#define SH_C0 0.28209479177387814f    /* 1/2 sqrt(1/pi)        */
#define SH_C1 0.4886025119029199f     /* sqrt(3/(4 pi))        */
#define SH_C2A 1.0925484305920792f    /* 1/2 sqrt(15/pi)       */
#define SH_C2B 0.31539156525252005f   /* 1/4 sqrt(5/pi)        */
#define SH_C2C 0.5462742152960396f    /* 1/4 sqrt(15/pi)       */
#define SH_C3A 0.5900435899266435f    /* 1/4 sqrt(35/(2 pi))   */
#define SH_C3B 2.890611442640554f     /* 1/2 sqrt(105/pi)      */
#define SH_C3C 0.4570457994644658f    /* 1/4 sqrt(21/(2 pi))   */
#define SH_C3D 0.3731763325901154f    /* 1/4 sqrt(7/pi)        */
#define SH_C3E 1.445305721320277f     /* 1/4 sqrt(105/pi)      */

// The 16 real SH basis values of DESIGN R16 at the unit direction (x, y, z), up to degree DEG.
template <int DEG>
__device__ __forceinline__ void sh_basis(float x, float y, float z, float *Y)
{
    Y[0] = SH_C0;
    if constexpr (DEG >= 1) {
        Y[1] = -SH_C1 * y; Y[2] = SH_C1 * z; Y[3] = -SH_C1 * x;
    }
    if constexpr (DEG >= 2) {
        const float xx = x * x, yy = y * y, zz = z * z;
        Y[4] = SH_C2A * x * y;
        Y[5] = -SH_C2A * y * z;
        Y[6] = SH_C2B * (2.0f * zz - xx - yy);
        Y[7] = -SH_C2A * x * z;
        Y[8] = SH_C2C * (xx - yy);
        if constexpr (DEG >= 3) {
            Y[9] = -SH_C3A * y * (3.0f * xx - yy);
            Y[10] = SH_C3B * x * y * z;
            Y[11] = -SH_C3C * y * (4.0f * zz - xx - yy);
            Y[12] = SH_C3D * z * (2.0f * zz - 3.0f * xx - 3.0f * yy);
            Y[13] = -SH_C3C * x * (4.0f * zz - xx - yy);
            Y[14] = SH_C3E * z * (xx - yy);
            Y[15] = -SH_C3A * x * (xx - 3.0f * yy);
        }
    }
}

template <bool DEBUG>
__global__ void __launch_bounds__(kPreBlock)
k_geometry(const SceneDev sc, const WorkspaceDev ws, const __grid_constant__ FrameParams p)
{
    __shared__ unsigned int s_warp_vis[kPreBlock / 32];
    __shared__ unsigned int s_base;
    __shared__ unsigned int s_cnt[2];               // n_sel, n_front of the block
    __shared__ unsigned long long s_pairs;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { s_cnt[0] = 0; s_cnt[1] = 0; s_pairs = 0; }
    const int i = (int)(blockIdx.x * kPreBlock) + tid;

    bool vis = false, sel = false, front = false;
    unsigned int n_tiles = 0;
    float mx2 = 0, my2 = 0, pz = 0, cA = 0, cB = 0, cC = 0;
    int tx0 = 0, ty0 = 0, tx1 = 0, ty1 = 0;
    float wx = 0, wy = 0, wz = 0;                   // world-space mean (for the view direction)
    long long g = 0;

    if (i < p.n_scan) {
        g = p.first_gid + i;
        int lv = 0;
#pragma unroll 1
        while (lv < p.n_levels - 1 && i >= p.level_end[lv]) ++lv;
        wx = __ldg(sc.mx + g); wy = __ldg(sc.my + g); wz = __ldg(sc.mz + g);
        // ---- a1 (O1): Eq. 6 predicate on squared Euclidean distance to the reference
        {
            float dx = fsub(wx, p.ref[0]), dy = fsub(wy, p.ref[1]), dz = fsub(wz, p.ref[2]);
            float d2 = fadd(fadd(fmul(dx, dx), fmul(dy, dy)), fmul(dz, dz));
            sel = (d2 >= p.lo2[lv]) && (d2 < p.hi2[lv]);
        }
        if (DEBUG) ws.mask[g] = sel ? 1 : 0;
        if (sel) {
            // ---- a2 (O2): p = R mu + t
            const float *R = p.R;
            float px = fadd(fadd(fadd(fmul(R[0], wx), fmul(R[1], wy)), fmul(R[2], wz)), p.t[0]);
            float py = fadd(fadd(fadd(fmul(R[3], wx), fmul(R[4], wy)), fmul(R[5], wz)), p.t[1]);
            pz = fadd(fadd(fadd(fmul(R[6], wx), fmul(R[7], wy)), fmul(R[8], wz)), p.t[2]);
            front = pz > p.z_near;
            float kap = front ? __ldg(sc.kappa + g) : -1.0f;
            if (front && kap >= 0.0f) {
                float ix = fdiv(px, pz), iy = fdiv(py, pz);
                mx2 = fadd(fmul(p.fx, ix), p.cx);
                my2 = fadd(fmul(p.fy, iy), p.cy);
                // ---- a3 (O3): J at the clamped point, M = J R, Sigma' = M Sigma M^T + 0.3 I
                float u = fminf(fmaxf(ix, -p.limx), p.limx);
                float v = fminf(fmaxf(iy, -p.limy), p.limy);
                float j00 = fdiv(p.fx, pz);
                float j02 = -fdiv(fmul(p.fx, u), pz);
                float j11 = fdiv(p.fy, pz);
                float j12 = -fdiv(fmul(p.fy, v), pz);
                float m00 = fadd(fmul(j00, R[0]), fmul(j02, R[6]));
                float m01 = fadd(fmul(j00, R[1]), fmul(j02, R[7]));
                float m02 = fadd(fmul(j00, R[2]), fmul(j02, R[8]));
                float m10 = fadd(fmul(j11, R[3]), fmul(j12, R[6]));
                float m11 = fadd(fmul(j11, R[4]), fmul(j12, R[7]));
                float m12 = fadd(fmul(j11, R[5]), fmul(j12, R[8]));
                float Sxx = __ldg(sc.cov[0] + g), Sxy = __ldg(sc.cov[1] + g), Sxz = __ldg(sc.cov[2] + g);
                float Syy = __ldg(sc.cov[3] + g), Syz = __ldg(sc.cov[4] + g), Szz = __ldg(sc.cov[5] + g);
                float v0x = fadd(fadd(fmul(Sxx, m00), fmul(Sxy, m01)), fmul(Sxz, m02));
                float v0y = fadd(fadd(fmul(Sxy, m00), fmul(Syy, m01)), fmul(Syz, m02));
                float v0z = fadd(fadd(fmul(Sxz, m00), fmul(Syz, m01)), fmul(Szz, m02));
                float v1x = fadd(fadd(fmul(Sxx, m10), fmul(Sxy, m11)), fmul(Sxz, m12));
                float v1y = fadd(fadd(fmul(Sxy, m10), fmul(Syy, m11)), fmul(Syz, m12));
                float v1z = fadd(fadd(fmul(Sxz, m10), fmul(Syz, m11)), fmul(Szz, m12));
                float a = fadd(fadd(fadd(fmul(m00, v0x), fmul(m01, v0y)), fmul(m02, v0z)), 0.3f);
                float b = fadd(fadd(fmul(m10, v0x), fmul(m11, v0y)), fmul(m12, v0z));
                float c = fadd(fadd(fadd(fmul(m10, v1x), fmul(m11, v1y)), fmul(m12, v1z)), 0.3f);
                float det = fsub(fmul(a, c), fmul(b, b));
                if (det > 0.0f) {
                    cA = fdiv(c, det); cB = -fdiv(b, det); cC = fdiv(a, det);
                    // ---- O4: padded box of the alpha = 1/255 contour, in 16x16 tiles
                    float hx = fadd(fmul(__fsqrt_rn(fmul(kap, a)), 1.0009765625f), 0.015625f);
                    float hy = fadd(fmul(__fsqrt_rn(fmul(kap, c)), 1.0009765625f), 0.015625f);
                    float fTX = (float)p.TX, fTY = (float)p.TY;
                    float x0 = fminf(fmaxf(floorf(fmul(fsub(mx2, hx), 0.0625f)), 0.0f), fTX);
                    float x1 = fminf(fmaxf(fadd(floorf(fmul(fadd(mx2, hx), 0.0625f)), 1.0f), 0.0f), fTX);
                    float y0 = fminf(fmaxf(floorf(fmul(fsub(my2, hy), 0.0625f)), 0.0f), fTY);
                    float y1 = fminf(fmaxf(fadd(floorf(fmul(fadd(my2, hy), 0.0625f)), 1.0f), 0.0f), fTY);
                    tx0 = (int)x0; tx1 = (int)x1; ty0 = (int)y0; ty1 = (int)y1;
                    n_tiles = (unsigned int)((tx1 - tx0) * (ty1 - ty0));
                    vis = n_tiles > 0;
                }
            }
        }
    }

    // ---- per-visible records, in place at the scan index i
    if (vis) {
        // DESIGN R25: factorised exponent from the ROUNDED conic, derived in fp64, rounded once
        const double LOG2E = 1.4426950408889634;
        const double dA = (double)cA, dB = (double)cB, dC = (double)cC;
        const float kk = (float)(dB / dA);
        const float a2 = (float)(-0.5 * LOG2E * dA);                   // stored negated: e = log2 o + a2 w^2 + d2 dy^2
        // <= 0 so that q >= 0 holds by construction in k_blend (the oracle clamps q at 0; a conic left indefinite by
        // rounding differs from its clamp by less than R25's evaluation error)
        const float d2 = fminf((float)(-0.5 * LOG2E * (dC - dB * dB / dA)), 0.0f);
        ws.gA[i] = make_float4(mx2, my2, kk, a2);
        reinterpret_cast<float2 *>(ws.gB)[2 * (size_t)i] = make_float2(d2, __ldg(sc.l2o + g));   // (r, g) by k_colour
        ws.rect[i] = make_ushort4((unsigned short)tx0, (unsigned short)ty0, (unsigned short)tx1, (unsigned short)ty1);
        ws.depth[i] = __float_as_uint(pz);
        ws.dirgid[i] = make_float4(wx - p.centre[0], wy - p.centre[1], wz - p.centre[2], __uint_as_float((unsigned int)g));
        // a5, first half: +1 over the rect in the 2-D difference grid of the per-tile pair counts
        const int gw = p.TX + 1;
        atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx0) * kCtrStride, 1);
        atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx1) * kCtrStride, -1);
        atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx0) * kCtrStride, -1);
        atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx1) * kCtrStride, 1);
    }
    if (DEBUG && i < p.n_scan) {
        flod_dbg_projected d;
        d.gid = vis ? (uint32_t)g : 0xffffffffu; d.mu2d[0] = mx2; d.mu2d[1] = my2; d.depth = pz;
        d.conic[0] = cA; d.conic[1] = cB; d.conic[2] = cC; d.opacity = vis ? __ldg(sc.opacity + g) : 0.0f;
        d.rgb[0] = 0.0f; d.rgb[1] = 0.0f; d.rgb[2] = 0.0f;                                    // by k_colour
        d.rect[0] = tx0; d.rect[1] = ty0; d.rect[2] = tx1; d.rect[3] = ty1;
        ws.dbg[i] = d;
    }

    // ---- block-aggregated counters and the unordered visible list
    const unsigned int bv = __ballot_sync(0xffffffffu, vis);
    const unsigned int bs = __ballot_sync(0xffffffffu, sel), bf = __ballot_sync(0xffffffffu, front);
    unsigned int wp = n_tiles;                       // warp sum of the tile counts (a rect has < 2^20 tiles)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) wp += __shfl_xor_sync(0xffffffffu, wp, o);
    __syncthreads();                                 // s_cnt / s_pairs were zeroed by thread 0
    if (lane == 0) {
        s_warp_vis[warp] = __popc(bv);
        if (bs) atomicAdd(&s_cnt[0], __popc(bs));
        if (bf) atomicAdd(&s_cnt[1], __popc(bf));
        if (wp) atomicAdd(&s_pairs, (unsigned long long)wp);
    }
    __syncthreads();
    if (tid == 0) {
        unsigned int tot = 0;
#pragma unroll
        for (int w = 0; w < kPreBlock / 32; ++w) { const unsigned int t = s_warp_vis[w]; s_warp_vis[w] = tot; tot += t; }
        s_base = tot ? atomicAdd(&ws.hdr->n_vis32, tot) : 0u;
        if (s_cnt[0]) atomicAdd(&ws.hdr->n_sel, (unsigned long long)s_cnt[0]);
        if (s_cnt[1]) atomicAdd(&ws.hdr->n_front, (unsigned long long)s_cnt[1]);
        if (s_pairs) atomicAdd(&ws.hdr->n_pairs, s_pairs);
    }
    __syncthreads();
    if (vis) ws.vis_list[s_base + s_warp_vis[warp] + __popc(bv & ((1u << lane) - 1))] = (uint32_t)i;
}

// ---- a4: colour of every visible Gaussian.  rgb = max(0, 0.5 + sum_k Y_k(dir) sh_k)  (R16)
// LANES threads share one Gaussian.  LANES = 4 needs the degree-3 row layout written by the upload: the row is 12
// float4; float4 number (4 i + j), i = 0..2, holds floats [4 i, 4 i + 4) of the 12 floats (k, channel) of the
// coefficients k = 4 j .. 4 j + 3, so one load instruction of the 4 lanes reads 64 contiguous bytes.
template <int DEG, int LANES, bool DEBUG>
__global__ void __launch_bounds__(256)
k_colour(const SceneDev sc, const WorkspaceDev ws)
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    const unsigned int n_vis = ws.hdr->n_vis32;
    const unsigned int sub = threadIdx.x % LANES;
    const unsigned int per_block = 256 / LANES;
    for (unsigned int base = blockIdx.x * per_block; base < n_vis; base += gridDim.x * per_block) {
        const unsigned int slot = base + threadIdx.x / LANES;
        const bool ok = slot < n_vis;
        float r = 0.0f, g = 0.0f, b = 0.0f;
        unsigned int ci = 0;
        if (ok) {
            ci = ws.vis_list[slot];
            const float4 dg = ws.dirgid[ci];
            const float *row = sc.sh + (size_t)__float_as_uint(dg.w) * sc.sh_stride;
            float Y[K];
            const float inv = DEG >= 1 ? 1.0f / sqrtf(dg.x * dg.x + dg.y * dg.y + dg.z * dg.z) : 0.0f;
            if constexpr (LANES == 4) {
                static_assert(DEG == 3 || LANES == 1, "4-lane layout is degree 3 only");
                const float4 *r4 = reinterpret_cast<const float4 *>(row);
                const float4 f0 = __ldg(r4 + sub), f1 = __ldg(r4 + 4 + sub), f2 = __ldg(r4 + 8 + sub);
                sh_basis<DEG>(dg.x * inv, dg.y * inv, dg.z * inv, Y);
                const float y0 = sub == 0 ? Y[0] : sub == 1 ? Y[4] : sub == 2 ? Y[8] : Y[12];
                const float y1 = sub == 0 ? Y[1] : sub == 1 ? Y[5] : sub == 2 ? Y[9] : Y[13];
                const float y2 = sub == 0 ? Y[2] : sub == 1 ? Y[6] : sub == 2 ? Y[10] : Y[14];
                const float y3 = sub == 0 ? Y[3] : sub == 1 ? Y[7] : sub == 2 ? Y[11] : Y[15];
                r = fmaf(y0, f0.x, fmaf(y1, f0.w, fmaf(y2, f1.z, y3 * f2.y)));
                g = fmaf(y0, f0.y, fmaf(y1, f1.x, fmaf(y2, f1.w, y3 * f2.z)));
                b = fmaf(y0, f0.z, fmaf(y1, f1.y, fmaf(y2, f2.x, y3 * f2.w)));
            } else {
                constexpr int NF = (3 * K + 3) / 4 * 4;
                float f[NF];
                const float4 *r4 = reinterpret_cast<const float4 *>(row);
#pragma unroll
                for (int q = 0; q < NF / 4; ++q) {
                    const float4 t = __ldg(r4 + q);
                    f[4 * q] = t.x; f[4 * q + 1] = t.y; f[4 * q + 2] = t.z; f[4 * q + 3] = t.w;
                }
                sh_basis<DEG>(dg.x * inv, dg.y * inv, dg.z * inv, Y);
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    r = fmaf(Y[k], f[3 * k], r);
                    g = fmaf(Y[k], f[3 * k + 1], g);
                    b = fmaf(Y[k], f[3 * k + 2], b);
                }
            }
        }
        if constexpr (LANES == 4) {
#pragma unroll
            for (int o = 1; o < 4; o <<= 1) {
                r += __shfl_xor_sync(0xffffffffu, r, o);
                g += __shfl_xor_sync(0xffffffffu, g, o);
                b += __shfl_xor_sync(0xffffffffu, b, o);
            }
        }
        if (ok && sub == 0) {
            r = fmaxf(r + 0.5f, 0.0f); g = fmaxf(g + 0.5f, 0.0f); b = fmaxf(b + 0.5f, 0.0f);
            reinterpret_cast<float2 *>(ws.gB)[2 * (size_t)ci + 1] = make_float2(r, g);
            ws.cB[ci] = b;
            if (DEBUG) { ws.dbg[ci].rgb[0] = r; ws.dbg[ci].rgb[1] = g; ws.dbg[ci].rgb[2] = b; }
        }
    }
}

int launch_geometry(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    if (c.flags & FLOD_OPT_DEBUG) k_geometry<true><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.scene, c.ws, p);
    else k_geometry<false><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.scene, c.ws, p);
    return 1;
}

template <int DEG, int LANES>
static void launch_colour_t(const Context &c, int grid, cudaStream_t s)
{
    if (c.flags & FLOD_OPT_DEBUG) k_colour<DEG, LANES, true><<<grid, 256, 0, s>>>(c.scene, c.ws);
    else k_colour<DEG, LANES, false><<<grid, 256, 0, s>>>(c.scene, c.ws);
}

int launch_colour(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    const int grid = c.sm_count * 8;
    switch (c.sh_degree) {
        case 0: launch_colour_t<0, 1>(c, grid, s); break;
        case 1: launch_colour_t<1, 1>(c, grid, s); break;
        case 2: launch_colour_t<2, 1>(c, grid, s); break;
        default: launch_colour_t<3, 4>(c, grid, s); break;
    }
    return 1;
}

}  // namespace flod
