// Steps a1-a6 of the hot path in ONE kernel:
//   a1 level selection (Eq. 6-7)         a2 cull + view transform
//   a3 EWA projection, conic, tile rect     a4 SH -> RGB
//   a5 exclusive scan of visible / tile counts      a6 (tile | depth) key duplication
// One thread per scanned Gaussian; a decoupled look-back over blocks (ordered by an atomic ticket) gives every
// block its compact-index base and pair base, so projected features are written compacted and pairs are emitted
// in ascending gid, row-major tile order with a block-cooperative, perfectly coalesced expansion.
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

template <int DEG>
__device__ __forceinline__ void sh_to_rgb(const float *__restrict__ row, float dx, float dy, float dz, float rgb[3])
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    constexpr int NF = (3 * K + 3) / 4 * 4;
    float f[NF];
    const float4 *r4 = reinterpret_cast<const float4 *>(row);
#pragma unroll
    for (int i = 0; i < NF / 4; ++i) {
        float4 v = __ldg(r4 + i);
        f[4 * i] = v.x; f[4 * i + 1] = v.y; f[4 * i + 2] = v.z; f[4 * i + 3] = v.w;
    }
    float Y[K];
    Y[0] = SH_C0;
    if constexpr (DEG >= 1) {
        float inv = 1.0f / sqrtf(dx * dx + dy * dy + dz * dz);
        float x = dx * inv, y = dy * inv, z = dz * inv;
        Y[1] = -SH_C1 * y; Y[2] = SH_C1 * z; Y[3] = -SH_C1 * x;
        if constexpr (DEG >= 2) {
            float xx = x * x, yy = y * y, zz = z * z;
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
    float r = 0.5f, g = 0.5f, b = 0.5f;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        r = fmaf(Y[k], f[3 * k], r);
        g = fmaf(Y[k], f[3 * k + 1], g);
        b = fmaf(Y[k], f[3 * k + 2], b);
    }
    rgb[0] = fmaxf(r, 0.0f); rgb[1] = fmaxf(g, 0.0f); rgb[2] = fmaxf(b, 0.0f);
}

constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagIncl = 2ull << 62, kFlagMask = 3ull << 62;
constexpr int kVisShift = 36;
constexpr unsigned long long kPairMask = (1ull << kVisShift) - 1, kVisMask = (1ull << 26) - 1;

template <int DEG, bool DEBUG>
__global__ void __launch_bounds__(kPreBlock)
k_preprocess(const SceneDev sc, const WorkspaceDev ws, const __grid_constant__ FrameParams p)
{
    __shared__ unsigned int s_vb;
    __shared__ unsigned long long s_warp_tot[kPreBlock / 32];
    __shared__ unsigned long long s_base;           // packed exclusive prefix of this block (status format)
    __shared__ unsigned int s_incl[kPreBlock];      // inclusive pair scan by local visible rank
    __shared__ unsigned int s_rect[kPreBlock];      // tx0 | ty0 << 16
    __shared__ unsigned int s_wd[kPreBlock];        // rect width
    __shared__ unsigned int s_depth[kPreBlock];     // depth bits
    __shared__ unsigned int s_cnt[2];               // n_sel, n_front of the block

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { s_vb = atomicAdd(&ws.hdr->pre_ticket, 1u); s_cnt[0] = 0; s_cnt[1] = 0; }
    __syncthreads();
    const unsigned int vb = s_vb;
    const int i = (int)(vb * kPreBlock) + tid;

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

    // ---- a5: block scan of (visible, n_tiles), packed vis << 40 | tiles
    unsigned long long v = ((unsigned long long)(vis ? 1 : 0) << 40) | n_tiles;
    unsigned long long incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long n = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += n;
    }
    if (lane == 31) s_warp_tot[warp] = incl;
    {
        unsigned int bs = __ballot_sync(0xffffffffu, sel), bf = __ballot_sync(0xffffffffu, front);
        if (lane == 0) { atomicAdd(&s_cnt[0], __popc(bs)); atomicAdd(&s_cnt[1], __popc(bf)); }
    }
    __syncthreads();
    unsigned long long warp_off = 0, block_tot = 0;
#pragma unroll
    for (int w = 0; w < kPreBlock / 32; ++w) {
        unsigned long long t = s_warp_tot[w];
        if (w < warp) warp_off += t;
        block_tot += t;
    }
    incl += warp_off;
    const unsigned int block_vis = (unsigned int)(block_tot >> 40);
    const unsigned long long block_pairs = block_tot & ((1ull << 40) - 1);
    const unsigned int rank = (unsigned int)(incl >> 40) - (vis ? 1u : 0u);          // local visible rank
    const unsigned int pair_incl = (unsigned int)(incl & ((1ull << 40) - 1));

    // ---- decoupled look-back over the blocks before this one (warp 0)
    if (warp == 0) {
        const unsigned long long agg = ((unsigned long long)block_vis << kVisShift) | block_pairs;
        unsigned long long excl = 0;
        if (vb == 0) {
            if (lane == 0) atomicExch(ws.pre_status + 0, kFlagIncl | agg);
        } else {
            if (lane == 0) atomicExch(ws.pre_status + vb, kFlagAgg | agg);
            long long j = (long long)vb - 1;
            while (true) {
                long long idx = j - lane;
                unsigned long long st = kFlagIncl;                 // lanes before block 0 read "inclusive 0"
                if (idx >= 0) {
                    volatile unsigned long long *ptr = ws.pre_status + idx;
                    do { st = *ptr; } while ((st & kFlagMask) == 0);
                }
                unsigned int incl_mask = __ballot_sync(0xffffffffu, (st & kFlagMask) == kFlagIncl);
                unsigned long long val = st & ~kFlagMask;
                int first = incl_mask ? (__ffs(incl_mask) - 1) : 31;
                unsigned long long contrib = (lane <= first) ? val : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
                excl += contrib;
                if (incl_mask) break;
                j -= 32;
            }
            if (lane == 0) atomicExch(ws.pre_status + vb, kFlagIncl | (excl + agg));
        }
        if (lane == 0) {
            s_base = excl;
            atomicAdd(&ws.hdr->n_sel, (unsigned long long)s_cnt[0]);
            atomicAdd(&ws.hdr->n_front, (unsigned long long)s_cnt[1]);
            if (vb == (unsigned int)p.n_pre_blocks - 1) {          // the last block knows the frame totals
                unsigned long long tot = excl + agg;
                unsigned long long np = tot & kPairMask;
                ws.hdr->n_vis = (tot >> kVisShift) & kVisMask;
                ws.hdr->n_pairs = np;
                ws.hdr->n_pairs_clamped = (unsigned int)(np < p.max_pairs ? np : p.max_pairs);
                ws.hdr->overflow = np > p.max_pairs ? 1u : 0u;
            }
        }
    }
    __syncthreads();
    const unsigned long long base = s_base;
    const unsigned int vis_base = (unsigned int)((base >> kVisShift) & kVisMask);
    const unsigned long long pair_base = base & kPairMask;

    // ---- write the compacted blend features (+ a4 colour) of visible Gaussians
    if (vis) {
        const unsigned int ci = vis_base + rank;
        float rgb[3];
        sh_to_rgb<DEG>(sc.sh + (size_t)g * sc.sh_stride, wx - p.centre[0], wy - p.centre[1], wz - p.centre[2], rgb);
        // DESIGN R25: factorised exponent from the ROUNDED conic, derived in fp64, rounded once
        const double LOG2E = 1.4426950408889634;
        double dA = (double)cA, dB = (double)cB, dC = (double)cC;
        float kk = (float)(dB / dA);
        float a2 = (float)(-0.5 * LOG2E * dA);                       // stored negated: e = log2 o + a2 w^2 + d2 dy^2
        float d2 = (float)(-0.5 * LOG2E * (dC - dB * dB / dA));
        ws.gA[ci] = make_float4(mx2, my2, kk, a2);
        ws.gB[ci] = make_float4(d2, __ldg(sc.l2o + g), rgb[0], rgb[1]);
        ws.cB[ci] = rgb[2];
        ws.cgid[ci] = (uint32_t)g;
        if (DEBUG) {
            flod_dbg_projected d;
            d.gid = (uint32_t)g; d.mu2d[0] = mx2; d.mu2d[1] = my2; d.depth = pz;
            d.conic[0] = cA; d.conic[1] = cB; d.conic[2] = cC; d.opacity = __ldg(sc.opacity + g);
            d.rgb[0] = rgb[0]; d.rgb[1] = rgb[1]; d.rgb[2] = rgb[2];
            d.rect[0] = tx0; d.rect[1] = ty0; d.rect[2] = tx1; d.rect[3] = ty1;
            ws.dbg[ci] = d;
        }
        s_incl[rank] = pair_incl;
        s_rect[rank] = (unsigned int)tx0 | ((unsigned int)ty0 << 16);
        s_wd[rank] = (unsigned int)(tx1 - tx0);
        s_depth[rank] = __float_as_uint(pz);
    }
    __syncthreads();

    // ---- a6: block-cooperative expansion, one pair per thread per step, coalesced stores
    unsigned long long *__restrict__ keys = ws.keys[0];
    uint32_t *__restrict__ vals = ws.vals[0];
    for (unsigned long long q = tid; q < block_pairs; q += kPreBlock) {
        const unsigned int qq = (unsigned int)q;
        int lo = 0, hi = (int)block_vis - 1;           // first rank with s_incl[rank] > qq
        while (lo < hi) {
            int mid = (lo + hi) >> 1;
            if (s_incl[mid] > qq) hi = mid; else lo = mid + 1;
        }
        const unsigned int r = (unsigned int)lo;
        const unsigned int start = r ? s_incl[r - 1] : 0u;
        const unsigned int k = qq - start;
        const unsigned int w = s_wd[r];
        const unsigned int ry = k / w, rx = k - ry * w;
        const unsigned int rc = s_rect[r];
        const unsigned int tile = ((rc >> 16) + ry) * (unsigned int)p.TX + ((rc & 0xffffu) + rx);
        const unsigned long long dst = pair_base + q;
        if (dst < p.max_pairs) {
            keys[dst] = ((unsigned long long)tile << 32) | s_depth[r];
            vals[dst] = vis_base + r;
        }
    }
}

template <int DEG>
static void launch_deg(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (c.flags & FLOD_OPT_DEBUG)
        k_preprocess<DEG, true><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.scene, c.ws, p);
    else
        k_preprocess<DEG, false><<<p.n_pre_blocks, kPreBlock, 0, s>>>(c.scene, c.ws, p);
}

int launch_preprocess(const Context &c, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    switch (c.sh_degree) {
        case 0: launch_deg<0>(c, p, s); break;
        case 1: launch_deg<1>(c, p, s); break;
        case 2: launch_deg<2>(c, p, s); break;
        default: launch_deg<3>(c, p, s); break;
    }
    return 1;
}

}  // namespace flod
