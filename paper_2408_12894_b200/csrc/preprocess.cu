// Steps a1-a4 of the hot path:
//   k_geometry  a1 level selection (Eq. 6-7), a2 cull + view transform, a3 EWA projection, conic,
//               tile rect.  A thread owns four consecutive Gaussians (16-byte loads from every SoA plane, all
//               loads of a phase in flight together); the block stages the records of its visible Gaussians in shared
//               memory and copies them out, in gid order, dense and coalesced, at the front of its own segment of
//               the per-frame arrays (no inter-block scan: see WorkspaceDev).  Every visible Gaussian also adds its rect to a 2-D
//               difference grid of the tile counts (four integer atomics whatever the rect size);
//   k_colour    a4 SH -> RGB, one block per segment; its block 0 runs the tile scan (a5 + a8, tile_scan.cuh).
//
// The geometry (a1-a3 and the rect) is the canonical fp32 sequence of DESIGN §2: each operation is one IEEE
// round-to-nearest binary32 operation (the *_rn intrinsics are never contracted into FMAs), in the written order.
#include "flod_internal.cuh"
#include "tile_scan.cuh"

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

// Shared staging of one block's records, slot = k * kGeoThreads + tid for Gaussian k of thread tid (conflict-free).
template <bool DEBUG>
struct GeoSmem {
    float4 a[kGeoBlock];                              // mu'x, mu'y, k, a2
    float4 dg[kGeoBlock];                             // mu - c_cam, gid bits
    float2 b[kGeoBlock];                              // d2, log2 o
    uint2 rect[kGeoBlock];                            // tx0 | ty0 << 16, tx1 | ty1 << 16
    uint32_t depth[kGeoBlock];
    float4 conic_o[DEBUG ? kGeoBlock : 1];            // A, B, C, o (debug records only)
    unsigned short map[kGeoBlock];                    // block-local compact position -> slot
    unsigned int warp_vis[kGeoThreads / 32];
    unsigned int cnt[2];                              // n_sel, n_front of the block
    unsigned long long pairs;
};

template <bool DEBUG>
__global__ void __launch_bounds__(kGeoThreads, 3)
k_geometry(const SceneDev sc, const WorkspaceDev ws, const __grid_constant__ FrameParams p)
{
    extern __shared__ __align__(16) unsigned char geo_smem_raw[];
    GeoSmem<DEBUG> &S = *reinterpret_cast<GeoSmem<DEBUG> *>(geo_smem_raw);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { S.cnt[0] = 0; S.cnt[1] = 0; S.pairs = 0; }
    const int bid = blockIdx.x;
    const long long g0 = p.quad_gid + ((long long)bid * kGeoThreads + tid) * kGeoPer;   // multiple of 4
    const long long g_end = p.first_gid + p.n_scan;

    // ---- phase 1 loads: mean and kappa of the quad (16-byte loads; the planes are padded to 256 B)
    float wx[4], wy[4], wz[4], kap[4];
    const bool quad_live = g0 < g_end && g0 + kGeoPer > p.first_gid;
    if (quad_live) {
        const float4 X = __ldg(reinterpret_cast<const float4 *>(sc.mx + g0));
        const float4 Y = __ldg(reinterpret_cast<const float4 *>(sc.my + g0));
        const float4 Z = __ldg(reinterpret_cast<const float4 *>(sc.mz + g0));
        const float4 K = __ldg(reinterpret_cast<const float4 *>(sc.kappa + g0));
        wx[0] = X.x; wx[1] = X.y; wx[2] = X.z; wx[3] = X.w;
        wy[0] = Y.x; wy[1] = Y.y; wy[2] = Y.z; wy[3] = Y.w;
        wz[0] = Z.x; wz[1] = Z.y; wz[2] = Z.z; wz[3] = Z.w;
        kap[0] = K.x; kap[1] = K.y; kap[2] = K.z; kap[3] = K.w;
    }
    const float *R = p.R;
    unsigned int m_sel = 0, m_front = 0, m_proj = 0;       // bit k: Gaussian k selected / in front / to be projected
    float px[4], py[4], pz[4];
    if (quad_live) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long long g = g0 + k;
            if (g < p.first_gid || g >= g_end) continue;
            const int i = (int)(g - p.first_gid);
            int lv = 0;
#pragma unroll 1
            while (lv < p.n_levels - 1 && i >= p.level_end[lv]) ++lv;
            // ---- a1 (O1): Eq. 6 predicate on squared Euclidean distance to the reference
            const float dx = fsub(wx[k], p.ref[0]), dy = fsub(wy[k], p.ref[1]), dz = fsub(wz[k], p.ref[2]);
            const float d2 = fadd(fadd(fmul(dx, dx), fmul(dy, dy)), fmul(dz, dz));
            const bool sel = (d2 >= p.lo2[lv]) && (d2 < p.hi2[lv]);
            if (DEBUG) ws.mask[g] = sel ? 1 : 0;
            if (!sel) continue;
            m_sel |= 1u << k;
            // ---- a2 (O2): p = R mu + t
            px[k] = fadd(fadd(fadd(fmul(R[0], wx[k]), fmul(R[1], wy[k])), fmul(R[2], wz[k])), p.t[0]);
            py[k] = fadd(fadd(fadd(fmul(R[3], wx[k]), fmul(R[4], wy[k])), fmul(R[5], wz[k])), p.t[1]);
            pz[k] = fadd(fadd(fadd(fmul(R[6], wx[k]), fmul(R[7], wy[k])), fmul(R[8], wz[k])), p.t[2]);
            if (!(pz[k] > p.z_near)) continue;
            m_front |= 1u << k;
            if (kap[k] >= 0.0f) m_proj |= 1u << k;           // kappa = -1 marks a dead Gaussian (o < 1/255)
        }
    }

    // ---- phase 2 loads: the six covariance planes, only for quads with something to project
    float4 S0, S1, S2, S3, S4, S5;
    if (m_proj) {
        S0 = __ldg(reinterpret_cast<const float4 *>(sc.cov[0] + g0));
        S1 = __ldg(reinterpret_cast<const float4 *>(sc.cov[1] + g0));
        S2 = __ldg(reinterpret_cast<const float4 *>(sc.cov[2] + g0));
        S3 = __ldg(reinterpret_cast<const float4 *>(sc.cov[3] + g0));
        S4 = __ldg(reinterpret_cast<const float4 *>(sc.cov[4] + g0));
        S5 = __ldg(reinterpret_cast<const float4 *>(sc.cov[5] + g0));
    }
    float4 L2O = make_float4(0.f, 0.f, 0.f, 0.f), OP = L2O;
    if (m_proj) {
        L2O = __ldg(reinterpret_cast<const float4 *>(sc.l2o + g0));
        if (DEBUG) OP = __ldg(reinterpret_cast<const float4 *>(sc.opacity + g0));
    }

    unsigned int m_vis = 0, my_pairs = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (!((m_proj >> k) & 1u)) continue;
        const float Sxx = k == 0 ? S0.x : k == 1 ? S0.y : k == 2 ? S0.z : S0.w;
        const float Sxy = k == 0 ? S1.x : k == 1 ? S1.y : k == 2 ? S1.z : S1.w;
        const float Sxz = k == 0 ? S2.x : k == 1 ? S2.y : k == 2 ? S2.z : S2.w;
        const float Syy = k == 0 ? S3.x : k == 1 ? S3.y : k == 2 ? S3.z : S3.w;
        const float Syz = k == 0 ? S4.x : k == 1 ? S4.y : k == 2 ? S4.z : S4.w;
        const float Szz = k == 0 ? S5.x : k == 1 ? S5.y : k == 2 ? S5.z : S5.w;
        const float l2o = k == 0 ? L2O.x : k == 1 ? L2O.y : k == 2 ? L2O.z : L2O.w;
        const float z = pz[k];
        const float ix = fdiv(px[k], z), iy = fdiv(py[k], z);
        const float mx2 = fadd(fmul(p.fx, ix), p.cx);
        const float my2 = fadd(fmul(p.fy, iy), p.cy);
        // ---- a3 (O3): J at the clamped point, M = J R, Sigma' = M Sigma M^T + 0.3 I
        const float u = fminf(fmaxf(ix, -p.limx), p.limx);
        const float v = fminf(fmaxf(iy, -p.limy), p.limy);
        const float j00 = fdiv(p.fx, z);
        const float j02 = -fdiv(fmul(p.fx, u), z);
        const float j11 = fdiv(p.fy, z);
        const float j12 = -fdiv(fmul(p.fy, v), z);
        const float m00 = fadd(fmul(j00, R[0]), fmul(j02, R[6]));
        const float m01 = fadd(fmul(j00, R[1]), fmul(j02, R[7]));
        const float m02 = fadd(fmul(j00, R[2]), fmul(j02, R[8]));
        const float m10 = fadd(fmul(j11, R[3]), fmul(j12, R[6]));
        const float m11 = fadd(fmul(j11, R[4]), fmul(j12, R[7]));
        const float m12 = fadd(fmul(j11, R[5]), fmul(j12, R[8]));
        const float v0x = fadd(fadd(fmul(Sxx, m00), fmul(Sxy, m01)), fmul(Sxz, m02));
        const float v0y = fadd(fadd(fmul(Sxy, m00), fmul(Syy, m01)), fmul(Syz, m02));
        const float v0z = fadd(fadd(fmul(Sxz, m00), fmul(Syz, m01)), fmul(Szz, m02));
        const float v1x = fadd(fadd(fmul(Sxx, m10), fmul(Sxy, m11)), fmul(Sxz, m12));
        const float v1y = fadd(fadd(fmul(Sxy, m10), fmul(Syy, m11)), fmul(Syz, m12));
        const float v1z = fadd(fadd(fmul(Sxz, m10), fmul(Syz, m11)), fmul(Szz, m12));
        const float a = fadd(fadd(fadd(fmul(m00, v0x), fmul(m01, v0y)), fmul(m02, v0z)), 0.3f);
        const float b = fadd(fadd(fmul(m10, v0x), fmul(m11, v0y)), fmul(m12, v0z));
        const float c = fadd(fadd(fadd(fmul(m10, v1x), fmul(m11, v1y)), fmul(m12, v1z)), 0.3f);
        const float det = fsub(fmul(a, c), fmul(b, b));
        if (!(det > 0.0f)) continue;
        const float cA = fdiv(c, det), cB = -fdiv(b, det), cC = fdiv(a, det);
        // ---- O4: padded box of the alpha = 1/255 contour, in 16x16 tiles
        const float hx = fadd(fmul(__fsqrt_rn(fmul(kap[k], a)), 1.0009765625f), 0.015625f);
        const float hy = fadd(fmul(__fsqrt_rn(fmul(kap[k], c)), 1.0009765625f), 0.015625f);
        const float fTX = (float)p.TX, fTY = (float)p.TY;
        const float x0 = fminf(fmaxf(floorf(fmul(fsub(mx2, hx), 0.0625f)), 0.0f), fTX);
        const float x1 = fminf(fmaxf(fadd(floorf(fmul(fadd(mx2, hx), 0.0625f)), 1.0f), 0.0f), fTX);
        const float y0 = fminf(fmaxf(floorf(fmul(fsub(my2, hy), 0.0625f)), 0.0f), fTY);
        const float y1 = fminf(fmaxf(fadd(floorf(fmul(fadd(my2, hy), 0.0625f)), 1.0f), 0.0f), fTY);
        const int tx0 = (int)x0, tx1 = (int)x1, ty0 = (int)y0, ty1 = (int)y1;
        const unsigned int n_tiles = (unsigned int)((tx1 - tx0) * (ty1 - ty0));
        if (n_tiles == 0) continue;
        m_vis |= 1u << k;
        my_pairs += n_tiles;
        // DESIGN R25: factorised exponent from the ROUNDED conic, derived in fp64, rounded once
        const double LOG2E = 1.4426950408889634;
        const double dA = (double)cA, dB = (double)cB, dC = (double)cC;
        const float kk = (float)(dB / dA);
        const float a2 = (float)(-0.5 * LOG2E * dA);                   // stored negated: e = log2 o + a2 w^2 + d2 dy^2
        // <= 0 so that q >= 0 holds by construction in k_blend (the oracle clamps q at 0; a conic left indefinite by
        // rounding differs from its clamp by less than R25's evaluation error)
        const float d2 = fminf((float)(-0.5 * LOG2E * (dC - dB * dB / dA)), 0.0f);
        const int slot = k * kGeoThreads + tid;
        S.a[slot] = make_float4(mx2, my2, kk, a2);
        S.b[slot] = make_float2(d2, l2o);
        S.rect[slot] = make_uint2((unsigned int)tx0 | ((unsigned int)ty0 << 16), (unsigned int)tx1 | ((unsigned int)ty1 << 16));
        S.depth[slot] = __float_as_uint(z);
        S.dg[slot] = make_float4(wx[k] - p.centre[0], wy[k] - p.centre[1], wz[k] - p.centre[2],
                                 __uint_as_float((unsigned int)(g0 + k)));
        if (DEBUG) S.conic_o[slot] = make_float4(cA, cB, cC, k == 0 ? OP.x : k == 1 ? OP.y : k == 2 ? OP.z : OP.w);
        // a5, first half: +1 over the rect in the 2-D difference grid of the per-tile pair counts
#ifndef FLOD_X_NO_GEO_ATOMICS
        const int gw = p.TX + 1;
        atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx0) * kCtrStride, 1);
        atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx1) * kCtrStride, -1);
        atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx0) * kCtrStride, -1);
        atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx1) * kCtrStride, 1);
#endif
    }

    // ---- block scan of the visible counts (gid order = thread order, then k), block totals of the statistics
    const unsigned int nv = __popc(m_vis);
    unsigned int incl = nv;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    unsigned int ws_sel = __popc(m_sel), ws_front = __popc(m_front), ws_pairs = my_pairs;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ws_sel += __shfl_xor_sync(0xffffffffu, ws_sel, o);
        ws_front += __shfl_xor_sync(0xffffffffu, ws_front, o);
        ws_pairs += __shfl_xor_sync(0xffffffffu, ws_pairs, o);
    }
    if (lane == 31) S.warp_vis[warp] = incl;
    __syncthreads();                                     // S.cnt / S.pairs were zeroed by thread 0
    if (lane == 0) {
        if (ws_sel) atomicAdd(&S.cnt[0], ws_sel);
        if (ws_front) atomicAdd(&S.cnt[1], ws_front);
        if (ws_pairs) atomicAdd(&S.pairs, (unsigned long long)ws_pairs);
    }
    __syncthreads();
    unsigned int local = incl - nv;                      // block-local compact position of the thread's first visible
#pragma unroll
    for (int w = 0; w < kGeoThreads / 32; ++w) if (w < warp) local += S.warp_vis[w];
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if ((m_vis >> k) & 1u) S.map[local++] = (unsigned short)(k * kGeoThreads + tid);
    unsigned int total = 0;
#pragma unroll
    for (int w = 0; w < kGeoThreads / 32; ++w) total += S.warp_vis[w];
    __syncthreads();
    if (tid == 0) {
        ws.seg_count[bid] = total;
        if (total) atomicAdd(&ws.hdr->n_vis32, total);
        if (S.cnt[0]) atomicAdd(&ws.hdr->n_sel, (unsigned long long)S.cnt[0]);
        if (S.cnt[1]) atomicAdd(&ws.hdr->n_front, (unsigned long long)S.cnt[1]);
        if (S.pairs) atomicAdd(&ws.hdr->n_pairs, S.pairs);
    }

    // ---- copy-out: the block's visible records, dense and coalesced, at the front of the block's segment
    const unsigned int base = (unsigned int)bid * kGeoBlock;
    for (unsigned int j = tid; j < total; j += kGeoThreads) {
        const int slot = S.map[j];
        const size_t c = (size_t)base + j;
        ws.gA[c] = S.a[slot];
        reinterpret_cast<float2 *>(ws.gB)[2 * c] = S.b[slot];          // (r, g) by k_colour
        const uint2 rc = S.rect[slot];
        ws.rect[c] = make_ushort4((unsigned short)(rc.x & 0xffffu), (unsigned short)(rc.x >> 16),
                                  (unsigned short)(rc.y & 0xffffu), (unsigned short)(rc.y >> 16));
        ws.depth[c] = S.depth[slot];
        ws.dirgid[c] = S.dg[slot];
        if (DEBUG) {
            const float4 a = S.a[slot], co = S.conic_o[slot];
            flod_dbg_projected d;
            d.gid = __float_as_uint(S.dg[slot].w); d.mu2d[0] = a.x; d.mu2d[1] = a.y; d.depth = __uint_as_float(S.depth[slot]);
            d.conic[0] = co.x; d.conic[1] = co.y; d.conic[2] = co.z; d.opacity = co.w;
            d.rgb[0] = 0.0f; d.rgb[1] = 0.0f; d.rgb[2] = 0.0f;                                // by k_colour
            d.rect[0] = (int)(rc.x & 0xffffu); d.rect[1] = (int)(rc.x >> 16);
            d.rect[2] = (int)(rc.y & 0xffffu); d.rect[3] = (int)(rc.y >> 16);
            ws.dbg[c] = d;
        }
    }
}

// ---- a4: colour of every visible Gaussian.  rgb = max(0, 0.5 + sum_k Y_k(dir) sh_k)  (R16)
// LANES threads share one Gaussian.  LANES = 4 needs the degree-3 row layout written by the upload: the row is 12
// float4; float4 number (4 i + j), i = 0..2, holds floats [4 i, 4 i + 4) of the 12 floats (k, channel) of the
// coefficients k = 4 j .. 4 j + 3, so one load instruction of the 4 lanes reads 64 contiguous bytes.
template <int DEG, int LANES, bool DEBUG>
__global__ void __launch_bounds__(256)
k_colour(const SceneDev sc, const WorkspaceDev ws, int TX, int TY, unsigned int max_pairs)
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    if (blockIdx.x == 0) { tile_scan_block(ws, TX, TY, max_pairs); return; }
    const unsigned int sub = threadIdx.x % LANES;
    const unsigned int per_block = 256 / LANES;
    const unsigned int seg = blockIdx.x - 1;             // one block per segment of k_geometry
    const unsigned int n_here = ws.seg_count[seg];
    for (unsigned int j0 = 0; j0 < n_here; j0 += per_block) {
        const unsigned int j = j0 + threadIdx.x / LANES;
        const bool ok = j < n_here;
        const unsigned int slot = seg * kGeoBlock + j;
        float r = 0.0f, g = 0.0f, b = 0.0f;
        unsigned int ci = 0;
        if (ok) {
            ci = slot;
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
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(k_geometry<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GeoSmem<true>));
        cudaFuncSetAttribute(k_geometry<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(GeoSmem<false>));
        attr_set = true;
    }
    if (c.flags & FLOD_OPT_DEBUG) k_geometry<true><<<p.n_pre_blocks, kGeoThreads, sizeof(GeoSmem<true>), s>>>(c.scene, c.ws, p);
    else k_geometry<false><<<p.n_pre_blocks, kGeoThreads, sizeof(GeoSmem<false>), s>>>(c.scene, c.ws, p);
    return 1;
}

template <int DEG, int LANES>
static void launch_colour_t(const Context &c, const FrameParams &p, int grid, cudaStream_t s)
{
    if (c.flags & FLOD_OPT_DEBUG) k_colour<DEG, LANES, true><<<grid, 256, 0, s>>>(c.scene, c.ws, p.TX, p.TY, p.max_pairs);
    else k_colour<DEG, LANES, false><<<grid, 256, 0, s>>>(c.scene, c.ws, p.TX, p.TY, p.max_pairs);
}

int launch_colour(const Context &c, const FrameParams &p, cudaStream_t s)
{
    const int grid = max(p.n_pre_blocks, 0) + 1;        // block 0 = tile scan: runs even when nothing is scanned
    switch (c.sh_degree) {
        case 0: launch_colour_t<0, 1>(c, p, grid, s); break;
        case 1: launch_colour_t<1, 1>(c, p, grid, s); break;
        case 2: launch_colour_t<2, 1>(c, p, grid, s); break;
        default: launch_colour_t<3, 4>(c, p, grid, s); break;
    }
    return 1;
}

}  // namespace flod
