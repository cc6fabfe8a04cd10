// Steps a1-a4 of the hot path:
//   k_geometry  a1 level selection (Eq. 6-7), a2 cull + view transform, a3 EWA projection, conic,
//               tile rect.  Phase 1: a thread owns eight consecutive Gaussians (two 16-byte loads per mean
//               plane), selects, transforms, culls and applies a conservative off-screen test; the block lists the
//               survivors.  Phase 2: one survivor per thread, all lanes busy, runs the projection; a visible Gaussian
//               writes its records at the front of the block's segment of the per-frame arrays, in gid order (no
//               inter-block scan: see WorkspaceDev), and adds its rect to a 2-D difference grid of the tile counts
//               (four integer atomics whatever the rect size);
//   k_colour    a4 SH -> RGB, one block per segment; its block 0 runs the tile scan (a5 + a8, tile_scan.cuh).
//
// The geometry (a1-a3 and the rect) is the canonical fp32 sequence of DESIGN §2: each operation is one IEEE
// round-to-nearest binary32 operation (the *_rn intrinsics are never contracted into FMAs), in the written order.
#include "flod_internal.cuh"
#include "tile_scan.cuh"

// An SH row is read once per frame and never again: evict-first (ld.global.cs) loads keep the 300 MB of rows from
// pushing the frame's L2-resident workspace out (k_colour 63 -> 56 us on config 1).  The same on the planes k_geometry
// reads changed nothing.
#define FLOD_LD_STREAM(p) __ldcs(p)

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

// Shared memory of k_geometry.
struct GeoSmem {
    unsigned short cand[kGeoBlock];                   // candidate slot -> index of the Gaussian inside the block (gid order)
    unsigned int warp_cnt[kGeoThreads / 32];
    unsigned int warp_vis[2][kGeoThreads / 32];       // double-buffered over the steps of phase 2
    unsigned int cnt[2];                              // n_sel, n_front of the block
    unsigned long long pairs;
};

__device__ __forceinline__ void red_add_f32x4(float *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

template <bool DEBUG, bool ELLIPSE>
__global__ void __launch_bounds__(kGeoThreads, 10)     // 48 registers: ten blocks per SM
k_geometry(const SceneDev sc, const WorkspaceDev ws, const __grid_constant__ FrameParams p)
{
    __shared__ GeoSmem S;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) { S.cnt[0] = 0; S.cnt[1] = 0; S.pairs = 0; }
    cudaGridDependencySynchronize();                    // launched programmatically behind the previous frame's last kernel
    const int bid = blockIdx.x;
    const long long gb = p.quad_gid + (long long)bid * kGeoBlock;           // first gid of the block (multiple of 4)
    const long long g0 = gb + tid * kGeoPer;
    const long long g_end = p.first_gid + p.n_scan;
    const float *R = p.R;

    // ================= phase 1: a thread owns kGeoPer = 8 consecutive Gaussians (two 16-byte loads per mean / rho2 plane)
    // a1 level selection, a2 view transform and z cull (canonical fp32), then a conservative off-screen test that
    // needs no covariance.  What survives is a CANDIDATE; the candidates of the block are listed in gid order.
    unsigned int m_sel = 0, m_front = 0, m_cand = 0;
    {
        // kGeoPer / 4 quads per thread, every load issued before the first use (bytes in flight are what a streaming
        // kernel of short blocks lives on)
        constexpr int NQ = kGeoPer / 4;
        float wx[kGeoPer], wy[kGeoPer], wz[kGeoPer], rho2[kGeoPer];
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const long long gq = g0 + 4 * q;
            float4 X = make_float4(0.f, 0.f, 0.f, 0.f), Y = X, Z = X, Q = X;
            if (gq < g_end && gq + 4 > p.first_gid) {
                X = __ldg(reinterpret_cast<const float4 *>(sc.mx + gq));
                Y = __ldg(reinterpret_cast<const float4 *>(sc.my + gq));
                Z = __ldg(reinterpret_cast<const float4 *>(sc.mz + gq));
                Q = __ldg(reinterpret_cast<const float4 *>(sc.rho2 + gq));
            }
            wx[4 * q] = X.x; wx[4 * q + 1] = X.y; wx[4 * q + 2] = X.z; wx[4 * q + 3] = X.w;
            wy[4 * q] = Y.x; wy[4 * q + 1] = Y.y; wy[4 * q + 2] = Y.z; wy[4 * q + 3] = Y.w;
            wz[4 * q] = Z.x; wz[4 * q + 1] = Z.y; wz[4 * q + 2] = Z.z; wz[4 * q + 3] = Z.w;
            rho2[4 * q] = Q.x; rho2[4 * q + 1] = Q.y; rho2[4 * q + 2] = Q.z; rho2[4 * q + 3] = Q.w;
        }
#pragma unroll
        for (int k = 0; k < kGeoPer; ++k) {
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
            if (DEBUG) ws.mask[sc.src_gid ? (long long)__ldg(sc.src_gid + g) : g] = sel ? 1 : 0;   // (a snapshot holds selected ones only)
            if (!sel) continue;
            m_sel |= 1u << k;
            // ---- a2 (O2): p = R mu + t
            const float px = fadd(fadd(fadd(fmul(R[0], wx[k]), fmul(R[1], wy[k])), fmul(R[2], wz[k])), p.t[0]);
            const float py = fadd(fadd(fadd(fmul(R[3], wx[k]), fmul(R[4], wy[k])), fmul(R[5], wz[k])), p.t[1]);
            const float pz = fadd(fadd(fadd(fmul(R[6], wx[k]), fmul(R[7], wy[k])), fmul(R[8], wz[k])), p.t[2]);
            if (!(pz > p.z_near)) continue;
            m_front |= 1u << k;
            if (!(rho2[k] >= 0.0f)) continue;                  // rho2 = -1 marks a dead Gaussian (o < 1/255)
            // ---- conservative off-screen test.  O4's half extents obey h <= sqrt(kappa (lambda_max |J row|^2 + 0.3))
            // (1 + 2^-10) + 2^-6 with |J row|^2 <= pre_c1 / z^2 and kappa <= 2 ln 255, so with the margins below
            // (1 % and one pixel, far above the rounding of this approximate arithmetic) a Gaussian dropped here
            // would have got an empty tile rect from the exact sequence of phase 2.
            const float rz = __frcp_rn(pz);
            const float ax = fmaf(p.fx * px, rz, p.cx), ay = fmaf(p.fy * py, rz, p.cy);
            const float bnd = sqrtf(fmaf(rho2[k] * p.pre_c1, rz * rz, 3.33f)) * 1.01f + 1.0f + 1e-5f * (fabsf(ax) + fabsf(ay));
            const bool off = ax + bnd < 0.0f || ax - bnd > (float)(p.TX * kTile) ||
                             ay + bnd < (float)(p.ty_begin * kTile) || ay - bnd > (float)(p.ty_end * kTile);
            if (!off) m_cand |= 1u << k;                       // (a NaN or infinite bound keeps the Gaussian)
        }
    }
    // block scan of the candidate counts (gid order = thread order, then k); block totals of the statistics
    const unsigned int nc = __popc(m_cand);
    unsigned int incl = nc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    unsigned int ws_sel = __popc(m_sel), ws_front = __popc(m_front);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ws_sel += __shfl_xor_sync(0xffffffffu, ws_sel, o);
        ws_front += __shfl_xor_sync(0xffffffffu, ws_front, o);
    }
    if (lane == 31) S.warp_cnt[warp] = incl;
    __syncthreads();                                     // S.cnt / S.pairs were zeroed by thread 0
    if (lane == 0) {
        if (ws_sel) atomicAdd(&S.cnt[0], ws_sel);
        if (ws_front) atomicAdd(&S.cnt[1], ws_front);
    }
    unsigned int local = incl - nc, n_cand = 0;
#pragma unroll
    for (int w = 0; w < kGeoThreads / 32; ++w) {
        const unsigned int t = S.warp_cnt[w];
        if (w < warp) local += t;
        n_cand += t;
    }
#pragma unroll
    for (int k = 0; k < kGeoPer; ++k)
        if ((m_cand >> k) & 1u) S.cand[local++] = (unsigned short)(tid * kGeoPer + k);
    __syncthreads();

    // ================= phase 2: one candidate per thread and step, all lanes busy.  a3 EWA projection, conic, tile
    // rect: the canonical fp32 sequence of DESIGN §2 (p is recomputed from the mean by the same operations as in
    // phase 1, so it has the same bits).  A visible Gaussian writes its records straight to the block's segment, at
    // the position a ballot scan gives it: gid order is kept because the candidate list is in gid order.
    const unsigned int seg_base = (unsigned int)bid * kGeoBlock;
    unsigned int n_vis_before = 0, my_pairs = 0;
    for (unsigned int s0 = 0, step = 0; s0 < n_cand; s0 += kGeoThreads, ++step) {
        const unsigned int s = s0 + tid;
        bool vis = false;
        float mx2 = 0.f, my2 = 0.f, z = 0.f, cA = 0.f, cB = 0.f, cC = 0.f, l2o = 0.f, wxk = 0.f, wyk = 0.f, wzk = 0.f, kap = 0.f;
        int tx0 = 0, tx1 = 0, ty0 = 0, ty1 = 0, rty0 = 0, rty1 = 0;
        long long g = 0;
        if (s < n_cand) {
            g = gb + S.cand[s];
            wxk = __ldg(sc.mx + g); wyk = __ldg(sc.my + g); wzk = __ldg(sc.mz + g);
            const float4 r0 = __ldg(sc.rec + 2 * g), r1 = __ldg(sc.rec + 2 * g + 1);      // one 32-byte sector
            const float Sxx = r0.x, Sxy = r0.y, Sxz = r0.z, Syy = r0.w, Syz = r1.x, Szz = r1.y;
            kap = r1.z; l2o = r1.w;
            const float px = fadd(fadd(fadd(fmul(R[0], wxk), fmul(R[1], wyk)), fmul(R[2], wzk)), p.t[0]);
            const float py = fadd(fadd(fadd(fmul(R[3], wxk), fmul(R[4], wyk)), fmul(R[5], wzk)), p.t[1]);
            z = fadd(fadd(fadd(fmul(R[6], wxk), fmul(R[7], wyk)), fmul(R[8], wzk)), p.t[2]);
            const float ix = fdiv(px, z), iy = fdiv(py, z);
            mx2 = fadd(fmul(p.fx, ix), p.cx);
            my2 = fadd(fmul(p.fy, iy), p.cy);
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
            if (det > 0.0f) {
                cA = fdiv(c, det); cB = -fdiv(b, det); cC = fdiv(a, det);
                // ---- O4: padded box of the alpha = 1/255 contour, in 16x16 tiles
                const float hx = fadd(fmul(__fsqrt_rn(fmul(kap, a)), 1.0009765625f), 0.015625f);
                const float hy = fadd(fmul(__fsqrt_rn(fmul(kap, c)), 1.0009765625f), 0.015625f);
                const float fTX = (float)p.TX, fTY = (float)p.TY;
                const float x0 = fminf(fmaxf(floorf(fmul(fsub(mx2, hx), 0.0625f)), 0.0f), fTX);
                const float x1 = fminf(fmaxf(fadd(floorf(fmul(fadd(mx2, hx), 0.0625f)), 1.0f), 0.0f), fTX);
                const float y0 = fminf(fmaxf(floorf(fmul(fsub(my2, hy), 0.0625f)), 0.0f), fTY);
                const float y1 = fminf(fmaxf(fadd(floorf(fmul(fadd(my2, hy), 0.0625f)), 1.0f), 0.0f), fTY);
                tx0 = (int)x0; tx1 = (int)x1; ty0 = (int)y0; ty1 = (int)y1;
                rty0 = ty0; rty1 = ty1;                    // the canonical rect (debug record)
                ty0 = max(ty0, p.ty_begin); ty1 = min(ty1, p.ty_end);      // ... clipped to the frame's strip of tile rows
                vis = (tx1 - tx0) > 0 && (ty1 - ty0) > 0;
            }
        }
        // ---- position of the visible ones: ballot inside the warp, warp totals through shared memory
        const unsigned int bal = __ballot_sync(0xffffffffu, vis);
        if (lane == 0) S.warp_vis[step & 1][warp] = __popc(bal);
        __syncthreads();
        unsigned int pos = n_vis_before + __popc(bal & ((1u << lane) - 1)), step_total = 0;
#pragma unroll
        for (int w = 0; w < kGeoThreads / 32; ++w) {
            const unsigned int t = S.warp_vis[step & 1][w];
            if (w < warp) pos += t;
            step_total += t;
        }
        n_vis_before += step_total;
        if (vis) {
            // DESIGN R25: factorised exponent from the ROUNDED conic, derived in fp64, rounded once.  Canonical (every
            // operation one IEEE binary64 operation, written order): pair rule 2 (R26, span.cuh) takes the contour from
            // these values, and the oracle restates the derivation.
            const double HL2E = -0.5 * 1.4426950408889634;
            const double dA = (double)cA, dB = (double)cB, dC = (double)cC;
            const double rA = __ddiv_rn(1.0, dA);
            const float kk = (float)__dmul_rn(dB, rA);
            const float a2 = (float)__dmul_rn(HL2E, dA);                 // stored negated: e = log2 o + a2 w^2 + d2 dy^2
            // <= 0 so that q >= 0 holds by construction in k_blend (the oracle clamps q at 0; a conic left indefinite by
            // rounding differs from its clamp by less than R25's evaluation error)
            const float d2 = fminf((float)__dmul_rn(HL2E, __dsub_rn(dC, __dmul_rn(__dmul_rn(dB, dB), rA))), 0.0f);
            const size_t c = (size_t)seg_base + pos;
            ws.gA[c] = make_float4(mx2, my2, kk, a2);
            reinterpret_cast<float2 *>(ws.gB)[2 * c] = make_float2(d2, l2o);          // (r, g) by k_colour
            ws.rect[c] = make_ushort4((unsigned short)tx0, (unsigned short)ty0, (unsigned short)tx1, (unsigned short)ty1);
            ws.depth[c] = __float_as_uint(z);
            const unsigned int g_scene = sc.src_gid ? __ldg(sc.src_gid + g) : (unsigned int)g;     // the SH row's gid
            ws.dirgid[c] = make_float4(wxk - p.centre[0], wyk - p.centre[1], wzk - p.centre[2], __uint_as_float(g_scene));
            if (DEBUG) {
                flod_dbg_projected d;
                d.gid = g_scene; d.mu2d[0] = mx2; d.mu2d[1] = my2; d.depth = z;
                d.conic[0] = cA; d.conic[1] = cB; d.conic[2] = cC; d.opacity = __ldg(sc.opacity + g);
                d.rgb[0] = 0.0f; d.rgb[1] = 0.0f; d.rgb[2] = 0.0f;                                // by k_colour
                d.rect[0] = tx0; d.rect[1] = rty0; d.rect[2] = tx1; d.rect[3] = rty1;
                ws.dbg[c] = d;
            }
            // a5, first half: the difference grid of the per-tile pair counts
            const int gw = p.TX + 1;
            if (!ELLIPSE) {
                my_pairs += (unsigned int)((tx1 - tx0) * (ty1 - ty0));
                // The reductions below go to scattered addresses in L2 and cost the kernel a fifth of its time (measured
                // without them: 60 -> 48 us on config 1), so a rect issues as few as it can.  The usual rect lies in at
                // most 2x2 GROUPS of 2x2 tiles (config 1: 2.05 groups per rect): one float4 reduction per group adds 1 to
                // each of the group's tiles the rect covers (exact below 2^24 per tile, the limit k_duplicate's float
                // append counters have anyway).  A larger rect adds +1 -1 -1 +1 at its corners in the 2-D difference
                // grid: four reductions whatever its area.  The tile scan sums the two.
                const int gx0 = tx0 >> 1, gx1 = (tx1 + 1) >> 1, gy0 = ty0 >> 1, gy1 = (ty1 + 1) >> 1;
                if (gx1 - gx0 <= 2 && gy1 - gy0 <= 2) {
                    // straight-line over the (up to) four groups: which of a group's two tile columns / rows the rect covers
                    const int GX = (p.TX + 1) >> 1;
                    const float xa0 = 2 * gx0 >= tx0 ? 1.0f : 0.0f, xa1 = 2 * gx0 + 1 < tx1 ? 1.0f : 0.0f;      // first group column
                    const float xb1 = 2 * gx0 + 3 < tx1 ? 1.0f : 0.0f;                                          // second (its first tile is covered)
                    const float ya0 = 2 * gy0 >= ty0 ? 1.0f : 0.0f, ya1 = 2 * gy0 + 1 < ty1 ? 1.0f : 0.0f;
                    const float yb1 = 2 * gy0 + 3 < ty1 ? 1.0f : 0.0f;
                    const bool two_x = gx1 - gx0 == 2, two_y = gy1 - gy0 == 2;
                    float *g00 = ws.cnt4 + (size_t)(gy0 * GX + gx0) * kCtrStride;
                    red_add_f32x4(g00, xa0 * ya0, xa1 * ya0, xa0 * ya1, xa1 * ya1);
                    if (two_x) red_add_f32x4(g00 + kCtrStride, ya0, xb1 * ya0, ya1, xb1 * ya1);
                    if (two_y) red_add_f32x4(g00 + (size_t)GX * kCtrStride, xa0, xa1, xa0 * yb1, xa1 * yb1);
                    if (two_x && two_y) red_add_f32x4(g00 + (size_t)(GX + 1) * kCtrStride, 1.0f, xb1, yb1, xb1 * yb1);
                } else {
                    atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx0) * kCtrStride, 1);
                    atomicAdd(ws.tile_diff + (size_t)(ty0 * gw + tx1) * kCtrStride, -1);
                    atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx0) * kCtrStride, -1);
                    atomicAdd(ws.tile_diff + (size_t)(ty1 * gw + tx1) * kCtrStride, 1);
                }
            }
            // (R26, pair rule 2: phase 3 counts the listed tiles)
        }
    }
    // ================= phase 3 (pair rule 2, DESIGN R26): one VISIBLE Gaussian per thread -- the block's visible ones sit
    // densely at the front of its segment, so all lanes are busy here, unlike in phase 2 where the lanes of culled
    // candidates idle.  The span of listed tiles of every tile row of the rect (span.cuh: canonical fp32 from the blend
    // features just written) is counted with +1 / -1 at its ends in a row-wise difference grid.
    if (ELLIPSE) {
        __syncthreads();                                   // the records of phase 2 are visible to the whole block
        const int gw = p.TX + 1;
        for (unsigned int j = tid; j < n_vis_before; j += kGeoThreads) {
            const size_t c = (size_t)seg_base + j;
            const float4 fa = ws.gA[c];
            const float2 fb = *reinterpret_cast<const float2 *>(ws.gB + c);
            const ushort4 rc = ws.rect[c];
            const SpanCoef sp = span_coefficients(fa.x, fa.y, fa.z, fa.w, fb.x, fb.y);
            for (int ty = rc.y; ty < (int)rc.w; ++ty) {
                int ta, tb;
                const int n = span_of_row(sp, (int)rc.x, (int)rc.z, ty, &ta, &tb);
                if (n == 0) continue;
                my_pairs += (unsigned int)n;
                atomicAdd(ws.tile_diff + (size_t)(ty * gw + ta) * kCtrStride, 1);
                atomicAdd(ws.tile_diff + (size_t)(ty * gw + tb + 1) * kCtrStride, -1);
            }
        }
    }
    // ---- block totals
    unsigned int ws_pairs = my_pairs;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ws_pairs += __shfl_xor_sync(0xffffffffu, ws_pairs, o);
    if (lane == 0 && ws_pairs) atomicAdd(&S.pairs, (unsigned long long)ws_pairs);
    __syncthreads();
    if (tid == 0) {
        ws.seg_count[bid] = n_vis_before;
        if (n_vis_before) atomicAdd(&ws.hdr->n_vis32, n_vis_before);
        if (S.cnt[0]) atomicAdd(&ws.hdr->n_sel, (unsigned long long)S.cnt[0]);
        if (S.cnt[1]) atomicAdd(&ws.hdr->n_front, (unsigned long long)S.cnt[1]);
        if (S.pairs) atomicAdd(&ws.hdr->n_pairs, S.pairs);
    }
}

// ---- a4: colour of every visible Gaussian.  rgb = max(0, 0.5 + sum_k Y_k(dir) sh_k)  (R16)
// LANES threads share one Gaussian.  LANES = 4 needs the degree-3 row layout written by the upload: the row is 12
// float4; float4 number (4 i + j), i = 0..2, holds floats [4 i, 4 i + 4) of the 12 floats (k, channel) of the
// coefficients k = 4 j .. 4 j + 3, so one load instruction of the 4 lanes reads 64 contiguous bytes.
template <int DEG, int LANES, bool DEBUG>
__global__ void __launch_bounds__(256)
k_colour(const SceneDev sc, const WorkspaceDev ws, int TX, int TY, unsigned int max_pairs, int pair_rule)
{
    constexpr int K = (DEG + 1) * (DEG + 1);
    cudaGridDependencySynchronize();
    if (blockIdx.x == 0) { tile_scan_block(ws, TX, TY, max_pairs, pair_rule != FLOD_PAIR_RULE_BOX); return; }
    const unsigned int sub = threadIdx.x % LANES;
    const unsigned int per_block = 256 / LANES;
    const unsigned int seg = blockIdx.x - 1;             // one block per segment of k_geometry
    const unsigned int n_here = ws.seg_count[seg];
    // U Gaussians per lane group and step: the U direction records are loaded first, then the U SH rows, then the
    // arithmetic.  (U = 2 -- two dependent round trips per step instead of per Gaussian -- was worth 2 us in round 1;
    // with evict-first rows and programmatic launch U = 1 measures 59.5 against 61.0 us on config 1, 97 against 102 on
    // config 4 at 1920x1080, 48.4 against 47.4 on config 3 level 5)
    constexpr int U = 1;
    for (unsigned int j0 = 0; j0 < n_here; j0 += U * per_block) {
        bool ok[U];
        unsigned int ci[U];
        float4 dg[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const unsigned int j = j0 + u * per_block + threadIdx.x / LANES;
            ok[u] = j < n_here;
            ci[u] = seg * kGeoBlock + j;
            dg[u] = ok[u] ? ws.dirgid[ci[u]] : make_float4(0.f, 0.f, 1.f, 0.f);
        }
        float r[U], g[U], b[U];
        if constexpr (LANES == 4) {
            static_assert(DEG == 3 || LANES == 1, "4-lane layout is degree 3 only");
            float4 f0[U], f1[U], f2[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                f0[u] = f1[u] = f2[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (ok[u]) {
                    const float4 *r4 = reinterpret_cast<const float4 *>(sc.sh + (size_t)__float_as_uint(dg[u].w) * sc.sh_stride);
                    f0[u] = FLOD_LD_STREAM(r4 + sub); f1[u] = FLOD_LD_STREAM(r4 + 4 + sub); f2[u] = FLOD_LD_STREAM(r4 + 8 + sub);
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                float Y[K];
                const float inv = 1.0f / sqrtf(dg[u].x * dg[u].x + dg[u].y * dg[u].y + dg[u].z * dg[u].z);
                sh_basis<DEG>(dg[u].x * inv, dg[u].y * inv, dg[u].z * inv, Y);
                const float y0 = sub == 0 ? Y[0] : sub == 1 ? Y[4] : sub == 2 ? Y[8] : Y[12];
                const float y1 = sub == 0 ? Y[1] : sub == 1 ? Y[5] : sub == 2 ? Y[9] : Y[13];
                const float y2 = sub == 0 ? Y[2] : sub == 1 ? Y[6] : sub == 2 ? Y[10] : Y[14];
                const float y3 = sub == 0 ? Y[3] : sub == 1 ? Y[7] : sub == 2 ? Y[11] : Y[15];
                r[u] = fmaf(y0, f0[u].x, fmaf(y1, f0[u].w, fmaf(y2, f1[u].z, y3 * f2[u].y)));
                g[u] = fmaf(y0, f0[u].y, fmaf(y1, f1[u].x, fmaf(y2, f1[u].w, y3 * f2[u].z)));
                b[u] = fmaf(y0, f0[u].z, fmaf(y1, f1[u].y, fmaf(y2, f2[u].x, y3 * f2[u].w)));
#pragma unroll
                for (int o = 1; o < 4; o <<= 1) {
                    r[u] += __shfl_xor_sync(0xffffffffu, r[u], o);
                    g[u] += __shfl_xor_sync(0xffffffffu, g[u], o);
                    b[u] += __shfl_xor_sync(0xffffffffu, b[u], o);
                }
            }
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                r[u] = g[u] = b[u] = 0.0f;
                if (!ok[u]) continue;
                constexpr int NF = (3 * K + 3) / 4 * 4;
                float f[NF], Y[K];
                const float4 *r4 = reinterpret_cast<const float4 *>(sc.sh + (size_t)__float_as_uint(dg[u].w) * sc.sh_stride);
#pragma unroll
                for (int q = 0; q < NF / 4; ++q) {
                    const float4 t = FLOD_LD_STREAM(r4 + q);
                    f[4 * q] = t.x; f[4 * q + 1] = t.y; f[4 * q + 2] = t.z; f[4 * q + 3] = t.w;
                }
                const float inv = DEG >= 1 ? 1.0f / sqrtf(dg[u].x * dg[u].x + dg[u].y * dg[u].y + dg[u].z * dg[u].z) : 0.0f;
                sh_basis<DEG>(dg[u].x * inv, dg[u].y * inv, dg[u].z * inv, Y);
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    r[u] = fmaf(Y[k], f[3 * k], r[u]);
                    g[u] = fmaf(Y[k], f[3 * k + 1], g[u]);
                    b[u] = fmaf(Y[k], f[3 * k + 2], b[u]);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (ok[u] && sub == 0) {
                const float rr = fmaxf(r[u] + 0.5f, 0.0f), gg = fmaxf(g[u] + 0.5f, 0.0f), bb = fmaxf(b[u] + 0.5f, 0.0f);
                reinterpret_cast<float2 *>(ws.gB)[2 * (size_t)ci[u] + 1] = make_float2(rr, gg);
                ws.cB[ci[u]] = bb;
                if (DEBUG) { ws.dbg[ci[u]].rgb[0] = rr; ws.dbg[ci[u]].rgb[1] = gg; ws.dbg[ci[u]].rgb[2] = bb; }
            }
        }
    }
}

int launch_geometry(const Context &c, const SceneDev &sc, const FrameParams &p, cudaStream_t s)
{
    if (p.n_pre_blocks <= 0) return 0;
    const bool ell = p.pair_rule != FLOD_PAIR_RULE_BOX;
    if (c.flags & FLOD_OPT_DEBUG) {
        if (ell) launch_pdl(k_geometry<true, true>, p.n_pre_blocks, kGeoThreads, 0, s, sc, c.ws, p);
        else launch_pdl(k_geometry<true, false>, p.n_pre_blocks, kGeoThreads, 0, s, sc, c.ws, p);
    } else {
        if (ell) launch_pdl(k_geometry<false, true>, p.n_pre_blocks, kGeoThreads, 0, s, sc, c.ws, p);
        else launch_pdl(k_geometry<false, false>, p.n_pre_blocks, kGeoThreads, 0, s, sc, c.ws, p);
    }
    return 1;
}

template <int DEG, int LANES>
static void launch_colour_t(const Context &c, const FrameParams &p, int grid, cudaStream_t s)
{
    if (c.flags & FLOD_OPT_DEBUG) launch_pdl(k_colour<DEG, LANES, true>, grid, 256, 0, s, c.scene, c.ws, p.TX, p.TY, p.max_pairs, p.pair_rule);
    else launch_pdl(k_colour<DEG, LANES, false>, grid, 256, 0, s, c.scene, c.ws, p.TX, p.TY, p.max_pairs, p.pair_rule);
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
