// Backward pass of the rasterizer (Alg. 1 P:581-583 "Rasterize ... Loss ... Adam(grad L)"):
// the gradient of <dL/dI, I> with respect to mean, log-scale, quaternion, opacity logit and SH coefficients of every
// Gaussian the LAST forward frame drew.  Two kernels over that frame's workspace (lists, ranges, blend features):
//   k_blend_backward  a9 backwards.  One CTA per tile, one pixel per thread.  Pass 1 walks the tile's list front to back
//                     with the forward rules (skip below 1/255, stop after T < 1e-4) to get every pixel's final T and the
//                     number of entries it processed; pass 2 walks it back to front, undoing T <- T (1 - alpha) and
//                     accumulating, per list entry, dL/d(mu'x, mu'y, A, B, C, o, r, g, b): reduced over the warp by
//                     shuffles, over the CTA in shared memory, one atomicAdd per value, entry and tile into g9.
//   k_project_backward  a2-a4 backwards.  One thread per visible Gaussian: recomputes the projection from the scene planes
//                     and chains g9 through the conic, Sigma' = M Sigma M^T + 0.3 I, the Jacobian (R8's clamp has zero
//                     slope outside), mu' = pinhole(p), Sigma = R S^2 R^T (Eq. 1), the sigmoid and the SH evaluation
//                     (R16); writes the per-gid gradient arrays (no atomics: one thread per Gaussian).
// The discrete decisions of the forward pass are constants; min(0.99, .) and max(0, .) have their mathematical slope.
// Plain fp32 (the forward's factorised exponent, R25, is the same function: the conic is recovered from its features).
#include "flod_internal.cuh"

namespace flod {

constexpr int kBwdThreads = 256;
constexpr int kBwdBatch = 64;                      // list entries reduced through shared memory at a time
constexpr float kLn2x2 = 1.3862943611198906f;      // 2 ln 2: a2 = -A log2(e) / 2  <=>  A = -a2 * 2 ln 2

struct BwdEntry { float mx, my, A, B, C, o, r, g, b; };

__device__ __forceinline__ BwdEntry bwd_entry(const WorkspaceDev &ws, unsigned int p)
{
    const float4 fa = ws.gA[p], fb = ws.gB[p];
    BwdEntry e;
    e.mx = fa.x; e.my = fa.y;
    e.A = -fa.w * kLn2x2;                          // gA = (mu'x, mu'y, k = B/A, a2), gB = (d2 = -(C - B^2/A) log2(e)/2, log2 o, r, g)
    e.B = fa.z * e.A;
    e.C = -fb.x * kLn2x2 + fa.z * e.B;
    e.o = exp2f(fb.y);
    e.r = fb.z; e.g = fb.w; e.b = ws.cB[p];
    return e;
}

// alpha of an entry at a pixel, with the forward's rules; G and the clamp flags for the backward chain
__device__ __forceinline__ float bwd_alpha(const BwdEntry &e, float px, float py, float *G_out, bool *free_out, float *dx_out, float *dy_out)
{
    const float dx = e.mx - px, dy = e.my - py;
    const float q = 0.5f * (e.A * dx * dx + e.C * dy * dy) + e.B * dx * dy;
    const float G = __expf(-fmaxf(q, 0.0f));
    const float raw = e.o * G;
    *G_out = G; *dx_out = dx; *dy_out = dy;
    *free_out = raw < 0.99f;                       // min(0.99, .) passes the slope only on its free side
    return fminf(raw, 0.99f);
}

__global__ void __launch_bounds__(kBwdThreads)
k_blend_backward(const WorkspaceDev ws, const float *__restrict__ dL_dimage, float *__restrict__ g9, int W, int H, int TX,
                 float bg0, float bg1, float bg2)
{
    __shared__ BwdEntry s_e[kBwdBatch];
    __shared__ unsigned int s_pos[kBwdBatch];
    __shared__ float s_part[kBwdThreads / 32][kBwdBatch][9];
    __shared__ unsigned int s_max;
    const int tile = blockIdx.x, tx = tile % TX, ty = tile / TX;
    if (ws.hdr->overflow) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ix = tx * kTile + (tid & 15), iy = ty * kTile + (tid >> 4);
    const bool inside = ix < W && iy < H;
    const float px = (float)ix + 0.5f, py = (float)iy + 0.5f;
    const uint2 rg = ws.ranges[tile];
    const unsigned int L = rg.y - rg.x;
    const float thr = 0.003921568859368563f;       // (float)(1/255)
    if (tid == 0) s_max = 0;

    // ---- pass 1: the forward walk -> T_final and n_proc (entries this pixel processed) per pixel
    float T = inside ? 1.0f : 0.0f;
    unsigned int n_proc = 0;
    bool done = !inside;
    for (unsigned int b0 = 0; b0 < L; b0 += kBwdBatch) {
        __syncthreads();
        if (tid < kBwdBatch && b0 + tid < L) s_e[tid] = bwd_entry(ws, ws.vals[rg.x + b0 + tid]);
        __syncthreads();
        if (__syncthreads_and(done)) break;
        const unsigned int m = min((unsigned int)kBwdBatch, L - b0);
        for (unsigned int j = 0; j < m && !done; ++j) {
            float G, dx, dy; bool fr;
            const float a = bwd_alpha(s_e[j], px, py, &G, &fr, &dx, &dy);
            n_proc = b0 + j + 1;
            if (a < thr) continue;
            T *= 1.0f - a;
            if (T < 1e-4f) done = true;            // the blend that takes T below 1e-4 is the last one (R12)
        }
    }
    const float T_final = T;
    atomicMax(&s_max, n_proc);
    __syncthreads();
    const unsigned int n_max = s_max;

    float dl0 = 0.f, dl1 = 0.f, dl2 = 0.f;
    if (inside) {
        const size_t o = (size_t)iy * W + ix, plane = (size_t)W * H;
        dl0 = dL_dimage[o]; dl1 = dL_dimage[plane + o]; dl2 = dL_dimage[2 * plane + o];
    }
    const float bg_dot = bg0 * dl0 + bg1 * dl1 + bg2 * dl2;

    // ---- pass 2: back to front
    float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, last_a = 0.f, lc0 = 0.f, lc1 = 0.f, lc2 = 0.f;
    for (unsigned int hi = n_max; hi > 0;) {
        const unsigned int b0 = (hi - 1) / kBwdBatch * kBwdBatch, m = hi - b0;
        __syncthreads();
        if (tid < (int)m) { const unsigned int p = ws.vals[rg.x + b0 + tid]; s_pos[tid] = p; s_e[tid] = bwd_entry(ws, p); }
        for (unsigned int i = tid; i < (kBwdThreads / 32) * kBwdBatch * 9; i += kBwdThreads) (&s_part[0][0][0])[i] = 0.0f;
        __syncthreads();
        for (int j = (int)m - 1; j >= 0; --j) {
            float v[9] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            bool contrib = false;
            if (b0 + (unsigned int)j < n_proc) {
                const BwdEntry e = s_e[j];
                float G, dx, dy; bool fr;
                const float a = bwd_alpha(e, px, py, &G, &fr, &dx, &dy);
                if (a >= thr) {
                    contrib = true;
                    T = T / (1.0f - a);                                       // transmittance in front of this entry
                    const float w = a * T;
                    v[6] = w * dl0; v[7] = w * dl1; v[8] = w * dl2;           // dL/d rgb
                    acc0 = last_a * lc0 + (1.0f - last_a) * acc0;             // colour arriving from behind this entry
                    acc1 = last_a * lc1 + (1.0f - last_a) * acc1;
                    acc2 = last_a * lc2 + (1.0f - last_a) * acc2;
                    lc0 = e.r; lc1 = e.g; lc2 = e.b; last_a = a;
                    float dL_da = ((e.r - acc0) * dl0 + (e.g - acc1) * dl1 + (e.b - acc2) * dl2) * T;
                    dL_da -= T_final / (1.0f - a) * bg_dot;                   // the background seen through everything
                    if (fr) {
                        const float q = 0.5f * (e.A * dx * dx + e.C * dy * dy) + e.B * dx * dy;
                        v[5] = G * dL_da;                                     // dL/do
                        if (q > 0.0f) {                                       // max(0, q): no slope below
                            const float dL_dG = e.o * dL_da, gG = G * dL_dG;
                            v[0] = -gG * (e.A * dx + e.B * dy);               // dL/dmu'x (d = mu' - pixel)
                            v[1] = -gG * (e.C * dy + e.B * dx);
                            v[2] = -0.5f * gG * dx * dx;                      // dL/dA
                            v[3] = -gG * dx * dy;                             // dL/dB
                            v[4] = -0.5f * gG * dy * dy;                      // dL/dC
                        }
                    }
                }
            }
            if (!__any_sync(0xffffffffu, contrib)) continue;
#pragma unroll
            for (int k = 0; k < 9; ++k) {
                float x = v[k];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
                if (lane == 0) s_part[warp][j][k] = x;
            }
        }
        __syncthreads();
        for (unsigned int i = tid; i < m * 9; i += kBwdThreads) {
            const unsigned int j = i / 9, k = i % 9;
            float x = 0.0f;
#pragma unroll
            for (int w = 0; w < kBwdThreads / 32; ++w) x += s_part[w][j][k];
            if (x != 0.0f) atomicAdd(g9 + (size_t)s_pos[j] * 9 + k, x);
        }
        hi = b0;
    }
}

// real SH constants of DESIGN R16 (as in preprocess.cu)
#define BSH_C0 0.28209479177387814f
#define BSH_C1 0.4886025119029199f
#define BSH_C2A 1.0925484305920792f
#define BSH_C2B 0.31539156525252005f
#define BSH_C2C 0.5462742152960396f
#define BSH_C3A 0.5900435899266435f
#define BSH_C3B 2.890611442640554f
#define BSH_C3C 0.4570457994644658f
#define BSH_C3D 0.3731763325901154f
#define BSH_C3E 1.445305721320277f

// Y_k and its gradient with respect to the (unit) direction, k < (deg + 1)^2
__device__ void sh_basis_grad(int deg, float x, float y, float z, float *Y, float (*dY)[3])
{
    Y[0] = BSH_C0; dY[0][0] = dY[0][1] = dY[0][2] = 0.f;
    if (deg < 1) return;
    Y[1] = -BSH_C1 * y; dY[1][0] = 0.f; dY[1][1] = -BSH_C1; dY[1][2] = 0.f;
    Y[2] = BSH_C1 * z;  dY[2][0] = 0.f; dY[2][1] = 0.f; dY[2][2] = BSH_C1;
    Y[3] = -BSH_C1 * x; dY[3][0] = -BSH_C1; dY[3][1] = 0.f; dY[3][2] = 0.f;
    if (deg < 2) return;
    const float xx = x * x, yy = y * y, zz = z * z;
    Y[4] = BSH_C2A * x * y;  dY[4][0] = BSH_C2A * y; dY[4][1] = BSH_C2A * x; dY[4][2] = 0.f;
    Y[5] = -BSH_C2A * y * z; dY[5][0] = 0.f; dY[5][1] = -BSH_C2A * z; dY[5][2] = -BSH_C2A * y;
    Y[6] = BSH_C2B * (2.f * zz - xx - yy); dY[6][0] = -2.f * BSH_C2B * x; dY[6][1] = -2.f * BSH_C2B * y; dY[6][2] = 4.f * BSH_C2B * z;
    Y[7] = -BSH_C2A * x * z; dY[7][0] = -BSH_C2A * z; dY[7][1] = 0.f; dY[7][2] = -BSH_C2A * x;
    Y[8] = BSH_C2C * (xx - yy); dY[8][0] = 2.f * BSH_C2C * x; dY[8][1] = -2.f * BSH_C2C * y; dY[8][2] = 0.f;
    if (deg < 3) return;
    Y[9] = -BSH_C3A * y * (3.f * xx - yy); dY[9][0] = -BSH_C3A * 6.f * x * y; dY[9][1] = -BSH_C3A * (3.f * xx - 3.f * yy); dY[9][2] = 0.f;
    Y[10] = BSH_C3B * x * y * z; dY[10][0] = BSH_C3B * y * z; dY[10][1] = BSH_C3B * x * z; dY[10][2] = BSH_C3B * x * y;
    Y[11] = -BSH_C3C * y * (4.f * zz - xx - yy);
    dY[11][0] = BSH_C3C * 2.f * x * y; dY[11][1] = -BSH_C3C * (4.f * zz - xx - 3.f * yy); dY[11][2] = -BSH_C3C * 8.f * y * z;
    Y[12] = BSH_C3D * z * (2.f * zz - 3.f * xx - 3.f * yy);
    dY[12][0] = -BSH_C3D * 6.f * x * z; dY[12][1] = -BSH_C3D * 6.f * y * z; dY[12][2] = BSH_C3D * (6.f * zz - 3.f * xx - 3.f * yy);
    Y[13] = -BSH_C3C * x * (4.f * zz - xx - yy);
    dY[13][0] = -BSH_C3C * (4.f * zz - 3.f * xx - yy); dY[13][1] = BSH_C3C * 2.f * x * y; dY[13][2] = -BSH_C3C * 8.f * x * z;
    Y[14] = BSH_C3E * z * (xx - yy); dY[14][0] = BSH_C3E * 2.f * x * z; dY[14][1] = -BSH_C3E * 2.f * y * z; dY[14][2] = BSH_C3E * (xx - yy);
    Y[15] = -BSH_C3A * x * (xx - 3.f * yy); dY[15][0] = -BSH_C3A * (3.f * xx - 3.f * yy); dY[15][1] = BSH_C3A * 6.f * x * y; dY[15][2] = 0.f;
}

// index of coefficient (k, ch) inside a stored SH row (degree 3 rows are laid out for k_colour's four lanes, see flod_upload_levels)
__device__ __forceinline__ int sh_slot(int deg, int k, int ch)
{
    const int f = 3 * k + ch;
    if (deg != 3) return f;
    const int j = f / 12, within = f % 12;
    return ((within / 4) * 4 + j) * 4 + (within % 4);
}

__global__ void __launch_bounds__(128)
k_project_backward(const SceneDev sc, const WorkspaceDev ws, const __grid_constant__ FrameParams p, const float *__restrict__ g9,
                   const flod_grads out)
{
    const unsigned int seg = blockIdx.x, nv = ws.seg_count[seg];
    const float *R = p.R;
    for (unsigned int j = threadIdx.x; j < nv; j += blockDim.x) {
        const size_t c = (size_t)seg * kGeoBlock + j;
        const size_t g = __float_as_uint(ws.dirgid[c].w);                    // gid (the frame scanned the scene itself)
        const float *gr = g9 + c * 9;
        const float gmx = gr[0], gmy = gr[1], gA = gr[2], gB = gr[3], gC = gr[4], go = gr[5];
        const float grgb[3] = {gr[6], gr[7], gr[8]};
        // ---- forward recomputed (plain fp32)
        const float wx = sc.mx[g], wy = sc.my[g], wz = sc.mz[g];
        const float S00 = sc.cov[0][g], S01 = sc.cov[1][g], S02 = sc.cov[2][g], S11 = sc.cov[3][g], S12 = sc.cov[4][g], S22 = sc.cov[5][g];
        const float x = R[0] * wx + R[1] * wy + R[2] * wz + p.t[0];
        const float y = R[3] * wx + R[4] * wy + R[5] * wz + p.t[1];
        const float z = R[6] * wx + R[7] * wy + R[8] * wz + p.t[2];
        const float rz = 1.0f / z, ix = x * rz, iy = y * rz;
        const float u = fminf(fmaxf(ix, -p.limx), p.limx), v = fminf(fmaxf(iy, -p.limy), p.limy);
        const float cu = (ix > -p.limx && ix < p.limx) ? 1.0f : 0.0f, cv = (iy > -p.limy && iy < p.limy) ? 1.0f : 0.0f;
        const float j00 = p.fx * rz, j02 = -p.fx * u * rz, j11 = p.fy * rz, j12 = -p.fy * v * rz;
        const float m0[3] = {j00 * R[0] + j02 * R[6], j00 * R[1] + j02 * R[7], j00 * R[2] + j02 * R[8]};
        const float m1[3] = {j11 * R[3] + j12 * R[6], j11 * R[4] + j12 * R[7], j11 * R[5] + j12 * R[8]};
        const float v0[3] = {S00 * m0[0] + S01 * m0[1] + S02 * m0[2], S01 * m0[0] + S11 * m0[1] + S12 * m0[2], S02 * m0[0] + S12 * m0[1] + S22 * m0[2]};
        const float v1[3] = {S00 * m1[0] + S01 * m1[1] + S02 * m1[2], S01 * m1[0] + S11 * m1[1] + S12 * m1[2], S02 * m1[0] + S12 * m1[1] + S22 * m1[2]};
        const float a = m0[0] * v0[0] + m0[1] * v0[1] + m0[2] * v0[2] + 0.3f;
        const float b = m1[0] * v0[0] + m1[1] * v0[1] + m1[2] * v0[2];
        const float cc = m1[0] * v1[0] + m1[1] * v1[1] + m1[2] * v1[2] + 0.3f;
        const float det = a * cc - b * b, id2 = 1.0f / (det * det);
        // ---- conic (A, B, C) = (c, -b, a) / det
        const float da = (-cc * cc * gA + b * cc * gB - b * b * gC) * id2;
        const float db = (2.0f * b * cc * gA - (det + 2.0f * b * b) * gB + 2.0f * a * b * gC) * id2;
        const float dc = (-b * b * gA + a * b * gB - a * a * gC) * id2;
        // ---- Sigma' = M Sigma M^T + 0.3 I: gradient with respect to Sigma (as a full symmetric matrix) and to M
        float Gs[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k)
#pragma unroll
            for (int l = 0; l < 3; ++l) Gs[k][l] = da * m0[k] * m0[l] + 0.5f * db * (m0[k] * m1[l] + m0[l] * m1[k]) + dc * m1[k] * m1[l];
        float dm0[3], dm1[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { dm0[k] = 2.0f * da * v0[k] + db * v1[k]; dm1[k] = 2.0f * dc * v1[k] + db * v0[k]; }
        const float dj00 = dm0[0] * R[0] + dm0[1] * R[1] + dm0[2] * R[2], dj02 = dm0[0] * R[6] + dm0[1] * R[7] + dm0[2] * R[8];
        const float dj11 = dm1[0] * R[3] + dm1[1] * R[4] + dm1[2] * R[5], dj12 = dm1[0] * R[6] + dm1[1] * R[7] + dm1[2] * R[8];
        // ---- J(p) and mu' = pinhole(p)
        const float rz2 = rz * rz;
        const float du = -p.fx * rz * dj02, dv = -p.fy * rz * dj12;
        float dx = p.fx * rz * gmx + cu * du * rz;
        float dy = p.fy * rz * gmy + cv * dv * rz;
        float dz = -(p.fx * x * gmx + p.fy * y * gmy) * rz2 - p.fx * rz2 * dj00 + p.fx * u * rz2 * dj02 - p.fy * rz2 * dj11 + p.fy * v * rz2 * dj12
                   - cu * du * x * rz2 - cv * dv * y * rz2;
        float dmean[3] = {R[0] * dx + R[3] * dy + R[6] * dz, R[1] * dx + R[4] * dy + R[7] * dz, R[2] * dx + R[5] * dy + R[8] * dz};
        // ---- Sigma = (R_g S)(R_g S)^T (Eq. 1): scale and rotation
        const float s[3] = {expf(sc.raw[0][g]), expf(sc.raw[1][g]), expf(sc.raw[2][g])};
        float qw = sc.raw[3][g], qx = sc.raw[4][g], qy = sc.raw[5][g], qz = sc.raw[6][g];
        const float qn = sqrtf(qw * qw + qx * qx + qy * qy + qz * qz), rq = 1.0f / qn;
        qw *= rq; qx *= rq; qy *= rq; qz *= rq;
        const float Rg[3][3] = {{1.f - 2.f * (qy * qy + qz * qz), 2.f * (qx * qy - qw * qz), 2.f * (qx * qz + qw * qy)},
                                {2.f * (qx * qy + qw * qz), 1.f - 2.f * (qx * qx + qz * qz), 2.f * (qy * qz - qw * qx)},
                                {2.f * (qx * qz - qw * qy), 2.f * (qy * qz + qw * qx), 1.f - 2.f * (qx * qx + qy * qy)}};
        float dM[3][3], dRg[3][3], dls[3];                                   // dL/d(R_g S) = 2 G (R_g S)
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int k = 0; k < 3; ++k) dM[i][k] = 2.0f * (Gs[i][0] * Rg[0][k] + Gs[i][1] * Rg[1][k] + Gs[i][2] * Rg[2][k]) * s[k];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            dls[k] = (dM[0][k] * Rg[0][k] + dM[1][k] * Rg[1][k] + dM[2][k] * Rg[2][k]) * s[k];      // d/d log s = s d/ds
#pragma unroll
            for (int i = 0; i < 3; ++i) dRg[i][k] = dM[i][k] * s[k];
        }
        float dq[4];
        dq[0] = 2.f * (-qz * dRg[0][1] + qy * dRg[0][2] + qz * dRg[1][0] - qx * dRg[1][2] - qy * dRg[2][0] + qx * dRg[2][1]);
        dq[1] = 2.f * (qy * dRg[0][1] + qz * dRg[0][2] + qy * dRg[1][0] - 2.f * qx * dRg[1][1] - qw * dRg[1][2] + qz * dRg[2][0] + qw * dRg[2][1] - 2.f * qx * dRg[2][2]);
        dq[2] = 2.f * (-2.f * qy * dRg[0][0] + qx * dRg[0][1] + qw * dRg[0][2] + qx * dRg[1][0] + qz * dRg[1][2] - qw * dRg[2][0] + qz * dRg[2][1] - 2.f * qy * dRg[2][2]);
        dq[3] = 2.f * (-2.f * qz * dRg[0][0] - qw * dRg[0][1] + qx * dRg[0][2] + qw * dRg[1][0] - 2.f * qz * dRg[1][1] + qy * dRg[1][2] + qx * dRg[2][0] + qy * dRg[2][1]);
        const float qd = qw * dq[0] + qx * dq[1] + qy * dq[2] + qz * dq[3];          // through q / |q|
        const float qh[4] = {qw, qx, qy, qz};
        // ---- colour: rgb = max(0, 0.5 + sum_k Y_k(dir) sh_k), dir = (mu - centre) / |mu - centre|
        const int deg = sc.sh_degree, K = (deg + 1) * (deg + 1);
        const float ddx = wx - p.centre[0], ddy = wy - p.centre[1], ddz = wz - p.centre[2];
        const float dn = sqrtf(ddx * ddx + ddy * ddy + ddz * ddz), rdn = 1.0f / dn;
        const float ux = ddx * rdn, uy = ddy * rdn, uz = ddz * rdn;
        float Y[16], dY[16][3];
        sh_basis_grad(deg, ux, uy, uz, Y, dY);
        const float *row = sc.sh + g * sc.sh_stride;
        float pre[3] = {0.5f, 0.5f, 0.5f};
        for (int k = 0; k < K; ++k)
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) pre[ch] += Y[k] * row[sh_slot(deg, k, ch)];
        float gch[3];
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) gch[ch] = pre[ch] > 0.0f ? grgb[ch] : 0.0f;
        float ddir[3] = {0.f, 0.f, 0.f};
        for (int k = 0; k < K; ++k) {
            float wsum = 0.0f;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                out.d_sh[(g * K + k) * 3 + ch] = Y[k] * gch[ch];
                wsum += row[sh_slot(deg, k, ch)] * gch[ch];
            }
            ddir[0] += dY[k][0] * wsum; ddir[1] += dY[k][1] * wsum; ddir[2] += dY[k][2] * wsum;
        }
        const float ud = ux * ddir[0] + uy * ddir[1] + uz * ddir[2];                  // through the normalisation
        dmean[0] += (ddir[0] - ux * ud) * rdn; dmean[1] += (ddir[1] - uy * ud) * rdn; dmean[2] += (ddir[2] - uz * ud) * rdn;
        // ---- write (one thread per Gaussian: no atomics)
        const float o = sc.opacity[g];
#pragma unroll
        for (int k = 0; k < 3; ++k) { out.d_mean[g * 3 + k] = dmean[k]; out.d_log_scale[g * 3 + k] = dls[k]; }
#pragma unroll
        for (int k = 0; k < 4; ++k) out.d_quat[g * 4 + k] = (dq[k] - qh[k] * qd) * rq;
        out.d_opacity_logit[g] = o * (1.0f - o) * go;
    }
}

int launch_backward(const Context &c, const FrameParams &p, const float *dL_dimage, float *g9, const flod_grads &out, cudaStream_t s)
{
    if (p.n_tiles > 0)
        k_blend_backward<<<p.n_tiles, kBwdThreads, 0, s>>>(c.ws, dL_dimage, g9, p.W, p.H, p.TX, p.bg[0], p.bg[1], p.bg[2]);
    if (p.n_pre_blocks > 0) k_project_backward<<<p.n_pre_blocks, 128, 0, s>>>(c.scene, c.ws, p, g9, out);
    return 2;
}

}  // namespace flod
