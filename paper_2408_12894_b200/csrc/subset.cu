// Materialised G_sel (Eq. 6-7; the paper's runtime for long trajectories):
// the Gaussians of the level range that pass Eq. 6 for one reference position are copied, in gid order, into a
// SNAPSHOT that k_geometry then scans instead of the scene (no predicate, no rejected Gaussians: N_sel instead of
// N_scan entries per frame).  Three kernels per rebuild, on whatever stream the caller gives (a second stream for an
// asynchronous rebuild):
//   k_subset_count    Eq. 6 per Gaussian (the canonical fp32 sequence O1 of DESIGN §2, as in k_geometry), selected
//                     Gaussians per block of 1024;
//   k_subset_scan     one CTA: exclusive scan of the block counts, total = N_sel;
//   k_subset_scatter  the predicate again, rank inside the block by ballot, the 15 plane values of every selected
//                     Gaussian copied to offset[block] + rank.  Stable, so gid order (the depth tie-break R15) is kept.
// Traffic per rebuild: 2 x 12 B x N_scan read + (56 B read + 60 B written) x N_sel.
#include "flod_internal.cuh"

namespace flod {

constexpr int kSubThreads = 256;
constexpr int kSubPer = 4;
constexpr int kSubBlock = kSubThreads * kSubPer;

// Eq. 6 for the four consecutive Gaussians g0 .. g0 + 3 of a thread (g0 a multiple of 4): bit k = selected.
// Same operations, same order as phase 1 of k_geometry (O1): d2 = (dx dx + dy dy) + dz dz, lo2 <= d2 < hi2.
__device__ __forceinline__ unsigned int subset_select4(const SceneDev &sc, const SubsetParams &q, long long g0)
{
    const long long g_end = q.first_gid + q.n_scan;
    if (!(g0 < g_end && g0 + kSubPer > q.first_gid)) return 0u;
    const float4 X = __ldg(reinterpret_cast<const float4 *>(sc.mx + g0));
    const float4 Y = __ldg(reinterpret_cast<const float4 *>(sc.my + g0));
    const float4 Z = __ldg(reinterpret_cast<const float4 *>(sc.mz + g0));
    const float wx[4] = {X.x, X.y, X.z, X.w}, wy[4] = {Y.x, Y.y, Y.z, Y.w}, wz[4] = {Z.x, Z.y, Z.z, Z.w};
    unsigned int m = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const long long g = g0 + k;
        if (g < q.first_gid || g >= g_end) continue;
        const int i = (int)(g - q.first_gid);
        int lv = 0;
#pragma unroll 1
        while (lv < q.n_levels - 1 && i >= q.level_end[lv]) ++lv;
        const float dx = __fsub_rn(wx[k], q.ref[0]), dy = __fsub_rn(wy[k], q.ref[1]), dz = __fsub_rn(wz[k], q.ref[2]);
        const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
        const bool sel = (d2 >= q.lo2[lv]) && (d2 < q.hi2[lv]);
        if (sel) m |= 1u << k;
    }
    return m;
}

__global__ void __launch_bounds__(kSubThreads)
k_subset_count(const SceneDev sc, const __grid_constant__ SubsetParams q, unsigned int *__restrict__ blk)
{
    __shared__ unsigned int s_tot;
    if (threadIdx.x == 0) s_tot = 0;
    __syncthreads();
    const long long g0 = (q.first_gid & ~3ll) + (long long)blockIdx.x * kSubBlock + threadIdx.x * kSubPer;
    unsigned int n = __popc(subset_select4(sc, q, g0));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(&s_tot, n);
    __syncthreads();
    if (threadIdx.x == 0) blk[blockIdx.x] = s_tot;
}

// blk[0 .. n_blocks) counts -> exclusive offsets in place; blk[n_blocks] = *n_sel = total.
__global__ void __launch_bounds__(1024)
k_subset_scan(unsigned int *__restrict__ blk, int n_blocks, unsigned int *__restrict__ n_sel)
{
    __shared__ unsigned int s_wtot[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = (n_blocks + 1023) / 1024;
    const int b0 = min(tid * per, n_blocks), b1 = min(b0 + per, n_blocks);
    unsigned int sum = 0;
    for (int b = b0; b < b1; ++b) sum += blk[b];
    unsigned int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_wtot[warp] = incl;
    __syncthreads();
    unsigned int run = incl - sum, total = 0;
    for (int w = 0; w < 32; ++w) {
        const unsigned int t = s_wtot[w];
        if (w < warp) run += t;
        total += t;
    }
    for (int b = b0; b < b1; ++b) {
        const unsigned int c = blk[b];
        blk[b] = run;
        run += c;
    }
    if (tid == 0) { blk[n_blocks] = total; *n_sel = total; }
}

__global__ void __launch_bounds__(kSubThreads)
k_subset_scatter(const SceneDev sc, const __grid_constant__ SubsetParams q, const unsigned int *__restrict__ blk,
                 const SnapshotDev dst)
{
    __shared__ unsigned int s_warp[kSubThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long g0 = (q.first_gid & ~3ll) + (long long)blockIdx.x * kSubBlock + tid * kSubPer;
    const unsigned int m = subset_select4(sc, q, g0);
    const unsigned int n = __popc(m);
    unsigned int incl = n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned int pos = blk[blockIdx.x] + incl - n;           // gid order = thread order, then k
    for (int w = 0; w < warp; ++w) pos += s_warp[w];
    if (!m) return;
    const float *src[13] = {sc.mx, sc.my, sc.mz, sc.rho2, sc.kappa, sc.cov[0], sc.cov[1], sc.cov[2], sc.cov[3], sc.cov[4],
                            sc.cov[5], sc.l2o, sc.opacity};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (!((m >> k) & 1u)) continue;
        const long long g = g0 + k;
#pragma unroll
        for (int a = 0; a < 13; ++a) dst.plane[a][pos] = __ldg(src[a] + g);
        dst.src_gid[pos] = (unsigned int)g;
        dst.rec[2 * (size_t)pos] = __ldg(sc.rec + 2 * g); dst.rec[2 * (size_t)pos + 1] = __ldg(sc.rec + 2 * g + 1);
        ++pos;
    }
}

int launch_subset_build(const Context &c, const SnapshotDev &dst, const SubsetParams &q, cudaStream_t s)
{
    if (q.n_blocks > 0) k_subset_count<<<q.n_blocks, kSubThreads, 0, s>>>(c.scene, q, c.sub_blk);
    k_subset_scan<<<1, 1024, 0, s>>>(c.sub_blk, q.n_blocks, dst.n_sel);
    if (q.n_blocks > 0) k_subset_scatter<<<q.n_blocks, kSubThreads, 0, s>>>(c.scene, q, c.sub_blk, dst);
    return q.n_blocks > 0 ? 3 : 1;
}

}  // namespace flod
