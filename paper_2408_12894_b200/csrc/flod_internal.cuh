// Internal declarations of libflod (host context, device layouts, kernel launchers).
// Nothing here is shared with oracle/ -- the two implementations are written independently from DESIGN.md §2.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/flod.h"
#include "span.cuh"

namespace flod {

constexpr int kTile = FLOD_TILE;
constexpr int kPreBlock = 256;            // duplication: visible Gaussians per block step
constexpr int kGeoThreads = 128;   // geometry: threads per block, kGeoPer consecutive Gaussians per thread
constexpr int kGeoPer = 1024 / kGeoThreads;     // a block scans 1024 Gaussians = one segment
static_assert(kGeoPer % 4 == 0 && kGeoPer * kGeoThreads == 1024, "whole quads per thread, 1024 per block");
constexpr int kGeoBlock = kGeoThreads * kGeoPer;
constexpr int kSortCap = 4096;            // per-tile sort: lists up to this many keys are scattered into shared memory
constexpr int kCoarseBins = 256;          // ... longer ones are first cut into at most this many depth slices
// duplication: frames whose mean rect exceeds this many tiles are served by k_duplicate_shared (since several CTAs share a
// segment in k_duplicate it wins far beyond the 128 of round 1 -- config 3, level 1, mean rect 548 tiles: 240 -> 142 us,
// level 2, mean 210: 306 -> 198 us); FLOD_OPT_SMALL_WINDOWS keeps the old threshold, for the tests of that kernel
constexpr unsigned int kDupLargeArea = 1024, kDupLargeAreaTest = 128;
constexpr int kCtrStride = 64;            // ints between two per-tile atomic counters: one counter per 256 B, so that the
                                          // L2 slices share the atomic traffic (a dense 16 KB grid sits on a few slices)

// Scene planes in the caller's arena (SoA, one plane per attribute, gid order = levels concatenated).
struct SceneDev {
    const float *mx, *my, *mz;            // mean
    const float *cov[6];                  // Sigma xx,xy,xz,yy,yz,zz (Eq. 1)
    const float *opacity;                 // o (debug only on the device)
    const float *kappa;                   // 2 ln(255 o); -1 when dead
    const float *l2o;                     // log2(o)
    const float *rho2;                    // kappa * largest eigenvalue of Sigma, rounded up (squared bounding radius); -1 when dead
    const float4 *rec;                    // [n][2]: (Sxx, Sxy, Sxz, Syy), (Syz, Szz, kappa, log2 o) -- what phase 2 of k_geometry reads
                                          // of a candidate, as ONE 32-byte sector (the planes above cost nine sectors, most
                                          // of each unused at the 45 % density of the candidates)
    const float *raw[8];                  // the uploaded log_scale xyz, quat wxyz, opacity logit (read by the backward pass only)
    const float *sh;                      // [n][sh_stride] floats, row = K*3 coefficients padded to a multiple of 4
    int sh_stride;
    int sh_degree;
    const unsigned int *src_gid;          // snapshots only (subset.cu): scene gid of every entry; nullptr for the scene itself
};

// One materialised G_sel (subset.cu): compacted copies of the planes k_geometry reads, in gid order.
struct SnapshotDev {
    float *plane[13];                     // mx, my, mz, rho2, kappa, cov[0..5], l2o, opacity
    unsigned int *src_gid;
    float4 *rec;                          // [cap][2] as SceneDev::rec
    unsigned int *n_sel;                  // device copy of the count (written by the rebuild)
};

// Selection parameters of a rebuild (the selection half of FrameParams).
struct SubsetParams {
    float ref[3];
    long long first_gid;
    int n_scan, n_levels;
    int level_end[FLOD_MAX_LEVELS];
    float lo2[FLOD_MAX_LEVELS], hi2[FLOD_MAX_LEVELS];
    int n_blocks;
};

// Per-frame counters.  Two of them alternate from frame to frame: k_blend of frame k zeroes the header of frame k + 1 (its
// own is still wanted by flod_get_stats), the tile scan zeroes the cells of the difference grid as it reads them -- so a
// frame starts without a memset in the stream, and k_geometry can be launched programmatically behind the previous frame.
struct FrameHeader {
    unsigned int n_vis32;                 // visible Gaussians = length of the compact per-frame arrays
    unsigned int overflow;
    unsigned int n_pairs_clamped;         // min(n_pairs, max_pairs)
    unsigned int cursor_abs;              // k_duplicate's float counters hold absolute pair positions (the frame has <= 2^24 pairs)
    unsigned long long n_sel, n_front, n_pairs;   // n_pairs = pairs the frame requires (sum of rect areas)
    unsigned long long evals, blends;
    unsigned int n_todo;                  // blend-driven ordering: tiles whose first blend round asked for the rest of their list
    unsigned int pad2[3];
};

// Everything per Gaussian is indexed by the POSITION p = segment * kGeoBlock + j: block `segment` of k_geometry
// scans kGeoBlock consecutive gids and writes the records of its seg_count[segment] visible ones, in ascending gid
// order, at the front of its segment (j < seg_count).  So p-order = gid-order, every segment is a dense run of full
// sectors, and no inter-block scan is needed.  Blend features (DESIGN R25):
//   gA = (mu'x, mu'y, k = B/A, -A log2(e)/2)     gB = (min(0, -(C - B^2/A) log2(e)/2), log2 o, r, g)    cB = b
struct WorkspaceDev {
    FrameHeader *hdr;                     // this frame's header (one of hdr2)
    FrameHeader *hdr_next;                // the next frame's: zeroed by this frame's k_blend
    FrameHeader *hdr2[2];
    int *tile_diff;                       // [(TX+1)*(TY+1)][kCtrStride] 2-D difference grid of the tile counts (zeroed per frame)
    unsigned int *seg_count;              // [geometry blocks] visible Gaussians of every segment
    int *tile_cnt;                        // [(TX+1)*(TY+1)] dense copy, used by the tile scan when the grid exceeds shared memory
    uint2 *ranges;                        // [T_n] (start, end) of every tile's pair list
    float *cursor4;                       // [ceil(TX/2) * ceil(TY/2)][kCtrStride] first 4 floats: entries appended so far to the
                                          // lists of the 2x2 tile group (x, y), (x+1, y), (x, y+1), (x+1, y+1); zeroed by the tile scan
    unsigned int *cursor;                 // [T_n] the same per tile, dense (k_duplicate_shared); zeroed by the tile scan
    unsigned int dup_large_area;          // kDupLargeArea, or kDupLargeAreaTest under FLOD_OPT_SMALL_WINDOWS (set per frame by the host)
    float *cnt4;                          // [ceil(TX/2) * ceil(TY/2)][kCtrStride] first 4 floats: pairs of the group's four tiles that
                                          // come from rects of at most 2x2 groups (k_geometry, pair rule 1); read and zeroed by the tile scan
    float4 *gA, *gB;                      // [n_total + 2 kGeoBlock]
    float *cB;                            // [n_total + 2 kGeoBlock]
    float4 *dirgid;                       // [n_total + 2 kGeoBlock] (mu - c_cam, gid bits): input of the colour kernel
    ushort4 *rect;                        // [n_total + 2 kGeoBlock] tx0, ty0, tx1, ty1
    uint32_t *depth;                      // [n_total + 2 kGeoBlock] depth bits (p_z > 0, so unsigned order = float order)
    flod_dbg_projected *dbg;              // [n_total + 2 kGeoBlock] (written only with FLOD_OPT_DEBUG)
    uint8_t *mask;                        // [n_total + 2 kGeoBlock] (written only with FLOD_OPT_DEBUG)
    unsigned long long *pairs;            // [max_pairs] (depth bits << 32) | position, grouped by tile, unsorted
    unsigned long long *pairs_tmp;        // [max_pairs] scatter target of the per-tile sort for lists longer than kSortCap
    uint32_t *vals;                       // [max_pairs] positions, grouped by tile, sorted by (depth, gid)
    unsigned int *ovf_slots;              // [3] overflow word of the frame rendered into image[0], image[1], and of any other frame
    unsigned int *ovf_out;                // where THIS frame's tile scan reports (set on the host before the launches)
    uint4 *lazy;                          // [T_n] lists longer than kSortCap, blend-driven ordering: (keys in final order so far, next
                                          // slice to sort, slices, 1 = the blend wants the rest)
    unsigned int *slice_ends;             // [T_n][kCoarseBins] ends of the depth slices of those lists
    unsigned int *long_hint;              // mapped pinned host word, written by the tile scan when it changes: bit 0 = a quarter of the frame's pairs sit in
                                          // lists longer than kSortCap, bit 1 = the frame's rects are large (dup_large_rects): hints about cost for the next frames
                                          // the host reads it, unsynchronised, as a hint for the NEXT frame (lazy ordering or not)
    unsigned int *hint_state;             // device copy of what long_hint was last set to (| 0x100), zeroed by flod_set_workspace
    unsigned int *todo;                   // [T_n] those tiles (hdr->n_todo of them), in the order they asked
    float4 *tile_state;                   // [T_n][256] (T, r, g, b) of every pixel of a tile the blend left unfinished
    float *image[2];                      // 2 x [3][H][W] for flod_render_to_host(_async): double-buffered so that the copy
                                          // of frame k overlaps the kernels of frame k + 1
};

struct FrameParams {
    float R[9], t[3];
    float fx, fy, cx, cy, z_near;
    float limx, limy;                     // 1.3 W / (2 fx), 1.3 H / (2 fy), fp64 -> fp32 once
    float pre_c1;                         // max(fx, fy)^2 (1 + max(limx, limy)^2), rounded up
    float centre[3];                      // -R^T t, fp64 -> fp32 once
    float ref[3];                         // selection reference (R2)
    float bg[3];
    int W, H, TX, TY;
    long long first_gid;                  // gid of the first scanned Gaussian
    long long quad_gid;                   // first_gid rounded down to a multiple of 4: thread q of k_geometry owns
                                          // gids quad_gid + 4 q .. + 3 (16-byte aligned in every plane)
    int n_scan;
    int n_levels;                         // levels in the range
    int level_end[FLOD_MAX_LEVELS];       // cumulative end (scan index) of each level in the range
    float lo2[FLOD_MAX_LEVELS], hi2[FLOD_MAX_LEVELS];
    unsigned int max_pairs;
    int n_pre_blocks;                     // blocks of k_geometry
    int n_tiles;                          // TX * TY
    int pair_rule;                        // FLOD_PAIR_RULE_BOX / FLOD_PAIR_RULE_ELLIPSE
    int ty_begin, ty_end;                 // the strip of tile rows this frame renders ([0, TY) = the whole image): rects are
                                          // clipped to it, tiles outside it get no pairs and are not blended
    int out_row0, out_rows;               // out_rgb holds image rows [out_row0, out_row0 + out_rows) of every colour plane
    int lazy_sort;                        // blend-driven ordering of long lists (off for the debug / counting / training views)
    int dup_both;                         // both duplication kernels are launched and the device picks (the previous frames had
                                          // large rects); otherwise k_duplicate alone serves the frame, whatever its rects
};

struct Context {
    int device = 0;
    int sm_count = 148;
    std::string err;
    // scene
    bool uploaded = false;
    int n_levels = 0, first_level = 0, sh_degree = 0;
    int64_t level_off[FLOD_MAX_LEVELS + 1] = {0};
    float s_min[FLOD_MAX_LEVELS] = {0};
    int64_t n_total = 0;
    SceneDev scene{};
    void *arena = nullptr;
    // workspace
    bool has_ws = false;
    WorkspaceDev ws{};
    int ws_w = 0, ws_h = 0;
    int64_t max_pairs = 0;
    // options / state
    unsigned flags = 0;
    int pair_rule = FLOD_PAIR_RULE_BOX;
    bool has_ref = false;
    float ref[3] = {0, 0, 0};
    cudaStream_t last_stream = nullptr;
    bool rendered = false;
    FrameParams last_params{};            // of the last frame enqueued by flod_render (what flod_render_backward differentiates)
    bool last_full_scene = false;         // ... and whether it scanned the scene arena itself (not a snapshot)
    int last_w = 0, last_h = 0, last_tx = 0, last_ty = 0;
    int64_t last_first_gid = 0;
    int64_t last_n_scan = 0;
    int last_n_segs = 0;
    cudaEvent_t ev[FLOD_N_STAGES + 1] = {nullptr};
    cudaEvent_t ev_rendered[2] = {nullptr, nullptr};   // image[i] complete on the render stream
    cudaEvent_t ev_copied[2] = {nullptr, nullptr};     // image[i] copied out on the copy stream (free to overwrite)
    bool copy_pending[2] = {false, false};
    int img_turn = 0;
    int hdr_turn = 0;                     // which of ws.hdr2 the last frame used
    cudaStream_t last_copy_stream = nullptr;
    bool ev_valid = false;
    // materialised G_sel (subset.cu)
    bool has_subset = false;
    int sub_i0 = 0, sub_i1 = 0;           // level positions of the range
    SnapshotDev snap[2]{};
    unsigned int *sub_blk = nullptr;      // [n_blocks + 1] per-block counts, then exclusive offsets
    int sub_front = 0;                    // snap[sub_front] is rendered from, the other one is rebuilt
    bool sub_front_valid = false, sub_build_pending = false;
    int64_t sub_n[2] = {0, 0};            // N_sel of each snapshot (host copy, valid after the swap)
    unsigned int *sub_n_host = nullptr;   // pinned: the rebuild's count lands here
    cudaEvent_t ev_sub_built = nullptr;   // rebuild complete (on the build stream)
    cudaEvent_t ev_sub_read[2] = {nullptr, nullptr};   // last frame that read snap[i] (on the render stream)
    bool sub_read_pending[2] = {false, false};
};

// Launch with programmatic stream serialization (PDL): the kernel's CTAs may be scheduled while the previous kernel of the
// stream is draining its last wave; every such kernel calls cudaGridDependencySynchronize() before it touches memory, so
// the data dependence is the usual one -- what overlaps is the launch latency and the tail of the previous kernel.
template <class... KArgs, class... Args>
inline void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// kernel launchers (each enqueues on `s` and returns the number of kernels launched)
int launch_geometry(const Context &c, const SceneDev &sc, const FrameParams &p, cudaStream_t s);   // a1-a3 + tile-count grid + visible list
int launch_subset_build(const Context &c, const SnapshotDev &dst, const SubsetParams &q, cudaStream_t s);   // a1 materialised
int launch_colour(const Context &c, const FrameParams &p, cudaStream_t s);      // a4, and a5 + a8 (tile scan) in block 0
int launch_duplicate(const Context &c, const FrameParams &p, cudaStream_t s);   // a6
int init_duplicate();                                                            // once per device: shared-memory opt-in
int init_tile_sort();                                                            // once per device: shared-memory opt-in
int launch_tile_sort(const Context &c, const FrameParams &p, cudaStream_t s);   // a7
int launch_tile_sort_rest(const Context &c, const FrameParams &p, cudaStream_t s);   // a7, the lists the blend did not finish
int launch_blend_rest(const Context &c, const FrameParams &p, float *out_rgb, cudaStream_t s);   // a9, those tiles
int launch_blend(const Context &c, const FrameParams &p, float *out_rgb, cudaStream_t s);   // a9
// backward pass of a9 and of a2-a4 (backward.cu); g9 = [positions][9] screen-space gradients (workspace of the backward pass)
int launch_backward(const Context &c, const FrameParams &p, const float *dL_dimage, float *g9, const flod_grads &out, cudaStream_t s);

}  // namespace flod
