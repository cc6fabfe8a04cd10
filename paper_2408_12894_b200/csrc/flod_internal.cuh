// Internal declarations of libflod (host context, device layouts, kernel launchers).
// Nothing here is shared with oracle/ -- the two implementations are written independently from DESIGN.md §2.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/flod.h"

namespace flod {

constexpr int kTile = FLOD_TILE;
constexpr int kPreBlock = 256;            // geometry / duplication: Gaussians per block
constexpr int kRadixBits = 8;             // widest digit of any radix pass
constexpr int kRadix = 1 << kRadixBits;
constexpr int kDepthPasses = 4;           // 32 depth bits, 8 per pass
constexpr int kMaxTilePasses = 3;         // tile ids < 2^20 (16384 x 16384 pixels), <= 8 bits per pass
constexpr int kMaxPasses = kDepthPasses + kMaxTilePasses;
constexpr int kDepthSortTile = 256 * 8;   // keys per onesweep block, depth passes (threads x items)
constexpr int kTileSortTile = 512 * 8;   // keys per onesweep block, tile passes

// Scene planes in the caller's arena (SoA, one plane per attribute, gid order = levels concatenated).
struct SceneDev {
    const float *mx, *my, *mz;            // mean
    const float *cov[6];                  // Sigma xx,xy,xz,yy,yz,zz (Eq. 1)
    const float *opacity;                 // o (debug only on the device)
    const float *kappa;                   // 2 ln(255 o); -1 when dead
    const float *l2o;                     // log2(o)
    const float *sh;                      // [n][sh_stride] floats, row = K*3 coefficients padded to a multiple of 4
    int sh_stride;
    int sh_degree;
};

// Per-frame counters and small state, zeroed by one memset at the start of every frame.
struct FrameHeader {
    unsigned int pre_ticket;              // virtual block ids of the geometry kernel
    unsigned int dup_ticket;              // virtual block ids of the duplication kernel
    unsigned int sort_ticket[kMaxPasses]; // virtual block ids of each onesweep pass
    unsigned int overflow;
    unsigned int n_vis32;                 // visible Gaussians (what the depth sort / colour / duplication iterate over)
    unsigned int n_pairs_clamped;         // min(n_pairs, max_pairs): what the tile sort / ranges iterate over
    unsigned int pad;
    unsigned long long n_sel, n_front, n_vis, n_pairs;   // n_pairs = required pairs
    unsigned long long evals, blends;
    unsigned int hist[kMaxPasses][kRadix];  // global digit histograms: passes 0-3 depth, 4.. tile
};

// Blend features of one visible Gaussian (compact index ci, ascending gid): see DESIGN R25.
//   gA = (mu'x, mu'y, k = B/A, -A log2(e)/2)     gB = (-(C - B^2/A) log2(e)/2, log2 o, r, g)    cB = b
struct WorkspaceDev {
    FrameHeader *hdr;
    unsigned long long *scan_status;      // [2 * pre_blocks_max] look-back words: [2b] geometry scan, [2b+1] duplication scan
    unsigned long long *sort_status;      // [sort_blocks_max][kRadix] epoch-tagged look-back, shared by all passes
    float4 *gA, *gB;                      // [n_total]
    float *cB;                            // [n_total]
    float4 *dirgid;                       // [n_total] (mu - c_cam, gid bits): input of the colour kernel
    ushort4 *rect;                        // [n_total] tx0, ty0, tx1, ty1
    uint32_t *cgid;                       // [n_total] compact index -> gid
    uint32_t *depth;                      // [n_total] depth bits by compact index (pass-0 keys; never overwritten)
    uint32_t *dkeys[2];                   // [n_total] depth-sort ping-pong keys
    uint32_t *dvals[2];                   // [n_total] depth-sort ping-pong values (compact indices)
    flod_dbg_projected *dbg;              // [n_total] (written only with FLOD_OPT_DEBUG)
    uint8_t *mask;                        // [n_total] (written only with FLOD_OPT_DEBUG)
    void *tkeys[2];                       // [max_pairs] tile ids, uint16 when T_n <= 65536 else uint32
    uint32_t *vals[2];                    // [max_pairs] compact index
    uint2 *ranges;                        // [T_n] (start, end) into the sorted pairs
    float *image;                         // [3][H][W] for flod_render_to_host
};

struct FrameParams {
    float R[9], t[3];
    float fx, fy, cx, cy, z_near;
    float limx, limy;                     // 1.3 W / (2 fx), 1.3 H / (2 fy), fp64 -> fp32 once
    float centre[3];                      // -R^T t, fp64 -> fp32 once
    float ref[3];                         // selection reference (R2)
    float bg[3];
    int W, H, TX, TY;
    long long first_gid;                  // gid of the first scanned Gaussian
    int n_scan;
    int n_levels;                         // levels in the range
    int level_end[FLOD_MAX_LEVELS];       // cumulative end (scan index) of each level in the range
    float lo2[FLOD_MAX_LEVELS], hi2[FLOD_MAX_LEVELS];
    unsigned int max_pairs;
    int n_pre_blocks;
    int n_tiles;                          // TX * TY
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
    int sort_blocks_max = 0, pre_blocks_max = 0;
    // options / state
    unsigned flags = 0;
    bool has_ref = false;
    float ref[3] = {0, 0, 0};
    unsigned int epoch = 0;               // bumped once per onesweep pass, tags sort_status words
    cudaStream_t last_stream = nullptr;
    bool rendered = false;
    int last_w = 0, last_h = 0, last_tx = 0, last_ty = 0, last_final_buf = 0;
    int64_t last_n_scan = 0;
    cudaEvent_t ev[FLOD_N_STAGES + 1] = {nullptr};
    bool ev_valid = false;
};

// How the tile ids are sorted: `passes` stable passes of `bits` bits each (passes * bits >= tile_bits).
struct TileSortPlan { int passes, bits; bool wide; };    // wide: uint32 tile keys (T_n > 65536)
TileSortPlan tile_sort_plan(int n_tiles);

// kernel launchers (each enqueues on `s` and returns the number of kernels launched)
int launch_geometry(const Context &c, const FrameParams &p, cudaStream_t s);       // a1-a3 + compaction
int launch_colour(const Context &c, const FrameParams &p, cudaStream_t s);         // a4
int launch_depth_sort(Context &c, int *final_buf, cudaStream_t s);                 // a7, first half
int launch_duplicate(const Context &c, const FrameParams &p, int depth_buf, cudaStream_t s);   // a5-a6
int launch_tile_sort(Context &c, const FrameParams &p, int *final_buf, cudaStream_t s);        // a7, second half
int launch_ranges(const Context &c, const FrameParams &p, int final_buf, cudaStream_t s);      // a8
int launch_blend(const Context &c, const FrameParams &p, int final_buf, float *out_rgb, cudaStream_t s);   // a9

}  // namespace flod
