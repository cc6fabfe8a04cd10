// Internal declarations of libflod (host context, device layouts, kernel launchers).
// Nothing here is shared with oracle/ -- the two implementations are written independently from DESIGN.md §2.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/flod.h"

namespace flod {

constexpr int kTile = FLOD_TILE;
constexpr int kPreBlock = 256;            // preprocess: Gaussians per block
constexpr int kSortThreads = 512;         // onesweep: threads per block
constexpr int kSortItems = 8;             // onesweep: keys per thread
constexpr int kSortTile = kSortThreads * kSortItems;
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kMaxPasses = 8;

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
    unsigned int pre_ticket;              // virtual block ids of the preprocess kernel
    unsigned int sort_ticket[kMaxPasses]; // virtual block ids of each onesweep pass
    unsigned int blend_ticket;
    unsigned int overflow;
    unsigned long long n_sel, n_front, n_vis, n_pairs;   // n_pairs = required pairs
    unsigned long long evals, blends;
    unsigned int n_pairs_clamped;         // min(n_pairs, max_pairs): what sort / ranges / blend iterate over
    unsigned int pad;
    unsigned int hist[kMaxPasses][kRadix];  // global digit histograms of all passes
};

// Blend features of one visible Gaussian (compact index): see DESIGN R25.
//   gA = (mu'x, mu'y, k = B/A, -A log2(e)/2)     gB = (-(C - B^2/A) log2(e)/2, log2 o, r, g)    cB = b
struct WorkspaceDev {
    FrameHeader *hdr;
    unsigned long long *pre_status;       // [pre_blocks_max] decoupled look-back of the fused preprocess scan
    unsigned long long *sort_status;      // [sort_blocks_max][kRadix] epoch-tagged look-back, shared by all passes
    float4 *gA, *gB;                      // [n_total]
    float *cB;                            // [n_total]
    uint32_t *cgid;                       // [n_total] compact index -> gid
    flod_dbg_projected *dbg;              // [n_total] (written only with FLOD_OPT_DEBUG)
    uint8_t *mask;                        // [n_total] (written only with FLOD_OPT_DEBUG)
    unsigned long long *keys[2];          // [max_pairs] (tile << 32) | depth bits
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

// kernel launchers (each enqueues on `s` and returns the number of kernels launched)
int launch_preprocess(const Context &c, const FrameParams &p, cudaStream_t s);
int launch_sort(Context &c, int tile_bits, int *final_buf, cudaStream_t s);
int launch_ranges(const Context &c, int final_buf, cudaStream_t s);
int launch_blend(const Context &c, const FrameParams &p, int final_buf, float *out_rgb, cudaStream_t s);
int sort_passes_for(int tile_bits);

}  // namespace flod
