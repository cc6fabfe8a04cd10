/*
 * flod.h -- C ABI of the B200-native forward rasterizer for multi-level 3D Gaussian sets (FLoD, arXiv 2408.12894).
 *
 * Citations: P:n = PAPER.md line n, S:n = SPEC.md line n, Rk = reading k in DESIGN.md §3.
 *
 * The library renders a multi-level Gaussian set {G^(l)} at a single level, at the maximum level, or selectively
 * (Eq. 6-7): for l in [l_start, l_end] a level-l Gaussian is drawn iff
 *     d_proj^(l) <= |mu - ref| < d_proj^(l-1),   d_proj^(l) = s_min^(l) * fx / gamma,
 *     d_proj^(l_end) = 0,  d_proj^(l_start - 1) = +inf                                   (R1-R4).
 * Selected Gaussians are projected (mu', Sigma' of P:110, +0.3 px^2 dilation, R8-R9), binned to 16x16 tiles by the
 * box of their alpha = 1/255 contour (R13), ordered per tile by (depth, global id) (R15) and composited front
 * to back with alpha = min(0.99, o exp(-1/2 d^T Sigma'^-1 d)) (Eq. 2), skipping alpha < 1/255 and stopping
 * after the blend that takes the transmittance below 1e-4 (R11-R12).
 *
 * Ownership: ALL device memory is allocated and owned by the caller (scene arena, workspace, output image); the
 * library never allocates device memory, never creates streams, and never synchronises inside flod_render.
 * Pointers named *_dev are device pointers, everything else is a host pointer.  All arrays are fp32, C-contiguous.
 * Every function returns 0 (FLOD_OK) or a negative FLOD_E_* code; flod_last_error() gives the message.
 * One context = one scene on one device.  Calls on one context are not thread-safe; contexts are independent.
 * There is no CPU fallback anywhere.
 */
#ifndef FLOD_H
#define FLOD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define FLOD_API __attribute__((visibility("default")))
#else
#define FLOD_API
#endif

#define FLOD_ABI_VERSION 10
#define FLOD_MAX_LEVELS 16
#define FLOD_TILE 16                 /* tiles are 16x16 pixels */
#define FLOD_N_STAGES 5              /* 0 geometry (a1-a3), 1 colour (a4) with the tile scan (a5, a8) in one of its blocks,
                                        2 duplication (a6), 3 per-tile sort (a7), 4 blend (a9) */

enum {
    FLOD_OK = 0,
    FLOD_E_INVALID_ARG = -1,         /* null pointer, gamma <= 0 or non-finite, fx/fy <= 0, width/height < 1, z_near < 0 */
    FLOD_E_LEVEL_RANGE = -2,         /* not first_level <= l_start <= l_end <= last_level */
    FLOD_E_NOT_UPLOADED = -3,        /* render / workspace query before flod_upload_levels */
    FLOD_E_ARENA_TOO_SMALL = -4,     /* scene arena or workspace smaller than flod_*_bytes() says */
    FLOD_E_CAPACITY = -5,            /* previous frame needed more pairs than max_pairs (reported by flod_get_stats) */
    FLOD_E_CUDA = -6,                /* CUDA runtime error; text in flod_last_error */
    FLOD_E_NO_WORKSPACE = -7,        /* flod_render before flod_set_workspace */
    FLOD_E_STATIC_LIMIT = -8         /* flod_overlap_prune_static: n > flod_overlap_prune_static_max_n() */
};

typedef struct flod_ctx flod_ctx;    /* opaque, host side */

/* One level G^(l).  Host pointers, read-only, copied by flod_upload_levels. */
typedef struct {
    int64_t n;                       /* number of Gaussians (may be 0) */
    int     level;                   /* level id l, 1-based; uploaded levels are consecutive and ascending (R23) */
    float   s_min;                   /* Eq. 3 value s_min^(l) for this level; >= 0, strictly decreasing in l */
    const float *mean;               /* [n][3] world units */
    const float *log_scale;          /* [n][3] log of the EFFECTIVE scale s^(l) = exp(s_opt) + s_min (Eq. 4; Alg. 1; R6) */
    const float *quat;               /* [n][4] w,x,y,z; any non-zero norm */
    const float *opacity_logit;      /* [n]; o = sigmoid(logit) */
    const float *sh;                 /* [n][K][3], K = (sh_degree+1)^2, real SH of R16 */
} flod_level_desc;

/* Pinhole camera.  x_cam = R x_world + t; camera axes +x right, +y down, +z forward.
 * Pixel (i,j) covers [i,i+1)x[j,j+1) and is sampled at (i+.5, j+.5) (R14). */
typedef struct {
    float R[9];                      /* row-major */
    float t[3];
    float fx, fy, cx, cy;            /* pixels */
    int   width, height;
    float z_near;                    /* cull z_cam <= z_near; must be >= 0 (R10, R24) */
    float bg[3];                     /* background colour */
} flod_camera;

/* Which levels to render, by level id, inclusive.  Single level l = {l,l}; maximum level = {L,L};
 * selective rendering = {l_start < l_end} (Eq. 6).  gamma is ignored (but validated) when l_start == l_end. */
typedef struct { int l_start, l_end; } flod_level_mode;

typedef struct {
    int64_t n_scan;                  /* Gaussians in levels l_start..l_end */
    int64_t n_sel;                   /* pass Eq. 6 */
    int64_t n_front;                 /* selected with z_cam > z_near */
    int64_t n_vis;                   /* also alive, det > 0, non-empty tile rect */
    int64_t n_pairs;                 /* (Gaussian, tile) pairs the frame REQUIRES (may exceed max_pairs) */
    int64_t max_pairs;               /* capacity given to flod_set_workspace */
    int     overflow;                /* non-zero: out_rgb of that frame is undefined.  bit 0: n_pairs > max_pairs (grow the
                                        workspace); bit 1: one tile's list exceeds 2^24 entries (a larger workspace does not help) */
    int64_t evals, blends;           /* E, B of DESIGN §6 when FLOD_OPT_COUNT is on, else 0 */
    float   ms_stage[FLOD_N_STAGES]; /* device time per stage when FLOD_OPT_PROFILE is on, else 0 */
    float   ms_total;
} flod_stats;

enum {                               /* flod_set_options bits */
    FLOD_OPT_DEBUG   = 1,            /* also write the selection mask and per-Gaussian projection records */
    FLOD_OPT_PROFILE = 2,            /* record CUDA events between stages (flod_get_stats reports ms) */
    FLOD_OPT_COUNT   = 4,            /* instrumented blend kernel counting evaluations and blends */
    FLOD_OPT_SMALL_WINDOWS = 8,      /* test knob: the large-rect duplication kernel serves frames from a mean rect of 128 tiles
                                        (default: 1024) and walks the tiles in windows of 1024 (the path an image of more
                                        than 48 Ki tiles takes) */
    FLOD_OPT_FULL_SORT = 16          /* order every tile list completely.  By default a list of more than 4096 pairs is ordered
                                        only as far as the blend reads it (nearest depth slices first, the rest if pixels of
                                        the tile are still alive): same image bit for bit.  FLOD_OPT_DEBUG and FLOD_OPT_COUNT
                                        imply it; flod_render_backward needs it. */
};

enum {                               /* flod_debug_copy selectors; host_dst sizes in bytes */
    FLOD_DBG_MASK = 0,               /* uint8[n_total]: Eq. 6 membership, zero outside the range (needs FLOD_OPT_DEBUG) */
    FLOD_DBG_TILE_COUNTS = 1,        /* uint32[TX*TY]: pairs per tile */
    FLOD_DBG_PROJECTED = 2,          /* flod_dbg_projected[n_vis] in ascending gid (needs FLOD_OPT_DEBUG) */
    FLOD_DBG_SORTED_PAIRS = 3,       /* flod_dbg_pair[min(n_pairs,max_pairs)] in final order */
    FLOD_DBG_ACTIVATED = 4           /* float[n_total][8]: Sigma xx,xy,xz,yy,yz,zz, o, kappa (kappa = -1 when dead) */
};

typedef struct {
    uint32_t gid; float mu2d[2]; float depth; float conic[3]; float opacity; float rgb[3];
    int32_t rect[4];                 /* tx0, ty0, tx1, ty1 */
} flod_dbg_projected;

typedef struct { uint32_t tile; float depth; uint32_t gid; } flod_dbg_pair;

/* Create / destroy a context bound to CUDA device `device`.  No device memory is allocated. */
FLOD_API int flod_create(flod_ctx **out, int device);
FLOD_API int flod_destroy(flod_ctx *ctx);

/* Bytes of the scene arena needed for these levels (only n and sh_degree are read).  0 on invalid input. */
FLOD_API size_t flod_scene_bytes(int n_levels, const flod_level_desc *levels, int sh_degree);

/* Step a0 (Eq. 1): activate on the host in fp64 (s = exp(log_scale), Sigma = R S S^T R^T,
 * o = sigmoid, kappa = 2 ln(255 o), dead = o < 1/255), lay out as SoA planes and copy into the caller's arena.
 * The copy is enqueued on `stream` and the call returns after it completed; host arrays may then be freed.
 * Validates: consecutive ascending level ids, s_min >= 0 strictly decreasing, finite attributes, |mean| <= 1e15,
 * non-zero quaternions, 0 <= sh_degree <= 3, arena 256-byte aligned and large enough (R22, R23). */
FLOD_API int flod_upload_levels(flod_ctx *ctx, int n_levels, const flod_level_desc *levels, int sh_degree,
                       void *scene_arena_dev, size_t arena_bytes, void *stream);

/* Workspace needed to render images up to width x height with at most max_pairs (Gaussian, tile) pairs
 * (1 <= max_pairs < 2^30; width, height <= 16384).  0 on invalid input or before upload. */
FLOD_API size_t flod_workspace_bytes(const flod_ctx *ctx, int width, int height, int64_t max_pairs);

/* Hand the workspace to the context (256-byte aligned device pointer).  width/height/max_pairs are the same
 * values given to flod_workspace_bytes; flod_render rejects larger cameras. */
FLOD_API int flod_set_workspace(flod_ctx *ctx, void *workspace_dev, size_t bytes, int width, int height, int64_t max_pairs);

/* R2: position d_G is measured from.  NULL (default) = the camera centre of each frame;
 * a fixed position reproduces the paper's "average training camera" or "position at the last
 * rebuild" policies. */
FLOD_API int flod_set_selection_reference(flod_ctx *ctx, const float ref_pos[3]);

FLOD_API int flod_set_options(flod_ctx *ctx, unsigned flags);

/* Which tiles a visible Gaussian is listed in (R13, R26).  Both rules are conservative -- every pixel with
 * alpha >= 1/255 lies in a listed tile -- so the image is the same; per-tile pair counts, n_pairs and
 * the sorted pair sequence are those of the chosen rule.
 *   FLOD_PAIR_RULE_BOX      (default) every tile of the rect (the padded box of the alpha = 1/255 contour);
 *   FLOD_PAIR_RULE_ELLIPSE  the tiles of the rect that hold a pixel centre of the padded alpha = 1/255 ellipse of Eq. 2
 *                           (P:104-108): one span of tiles per tile row, canonical fp32 on the factorised exponent.
 *                           22-32 % fewer pairs; finding them costs about what they save on fine levels (config 1:
 *                           -2 % frames/s) and pays on coarse ones (config 3, levels 2-5: +2 .. +10 %). */
enum { FLOD_PAIR_RULE_BOX = 1, FLOD_PAIR_RULE_ELLIPSE = 2 };
FLOD_API int flod_set_pair_rule(flod_ctx *ctx, int rule);

/* Steps a1-a9 for one frame, asynchronous on `stream` (a cudaStream_t passed as void*).
 * out_rgb_dev: [3][height][width] planar fp32.  Errors detected on the host are returned here; a capacity
 * overflow is detected on the device: the frame is not silently truncated -- out_rgb is undefined, and
 * flod_get_stats reports the overflow bits and the required n_pairs so the caller can grow the workspace.
 * cam->R must be a rotation (max |R R^T - I| <= 1e-4), else FLOD_E_INVALID_ARG. */
FLOD_API int flod_render(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma,
                float *out_rgb_dev, void *stream);

/* One horizontal STRIP of a frame: the tile rows [ty_begin, ty_end) (0 <= ty_begin <= ty_end <= ceil(height / 16)), i.e. the
 * image rows [16 ty_begin, min(height, 16 ty_end)), written to out_strip_dev as [3][rows][width] planar fp32.  The unit of
 * screen-space sharding over GPUs: each rank culls the Gaussians to its strip (rects are clipped to
 * it), lists, orders and blends only its own tiles; the strips of all ranks, stacked, are the image flod_render writes,
 * bit for bit (a tile's list, its order and its arithmetic do not depend on the other tiles).  flod_get_stats then
 * counts what the strip needed (n_vis, n_pairs of the strip). */
FLOD_API int flod_render_rows(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma,
                     int ty_begin, int ty_end, float *out_strip_dev, void *stream);

/* Same, end to end with HOST buffers: renders into an image of the workspace and copies it to out_rgb_host
 * ([3][height][width] fp32, ideally pinned) on `stream`, then waits for the copy.  The frame's overflow word travels
 * with the image: FLOD_E_CAPACITY is returned (and the image is undefined) when the frame overflowed. */
FLOD_API int flod_render_to_host(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma,
                        float *out_rgb_host, void *stream);

/* Pipelined form of flod_render_to_host for frame sequences.  The kernels run on `stream`, the device-to-host copy
 * on `copy_stream` (both caller-owned cudaStream_t; pass two different streams to overlap the copy of frame k with
 * the kernels of frame k+1 -- the workspace holds two images and the library orders the two streams with its own
 * events).  Returns without waiting: out_rgb_host (pinned) must stay valid and must not be read before
 * flod_wait_host returns; give consecutive frames different host buffers if every frame is to be kept. */
FLOD_API int flod_render_to_host_async(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma,
                              float *out_rgb_host, void *stream, void *copy_stream);

/* Blocks the calling host thread until every copy issued by flod_render_to_host_async has landed.  Returns
 * FLOD_E_CAPACITY if one of the frames waited for overflowed (its image is undefined). */
FLOD_API int flod_wait_host(flod_ctx *ctx);

/* ---- Materialised G_sel (Eq. 6) reused over a run of frames and rebuilt in the background, the paper's
 * runtime for long trajectories: "G_sel ... is updated every 50 views" on a second thread.  A SNAPSHOT
 * is the stable (gid-order) compaction of the Gaussians of the level range that pass Eq. 6 for ONE reference
 * position (R2's "position at the last rebuild"; P:681's average training camera is the same call with that
 * position).  The subset arena holds two snapshots: frames are rendered from the FRONT one while the BACK one is
 * rebuilt on another stream; flod_subset_swap exchanges them between two frames.  A frame rendered from a snapshot
 * equals flod_render with flod_set_selection_reference(ref_pos) and the same fx and gamma, bit for bit. ---- */

/* Bytes of a subset arena for the level range `mode` (two snapshots, each sized for every Gaussian of the range:
 * 92 B per Gaussian and snapshot; SH rows stay in the scene arena).  0 on invalid input or before upload. */
FLOD_API size_t flod_subset_bytes(const flod_ctx *ctx, flod_level_mode mode);

/* Hand the subset arena (256-byte aligned device pointer, caller-owned) to the context and fix the level range. */
FLOD_API int flod_subset_set_arena(flod_ctx *ctx, void *arena_dev, size_t bytes, flod_level_mode mode);

/* Enqueue on `stream` the rebuild of the BACK snapshot: Eq. 6-7 with d_G = |mu - ref_pos| (fp32, as O1), thresholds
 * d_proj^(l) = s_min^(l) fx / gamma computed in fp64 and rounded once; selected Gaussians are copied in gid order.
 * Returns without waiting; `stream` may differ from the render stream (the library orders the rebuild after the last
 * frame that read the back snapshot).  FLOD_E_INVALID_ARG for a non-finite position, fx <= 0 or gamma <= 0. */
FLOD_API int flod_subset_build(flod_ctx *ctx, const float ref_pos[3], float fx, float gamma, void *stream);

/* 1 if the enqueued rebuild has completed (flod_subset_swap would not block), 0 if not, negative on error. */
FLOD_API int flod_subset_ready(flod_ctx *ctx);

/* Waits (host) for the rebuild, then makes the back snapshot the front one.  *n_selected (may be NULL) receives its
 * size N_sel.  FLOD_E_INVALID_ARG if no rebuild was enqueued since the last swap. */
FLOD_API int flod_subset_swap(flod_ctx *ctx, int64_t *n_selected);

/* flod_render from the FRONT snapshot: steps a2-a9 over its N_sel Gaussians (a1 was done by the rebuild).  The
 * camera's fx should be the one the snapshot was built with (Eq. 7); this is not checked. */
FLOD_API int flod_render_subset(flod_ctx *ctx, const flod_camera *cam, float *out_rgb_dev, void *stream);

/* Waits for the last frame's stream, then reports its counters (and FLOD_E_CAPACITY if it overflowed). */
FLOD_API int flod_get_stats(flod_ctx *ctx, flod_stats *out);

/* Copies an intermediate of the LAST rendered frame to host memory (synchronous).  `bytes` must be at least the
 * size implied by the selector; see the FLOD_DBG_* comments. */
FLOD_API int flod_debug_copy(flod_ctx *ctx, int what, void *host_dst, size_t bytes);

/* Number of kernel launches the last flod_render enqueued (5 to 8: one more after frames of large rects, two more after
 * frames of long lists; 6 before the first frame). */
FLOD_API int flod_launches_per_frame(const flod_ctx *ctx);

/* ---- Training-side kernels.  They need no context: all arrays are caller-owned device memory. ---- */

/* Backward pass of the rasterizer (Alg. 1 "Adam(grad L)"): the gradient of <dL_dimage, image> with
 * respect to every learnable parameter of the LAST frame rendered by flod_render on this context (its lists are still in
 * the workspace; cam must be that frame's camera, else FLOD_E_INVALID_ARG).  All arrays are device memory indexed by gid
 * (levels concatenated in upload order) over the whole scene; the call zeroes them and the Gaussians the frame drew add
 * their gradients: d_mean [n][3], d_log_scale [n][3] (of the stored log of the effective scale; d s / d s_opt =
 * exp(s_opt) of Eq. 4 is the caller's chain), d_quat [n][4] (of the un-normalised quaternion), d_opacity_logit [n],
 * d_sh [n][K][3].  The discrete decisions of the forward pass (selection, culls, order, the 1/255 skip, the stop at
 * T < 1e-4) are constants; min(0.99, .) and max(0, .) have their mathematical derivative.  fp32, sums in the order the
 * atomics are served (not bit-reproducible); asynchronous on `stream`.  workspace_dev: flod_backward_workspace_bytes,
 * 256-byte aligned, caller-owned. */
typedef struct { float *d_mean, *d_log_scale, *d_quat, *d_opacity_logit, *d_sh; } flod_grads;
FLOD_API size_t flod_backward_workspace_bytes(const flod_ctx *ctx);
FLOD_API int flod_render_backward(flod_ctx *ctx, const flod_camera *cam, const float *dL_dimage_dev, const flod_grads *grads,
                         void *workspace_dev, size_t workspace_bytes, void *stream);

/* Overlap pruning (§4.3; Alg. 1 "OverlapPruning()"): remove_dev[i] = 1 iff the average distance from
 * Gaussian i to its three nearest neighbours (by mean, Euclidean; k = n - 1 when n <= 3, nothing when n <= 1) is below
 * d_OP = s_min / 2, all decided on the set as given (simultaneous rule).  mean_dev is [n][3] fp32.
 * mean_dist_dev (may be NULL) receives that average where it is decided exactly -- whenever the third neighbour lies
 * within 3 d_OP -- and +inf otherwise (then it is >= d_OP, which is all the rule needs).  bbox_lo: any point with
 * bbox_lo <= mean componentwise (the grid's origin; the minimum of the means, or a bound of the scene).
 * Arithmetic (both sides of the parity test): d^2 = (dx dx + dy dy) + dz dz, mean = ((sqrt d1 + sqrt d2) + sqrt d3) / 3
 * with d1 <= d2 <= d3, compared with 0.5f * s_min, every operation one IEEE binary32 operation.
 * s_min must be > 0 (the rule is for levels below L_max).  Asynchronous on `stream`. */
FLOD_API size_t flod_overlap_prune_workspace_bytes(int64_t n);
FLOD_API int flod_overlap_prune(const float *mean_dev, int64_t n, float s_min, const float bbox_lo[3], unsigned char *remove_dev,
                       float *mean_dist_dev, void *workspace_dev, size_t workspace_bytes, void *stream);

/* The same operation for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): no workspace argument.  The scratch is a file-scope device array inside the library
 * (8.0 MiB, held by every GPU that loads libflod.so until the process exits), which bounds the size:
 * n <= flod_overlap_prune_static_max_n() = 262 144, else FLOD_E_STATIC_LIMIT (use flod_overlap_prune with a workspace).
 * Same arguments, arithmetic and results as flod_overlap_prune; mean_dev, remove_dev, mean_dist_dev stay the caller's.
 * The call runs no cudaMalloc / cudaFree and no allocating library routine: one cudaMemsetAsync (the bucket counters must
 * start at zero; the rest of the array keeps the last call's contents and is overwritten before it is read) and four
 * kernel launches on `stream`.  EVERY call on a device shares the one array: calls that overlap on the GPU (different
 * streams without an ordering between them, or two host threads) race; calls on one stream are ordered and safe.
 * The array's device address is asked from the runtime once per device, on the first call with that device current;
 * flod_overlap_prune_static_setup() does just that ahead of time (call it, with the device current, before a stream
 * capture begins).  Devices 0..63. */
FLOD_API int64_t flod_overlap_prune_static_max_n(void);
FLOD_API int flod_overlap_prune_static_setup(void);
FLOD_API int flod_overlap_prune_static(const float *mean_dev, int64_t n, float s_min, const float bbox_lo[3],
                                       unsigned char *remove_dev, float *mean_dist_dev, void *stream);

FLOD_API const char *flod_last_error(const flod_ctx *ctx);
FLOD_API int flod_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* FLOD_H */
