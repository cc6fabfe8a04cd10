// Host side of libflod: the C ABI of include/flod.h.  Argument checking, step a0 (upload + activation),
// workspace carving, per-frame constants and kernel sequencing.  No device allocation, no stream creation,
// no synchronisation inside flod_render.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <thread>
#include <vector>

#include "flod_internal.cuh"

using namespace flod;

struct flod_ctx : public flod::Context {};

namespace {

int fail(const flod_ctx *c, int code, const std::string &msg)
{
    if (c) const_cast<flod_ctx *>(c)->err = msg;
    return code;
}

#define CUDA_TRY(ctx, expr)                                                                         \
    do {                                                                                            \
        cudaError_t e__ = (expr);                                                                   \
        if (e__ != cudaSuccess)                                                                     \
            return fail(ctx, FLOD_E_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e__));     \
    } while (0)

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// FrameHeader.overflow: bit 0 = the frame needs more pairs than max_pairs, bit 1 = one tile's list exceeds 2^24 entries
const char *overflow_text(unsigned int bits)
{
    if (bits & 1u) return "frame needed more pairs than max_pairs (image undefined); grow the workspace to the reported n_pairs and re-render";
    return "one tile's list holds more than 2^24 entries (image undefined); a larger workspace does not help: render fewer levels or a larger image";
}

int sh_stride_for(int deg) { int k = (deg + 1) * (deg + 1); return (3 * k + 3) / 4 * 4; }

constexpr int kScenePlanes = 3 + 6 + 4 + 8;   // mean xyz, cov x6, opacity, kappa, log2 o, rho2; raw log_scale xyz, quat wxyz, logit

size_t scene_bytes_for(int64_t n, int sh_degree)
{
    size_t per_plane = align_up((size_t)std::max<int64_t>(n, 1) * sizeof(float));
    return per_plane * kScenePlanes + align_up((size_t)std::max<int64_t>(n, 1) * 8 * sizeof(float)) +
           align_up((size_t)std::max<int64_t>(n, 1) * sh_stride_for(sh_degree) * sizeof(float));
}

// Step a0 for one Gaussian (DESIGN §2 "O0"; Eq. 1).  fp64 from the fp32 inputs, rounded once.
void activate_one(const float *ls, const float *q, float logit, float cov[6], float *o_out, float *kappa, float *l2o,
                  float *rho2)
{
    const double s0 = exp((double)ls[0]), s1 = exp((double)ls[1]), s2 = exp((double)ls[2]);
    double w = q[0], x = q[1], y = q[2], z = q[3];
    const double nrm = sqrt(((w * w + x * x) + y * y) + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    const double r[3][3] = {
        {1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z), 2.0 * (x * z + w * y)},
        {2.0 * (x * y + w * z), 1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x)},
        {2.0 * (x * z - w * y), 2.0 * (y * z + w * x), 1.0 - 2.0 * (x * x + y * y)}};
    const double v0 = s0 * s0, v1 = s1 * s1, v2 = s2 * s2;
    int k = 0;
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j)
            cov[k++] = (float)((r[i][0] * v0 * r[j][0] + r[i][1] * v1 * r[j][1]) + r[i][2] * v2 * r[j][2]);
    const float o = (float)(1.0 / (1.0 + exp(-(double)logit)));
    const bool dead = o < (float)(1.0 / 255.0);
    *o_out = o;
    *kappa = dead ? -1.0f : (float)(2.0 * log(255.0 * (double)o));
    *l2o = dead ? -126.0f : (float)log2((double)o);
    // squared radius of the sphere around the mean that holds the alpha = 1/255 ellipsoid, rounded up; k_geometry's
    // conservative off-screen test uses it before any covariance is read.  -1 marks a dead Gaussian.
    const double r2 = 2.0 * log(255.0 * (double)o) * std::max(v0, std::max(v1, v2)) * (1.0 + 1e-4);
    *rho2 = dead ? -1.0f : (r2 < 3.0e38 ? nextafterf((float)r2, INFINITY) : INFINITY);
}

bool finite_all(const float *p, size_t n)
{
    for (size_t i = 0; i < n; ++i)
        if (!isfinite(p[i])) return false;
    return true;
}

template <class F>
void parallel_for(int64_t n, F f)
{
    unsigned hw = std::max(1u, std::min(std::thread::hardware_concurrency(), 32u));
    if (n < 4096 || hw == 1) { f(0, n); return; }
    std::vector<std::thread> th;
    int64_t chunk = (n + hw - 1) / hw;
    for (unsigned t = 0; t < hw; ++t) {
        int64_t b = t * chunk, e = std::min<int64_t>(n, b + chunk);
        if (b >= e) break;
        th.emplace_back([=] { f(b, e); });
    }
    for (auto &t : th) t.join();
}

struct WsLayout { WorkspaceDev ws; size_t bytes; };

// Carve the workspace.  [header | tile difference grid] come first and are zeroed together every frame.
WsLayout carve(unsigned char *base, int64_t n_total, int w, int h, int64_t max_pairs)
{
    WsLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return (unsigned char *)((uintptr_t)base + o); };
    const size_t tx = (size_t)(w + kTile - 1) / kTile, ty = (size_t)(h + kTile - 1) / kTile;
    const size_t tiles = tx * ty;
    const size_t nt = (size_t)std::max<int64_t>(n_total, 1) + 2 * kGeoBlock;   // segment positions (see WorkspaceDev)
    L.ws.hdr2[0] = (FrameHeader *)take(sizeof(FrameHeader));
    L.ws.hdr2[1] = (FrameHeader *)take(sizeof(FrameHeader));
    L.ws.hdr = L.ws.hdr2[0]; L.ws.hdr_next = L.ws.hdr2[1];
    L.ws.tile_diff = (int *)take((tx + 1) * (ty + 1) * kCtrStride * sizeof(int));
    L.ws.seg_count = (unsigned int *)take((nt / kGeoBlock + 2) * sizeof(unsigned int));
    L.ws.tile_cnt = (int *)take((tx + 1) * (ty + 1) * sizeof(int));
    L.ws.ranges = (uint2 *)take(tiles * sizeof(uint2));
    L.ws.cursor4 = (float *)take(((tx + 1) / 2) * ((ty + 1) / 2) * kCtrStride * sizeof(float));
    L.ws.cursor = (unsigned int *)take(tiles * sizeof(unsigned int));
    L.ws.cnt4 = (float *)take(((tx + 1) / 2) * ((ty + 1) / 2) * kCtrStride * sizeof(float));
    L.ws.gA = (float4 *)take(nt * sizeof(float4));
    L.ws.gB = (float4 *)take(nt * sizeof(float4));
    L.ws.cB = (float *)take(nt * sizeof(float));
    L.ws.dirgid = (float4 *)take(nt * sizeof(float4));
    L.ws.rect = (ushort4 *)take(nt * sizeof(ushort4));
    L.ws.depth = (uint32_t *)take(nt * sizeof(uint32_t));
    L.ws.dbg = (flod_dbg_projected *)take(nt * sizeof(flod_dbg_projected));
    L.ws.mask = (uint8_t *)take(nt);
    L.ws.pairs = (unsigned long long *)take((size_t)max_pairs * 8);
    L.ws.pairs_tmp = (unsigned long long *)take((size_t)max_pairs * 8);
    L.ws.vals = (uint32_t *)take((size_t)max_pairs * 4);
    L.ws.ovf_slots = (unsigned int *)take(4 * sizeof(unsigned int));
    L.ws.ovf_out = L.ws.ovf_slots + 2;
    L.ws.lazy = (uint4 *)take(tiles * sizeof(uint4));
    L.ws.slice_ends = (unsigned int *)take(tiles * kCoarseBins * sizeof(unsigned int));
    L.ws.hint_state = (unsigned int *)take(sizeof(unsigned int));
    L.ws.todo = (unsigned int *)take(tiles * sizeof(unsigned int));
    L.ws.tile_state = (float4 *)take(tiles * 256 * sizeof(float4));
    L.ws.image[0] = (float *)take((size_t)3 * w * h * sizeof(float));
    L.ws.image[1] = (float *)take((size_t)3 * w * h * sizeof(float));
    L.bytes = off;
    return L;
}

}  // namespace

extern "C" {

int flod_abi_version(void) { return FLOD_ABI_VERSION; }

const char *flod_last_error(const flod_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int flod_create(flod_ctx **out, int device)
{
    if (!out) return FLOD_E_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || device < 0 || device >= count) return FLOD_E_CUDA;
    flod_ctx *c = new flod_ctx();
    c->device = device;
    // the shared-memory opt-ins are per-device function attributes: set them for THIS device, every time
    if (cudaSetDevice(device) != cudaSuccess ||
        cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        init_duplicate() != 0 || init_tile_sort() != 0) {
        delete c;
        return FLOD_E_CUDA;
    }
    bool ok = true;
    for (auto &ev : c->ev) ok &= cudaEventCreate(&ev) == cudaSuccess;
    ok &= cudaEventCreateWithFlags(&c->ev_sub_built, cudaEventDisableTiming) == cudaSuccess;
    for (auto &ev : c->ev_sub_read) ok &= cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 2; ++i) {
        ok &= cudaEventCreateWithFlags(&c->ev_rendered[i], cudaEventDisableTiming) == cudaSuccess;
        ok &= cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming) == cudaSuccess;
    }
    // pinned words the device reports into: [0] N_sel of a rebuild, [1], [2] overflow flag of the frame in image[0], image[1]
    ok &= cudaHostAlloc((void **)&c->sub_n_host, 64, cudaHostAllocMapped) == cudaSuccess;
    if (!ok) { flod_destroy(c); return FLOD_E_CUDA; }      // releases whatever was created
    memset(c->sub_n_host, 0, 64);
    *out = c;
    return FLOD_OK;
}

int flod_destroy(flod_ctx *ctx)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    for (auto &ev : ctx->ev) if (ev) cudaEventDestroy(ev);
    if (ctx->ev_sub_built) cudaEventDestroy(ctx->ev_sub_built);
    for (auto &ev : ctx->ev_sub_read) if (ev) cudaEventDestroy(ev);
    if (ctx->sub_n_host) cudaFreeHost(ctx->sub_n_host);
    for (int i = 0; i < 2; ++i) {
        if (ctx->ev_rendered[i]) cudaEventDestroy(ctx->ev_rendered[i]);
        if (ctx->ev_copied[i]) cudaEventDestroy(ctx->ev_copied[i]);
    }
    delete ctx;
    return FLOD_OK;
}

size_t flod_scene_bytes(int n_levels, const flod_level_desc *levels, int sh_degree)
{
    if (n_levels < 1 || n_levels > FLOD_MAX_LEVELS || !levels || sh_degree < 0 || sh_degree > 3) return 0;
    int64_t n = 0;
    for (int l = 0; l < n_levels; ++l) { if (levels[l].n < 0) return 0; n += levels[l].n; }
    return scene_bytes_for(n, sh_degree);
}

int flod_upload_levels(flod_ctx *ctx, int n_levels, const flod_level_desc *levels, int sh_degree,
                       void *scene_arena_dev, size_t arena_bytes, void *stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (n_levels < 1 || n_levels > FLOD_MAX_LEVELS || !levels || sh_degree < 0 || sh_degree > 3 || !scene_arena_dev)
        return fail(ctx, FLOD_E_INVALID_ARG, "upload: bad n_levels / sh_degree / null pointer");
    if ((uintptr_t)scene_arena_dev % 256) return fail(ctx, FLOD_E_INVALID_ARG, "upload: arena must be 256-byte aligned");
    int64_t n = 0;
    const int K = (sh_degree + 1) * (sh_degree + 1);
    for (int l = 0; l < n_levels; ++l) {
        const flod_level_desc &d = levels[l];
        if (d.n < 0) return fail(ctx, FLOD_E_INVALID_ARG, "upload: negative count");
        if (d.n > 0 && (!d.mean || !d.log_scale || !d.quat || !d.opacity_logit || !d.sh))
            return fail(ctx, FLOD_E_INVALID_ARG, "upload: null attribute array");
        if (l > 0 && d.level != levels[l - 1].level + 1)
            return fail(ctx, FLOD_E_INVALID_ARG, "upload: level ids must be consecutive and ascending");
        if (d.level < 1) return fail(ctx, FLOD_E_INVALID_ARG, "upload: level ids are 1-based");
        if (!(d.s_min >= 0.0f) || !isfinite(d.s_min)) return fail(ctx, FLOD_E_INVALID_ARG, "upload: s_min must be >= 0");
        if (l > 0 && !(d.s_min < levels[l - 1].s_min))
            return fail(ctx, FLOD_E_INVALID_ARG, "upload: s_min must strictly decrease with the level (Eq. 3)");
        n += d.n;
    }
    if (n >= (1ll << 26)) return fail(ctx, FLOD_E_INVALID_ARG, "upload: at most 2^26 - 1 Gaussians per scene");
    if (arena_bytes < scene_bytes_for(n, sh_degree)) return fail(ctx, FLOD_E_ARENA_TOO_SMALL, "upload: arena too small");

    // validate values
    for (int l = 0; l < n_levels; ++l) {
        const flod_level_desc &d = levels[l];
        const size_t m = (size_t)d.n;
        if (!m) continue;
        if (!finite_all(d.mean, 3 * m) || !finite_all(d.log_scale, 3 * m) || !finite_all(d.quat, 4 * m) ||
            !finite_all(d.opacity_logit, m) || !finite_all(d.sh, 3 * (size_t)K * m))
            return fail(ctx, FLOD_E_INVALID_ARG, "upload: non-finite attribute");
        for (size_t i = 0; i < 3 * m; ++i)
            if (fabsf(d.mean[i]) > 1e15f) return fail(ctx, FLOD_E_INVALID_ARG, "upload: |mean| > 1e15");
        for (size_t i = 0; i < m; ++i) {
            const float *q = d.quat + 4 * i;
            if (q[0] == 0.0f && q[1] == 0.0f && q[2] == 0.0f && q[3] == 0.0f)
                return fail(ctx, FLOD_E_INVALID_ARG, "upload: zero quaternion");
        }
    }

    // activate into a host staging image of the arena, then one copy
    const size_t nn = (size_t)std::max<int64_t>(n, 1);
    const size_t plane = align_up(nn * sizeof(float));
    const int stride = sh_stride_for(sh_degree);
    const size_t total = scene_bytes_for(n, sh_degree);
    std::vector<unsigned char> stage(total, 0);
    float *pl[kScenePlanes];
    for (int i = 0; i < kScenePlanes; ++i) pl[i] = (float *)(stage.data() + plane * i);
    float *recp = (float *)(stage.data() + plane * kScenePlanes);
    float *shp = recp + align_up(nn * 8 * sizeof(float)) / sizeof(float);
    int64_t base = 0;
    for (int l = 0; l < n_levels; ++l) {
        const flod_level_desc d = levels[l];
        parallel_for(d.n, [&, d, base](int64_t b, int64_t e) {
            for (int64_t i = b; i < e; ++i) {
                const int64_t g = base + i;
                pl[0][g] = d.mean[3 * i]; pl[1][g] = d.mean[3 * i + 1]; pl[2][g] = d.mean[3 * i + 2];
                float cov[6], o, kap, l2o, rho2;
                activate_one(d.log_scale + 3 * i, d.quat + 4 * i, d.opacity_logit[i], cov, &o, &kap, &l2o, &rho2);
                for (int k = 0; k < 6; ++k) pl[3 + k][g] = cov[k];
                pl[9][g] = o; pl[10][g] = kap; pl[11][g] = l2o; pl[12][g] = rho2;
                for (int k = 0; k < 6; ++k) recp[8 * g + k] = cov[k];
                recp[8 * g + 6] = kap; recp[8 * g + 7] = l2o;
                for (int k = 0; k < 3; ++k) pl[13 + k][g] = d.log_scale[3 * i + k];
                for (int k = 0; k < 4; ++k) pl[16 + k][g] = d.quat[4 * i + k];
                pl[20][g] = d.opacity_logit[i];
                float *dst = shp + (size_t)g * stride;
                const float *src = d.sh + (size_t)i * 3 * K;
                if (sh_degree == 3) {
                    // 4-lane row layout of k_colour: lane j owns coefficients 4j..4j+3 = source floats [12j, 12j+12);
                    // its floats [4i, 4i+4) are float4 number 4i + j of the row
                    for (int f = 0; f < 48; ++f) {
                        const int j = f / 12, within = f % 12;
                        dst[((within / 4) * 4 + j) * 4 + (within % 4)] = src[f];
                    }
                } else {
                    memcpy(dst, src, sizeof(float) * 3 * K);
                }
            }
        });
        base += d.n;
    }
    cudaStream_t s = (cudaStream_t)stream;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaMemcpyAsync(scene_arena_dev, stage.data(), total, cudaMemcpyHostToDevice, s));
    CUDA_TRY(ctx, cudaStreamSynchronize(s));

    ctx->n_levels = n_levels; ctx->first_level = levels[0].level; ctx->sh_degree = sh_degree; ctx->n_total = n;
    ctx->level_off[0] = 0;
    for (int l = 0; l < n_levels; ++l) { ctx->level_off[l + 1] = ctx->level_off[l] + levels[l].n; ctx->s_min[l] = levels[l].s_min; }
    const float *dev = (const float *)scene_arena_dev;
    auto P = [&](int i) { return (const float *)((const unsigned char *)dev + plane * i); };
    ctx->scene.mx = P(0); ctx->scene.my = P(1); ctx->scene.mz = P(2);
    for (int k = 0; k < 6; ++k) ctx->scene.cov[k] = P(3 + k);
    ctx->scene.opacity = P(9); ctx->scene.kappa = P(10); ctx->scene.l2o = P(11); ctx->scene.rho2 = P(12);
    for (int k = 0; k < 8; ++k) ctx->scene.raw[k] = P(13 + k);
    ctx->scene.rec = (const float4 *)P(kScenePlanes);
    ctx->scene.sh = (const float *)((const unsigned char *)P(kScenePlanes) + align_up(nn * 8 * sizeof(float)));
    ctx->scene.sh_stride = stride; ctx->scene.sh_degree = sh_degree;
    ctx->arena = scene_arena_dev;
    ctx->uploaded = true; ctx->has_ws = false; ctx->rendered = false; ctx->has_subset = false;
    return FLOD_OK;
}

size_t flod_workspace_bytes(const flod_ctx *ctx, int width, int height, int64_t max_pairs)
{
    if (!ctx || !ctx->uploaded || width < 1 || height < 1 || width > 16384 || height > 16384 || max_pairs < 1 ||
        max_pairs >= (1ll << 30))
        return 0;
    return carve(nullptr, ctx->n_total, width, height, max_pairs).bytes;
}

int flod_set_workspace(flod_ctx *ctx, void *workspace_dev, size_t bytes, int width, int height, int64_t max_pairs)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ctx->uploaded) return fail(ctx, FLOD_E_NOT_UPLOADED, "set_workspace: no scene uploaded");
    size_t need = flod_workspace_bytes(ctx, width, height, max_pairs);
    if (!need || !workspace_dev || (uintptr_t)workspace_dev % 256)
        return fail(ctx, FLOD_E_INVALID_ARG, "set_workspace: bad size / null or unaligned pointer / max_pairs out of [1, 2^30)");
    if (bytes < need) return fail(ctx, FLOD_E_ARENA_TOO_SMALL, "set_workspace: workspace too small");
    WsLayout L = carve((unsigned char *)workspace_dev, ctx->n_total, width, height, max_pairs);
    ctx->ws = L.ws;
    ctx->ws_w = width; ctx->ws_h = height; ctx->max_pairs = max_pairs;
    for (int i = 0; i < 2; ++i)
        if (ctx->copy_pending[i]) { cudaEventSynchronize(ctx->ev_copied[i]); ctx->copy_pending[i] = false; }
    ctx->img_turn = 0;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaMemset(ctx->ws.hint_state, 0, sizeof(unsigned int)));     // no hint yet about this workspace's frames
    // both frame headers and the difference grid start at zero; from then on the frames keep them so (FrameHeader's comment)
    CUDA_TRY(ctx, cudaMemset(ctx->ws.hdr2[0], 0, sizeof(FrameHeader)));
    CUDA_TRY(ctx, cudaMemset(ctx->ws.hdr2[1], 0, sizeof(FrameHeader)));
    {
        const size_t tx = (size_t)(width + kTile - 1) / kTile, ty = (size_t)(height + kTile - 1) / kTile;
        CUDA_TRY(ctx, cudaMemset(ctx->ws.tile_diff, 0, (tx + 1) * (ty + 1) * kCtrStride * sizeof(int)));
        CUDA_TRY(ctx, cudaMemset(ctx->ws.cnt4, 0, ((tx + 1) / 2) * ((ty + 1) / 2) * kCtrStride * sizeof(float)));
    }
    ctx->hdr_turn = 1;
    ctx->sub_n_host[3] = 0;
    ctx->has_ws = true; ctx->rendered = false;
    return FLOD_OK;
}

int flod_set_selection_reference(flod_ctx *ctx, const float ref_pos[3])
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ref_pos) { ctx->has_ref = false; return FLOD_OK; }
    for (int i = 0; i < 3; ++i)
        if (!isfinite(ref_pos[i]) || fabsf(ref_pos[i]) > 1e15f) return fail(ctx, FLOD_E_INVALID_ARG, "reference must be finite, |x| <= 1e15");
    ctx->has_ref = true;
    memcpy(ctx->ref, ref_pos, sizeof(float) * 3);
    return FLOD_OK;
}

int flod_set_options(flod_ctx *ctx, unsigned flags)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    ctx->flags = flags;
    return FLOD_OK;
}

int flod_set_pair_rule(flod_ctx *ctx, int rule)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (rule != FLOD_PAIR_RULE_BOX && rule != FLOD_PAIR_RULE_ELLIPSE) return fail(ctx, FLOD_E_INVALID_ARG, "pair rule is 1 (box) or 2 (ellipse)");
    ctx->pair_rule = rule;
    return FLOD_OK;
}

int flod_launches_per_frame(const flod_ctx *ctx)
{
    if (!ctx || !ctx->has_ws) return 0;
    // geometry, colour (+ tile scan in its block 0), duplication (one kernel; two, one of which exits, on frames that follow
    // a frame of large rects), tile sort, blend; with blend-driven ordering (frames that follow a frame with long lists)
    // also the second round of the last two
    if (!ctx->rendered) return 6;
    return 5 + (ctx->last_params.dup_both ? 1 : 0) + (ctx->last_params.lazy_sort ? 2 : 0);
}

}  // extern "C"

namespace {

// host-side checks shared by flod_render and flod_render_subset
int check_frame_args(flod_ctx *ctx, const flod_camera *cam, const float *out_rgb_dev)
{
    if (!cam || !out_rgb_dev) return fail(ctx, FLOD_E_INVALID_ARG, "render: null pointer");
    if (!ctx->uploaded) return fail(ctx, FLOD_E_NOT_UPLOADED, "render: no scene uploaded");
    if (!ctx->has_ws) return fail(ctx, FLOD_E_NO_WORKSPACE, "render: no workspace set");
    if (!(cam->fx > 0.0f) || !(cam->fy > 0.0f) || !isfinite(cam->fx) || !isfinite(cam->fy) || cam->width < 1 || cam->height < 1)
        return fail(ctx, FLOD_E_INVALID_ARG, "render: fx, fy must be > 0 and width, height >= 1");
    if (!(cam->z_near >= 0.0f) || !isfinite(cam->z_near)) return fail(ctx, FLOD_E_INVALID_ARG, "render: z_near must be >= 0");
    if (cam->width > ctx->ws_w || cam->height > ctx->ws_h)
        return fail(ctx, FLOD_E_INVALID_ARG, "render: camera larger than the workspace was sized for");
    for (int i = 0; i < 9; ++i) if (!isfinite(cam->R[i])) return fail(ctx, FLOD_E_INVALID_ARG, "render: non-finite R");
    // R must be a rotation: k_geometry's covariance-free off-screen bound |row of J R|^2 <= pre_c1 / z^2 and the
    // meaning of depth both rest on it
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) {
            double d = 0.0;
            for (int k = 0; k < 3; ++k) d += (double)cam->R[3 * i + k] * (double)cam->R[3 * j + k];
            if (fabs(d - (i == j ? 1.0 : 0.0)) > 1e-4)
                return fail(ctx, FLOD_E_INVALID_ARG, "render: R is not orthonormal (max |R R^T - I| > 1e-4)");
        }
    for (int i = 0; i < 3; ++i) if (!isfinite(cam->t[i]) || !isfinite(cam->bg[i])) return fail(ctx, FLOD_E_INVALID_ARG, "render: non-finite t / bg");
    if (!isfinite(cam->cx) || !isfinite(cam->cy)) return fail(ctx, FLOD_E_INVALID_ARG, "render: non-finite principal point");
    return FLOD_OK;
}

// camera half of the per-frame constants: fp64, rounded once
void camera_params(FrameParams &p, const flod_camera *cam)
{
    memcpy(p.R, cam->R, sizeof(p.R)); memcpy(p.t, cam->t, sizeof(p.t)); memcpy(p.bg, cam->bg, sizeof(p.bg));
    p.fx = cam->fx; p.fy = cam->fy; p.cx = cam->cx; p.cy = cam->cy; p.z_near = cam->z_near;
    p.W = cam->width; p.H = cam->height;
    p.TX = (p.W + kTile - 1) / kTile; p.TY = (p.H + kTile - 1) / kTile;
    for (int i = 0; i < 3; ++i)
        p.centre[i] = (float)(-(((double)cam->R[i] * (double)cam->t[0] + (double)cam->R[3 + i] * (double)cam->t[1]) +
                                (double)cam->R[6 + i] * (double)cam->t[2]));
    p.limx = (float)(1.3 * (double)cam->width / (2.0 * (double)cam->fx));
    p.limy = (float)(1.3 * (double)cam->height / (2.0 * (double)cam->fy));
    {   // conservative off-screen test of k_geometry: |row of J|^2 <= pre_c1 / z^2 (R8's clamp bounds u and v)
        const double fm = std::max((double)cam->fx, (double)cam->fy), lm = std::max((double)p.limx, (double)p.limy);
        p.pre_c1 = (float)(fm * fm * (1.0 + lm * lm) * 1.0001);
    }
    p.n_tiles = p.TX * p.TY;
    p.ty_begin = 0; p.ty_end = p.TY; p.out_row0 = 0; p.out_rows = p.H;      // the whole image unless flod_render_rows says otherwise
}

// Eq. 7 thresholds of the level positions i0..i1 (squared, fp64 -> fp32 once): lo2[k], hi2[k], level_end[k]
void band_params(const flod_ctx *ctx, int i0, int i1, float fx, float gamma, int *level_end, float *lo2, float *hi2)
{
    for (int l = i0; l <= i1; ++l) {
        const int k = l - i0;
        level_end[k] = (int)(ctx->level_off[l + 1] - ctx->level_off[i0]);
        if (l == i1) lo2[k] = 0.0f;                                     // d_proj^(L_end) = 0
        else {
            const double d = (double)ctx->s_min[l] * (double)fx / (double)gamma;   // Eq. 7
            lo2[k] = (float)(d * d);
        }
    }
    for (int k = 0; k <= i1 - i0; ++k) hi2[k] = (k == 0) ? INFINITY : lo2[k - 1];  // d_proj^(L_start-1) = inf
}

// memset + the five kernels of a frame over `sc` (the scene, or a snapshot of it)
int enqueue_frame(flod_ctx *ctx, const SceneDev &sc, FrameParams &p, float *out_rgb_dev, cudaStream_t s)
{
    const int64_t n_scan = p.n_scan;
    p.max_pairs = (unsigned int)ctx->max_pairs;
    p.pair_rule = ctx->pair_rule;
    p.quad_gid = p.first_gid & ~3ll;
    p.n_pre_blocks = (int)((p.first_gid - p.quad_gid + n_scan + kGeoBlock - 1) / kGeoBlock);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    // Blend-driven ordering of long lists (two more launches), unless a view of the frame needs every list in its final
    // order -- and only when the previous frames had lists longer than kSortCap at all: the tile scan leaves that in a
    // mapped host word, read here without synchronisation.  It is a hint about cost, never about the result: either way
    // the frame's image is the same, bit for bit.
    {
        unsigned int *hint_dev = nullptr;
        CUDA_TRY(ctx, cudaHostGetDevicePointer((void **)&hint_dev, (void *)(ctx->sub_n_host + 3), 0));
        ctx->ws.long_hint = hint_dev;
    }
    const bool allowed = !(ctx->flags & (FLOD_OPT_DEBUG | FLOD_OPT_COUNT | FLOD_OPT_FULL_SORT));
    ctx->ws.dup_large_area = (ctx->flags & FLOD_OPT_SMALL_WINDOWS) ? kDupLargeAreaTest : kDupLargeArea;
    const unsigned int hint = *(volatile unsigned int *)(ctx->sub_n_host + 3);
    p.lazy_sort = (allowed && (hint & 1u)) ? 1 : 0;
    p.dup_both = (!(hint & 0x100u) || (hint & 2u)) ? 1 : 0;       // (no hint yet about this workspace's frames: both)
    const bool prof = ctx->flags & FLOD_OPT_PROFILE;
    // this frame's header was zeroed by the previous frame's k_blend (or by flod_set_workspace), the difference grid by
    // the previous tile scan: no memset in the stream
    ctx->hdr_turn ^= 1;
    ctx->ws.hdr = ctx->ws.hdr2[ctx->hdr_turn]; ctx->ws.hdr_next = ctx->ws.hdr2[ctx->hdr_turn ^ 1];
    if (ctx->flags & FLOD_OPT_DEBUG)   // the mask is zero outside the scanned levels
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->ws.mask, 0, (size_t)std::max<int64_t>(ctx->n_total, 1), s));
    int stage = 0;
    auto mark = [&]() { if (prof) cudaEventRecord(ctx->ev[stage], s); ++stage; };
    mark(); launch_geometry(*ctx, sc, p, s);
    mark(); launch_colour(*ctx, p, s);
    mark(); launch_duplicate(*ctx, p, s);
    mark(); launch_tile_sort(*ctx, p, s);
    mark();
    if (launch_blend(*ctx, p, out_rgb_dev, s) == 0)      // (an empty strip launches no blend kernel: zero the next header here)
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->ws.hdr_next, 0, sizeof(FrameHeader), s));
    launch_tile_sort_rest(*ctx, p, s); launch_blend_rest(*ctx, p, out_rgb_dev, s);     // (both exit at once unless a tile asked)
    mark();
    CUDA_TRY(ctx, cudaGetLastError());
    ctx->ev_valid = prof;
    ctx->last_stream = s; ctx->rendered = true;
    ctx->last_params = p; ctx->last_full_scene = sc.src_gid == nullptr;
    ctx->last_n_scan = n_scan; ctx->last_n_segs = p.n_pre_blocks;
    ctx->last_w = p.W; ctx->last_h = p.H; ctx->last_tx = p.TX; ctx->last_ty = p.TY; ctx->last_first_gid = p.first_gid;
    return FLOD_OK;
}

}  // namespace

extern "C" {

}  // extern "C"

namespace {

// flod_render / flod_render_rows: ty_end < 0 = the whole image into a [3][H][W] buffer
int render_impl(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma, int ty_begin, int ty_end,
                float *out_rgb_dev, void *stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (int rc = check_frame_args(ctx, cam, out_rgb_dev)) return rc;
    if (!(gamma > 0.0f) || !isfinite(gamma)) return fail(ctx, FLOD_E_INVALID_ARG, "render: gamma must be finite and > 0");
    const int last_level = ctx->first_level + ctx->n_levels - 1;
    if (mode.l_start < ctx->first_level || mode.l_end > last_level || mode.l_start > mode.l_end)
        return fail(ctx, FLOD_E_LEVEL_RANGE, "render: need first_level <= l_start <= l_end <= last_level");
    FrameParams p{};
    camera_params(p, cam);
    for (int i = 0; i < 3; ++i) p.ref[i] = ctx->has_ref ? ctx->ref[i] : p.centre[i];
    const int i0 = mode.l_start - ctx->first_level, i1 = mode.l_end - ctx->first_level;   // level positions
    p.n_levels = i1 - i0 + 1;
    p.first_gid = ctx->level_off[i0];
    p.n_scan = (int)(ctx->level_off[i1 + 1] - ctx->level_off[i0]);
    band_params(ctx, i0, i1, cam->fx, gamma, p.level_end, p.lo2, p.hi2);
    if (ty_end >= 0) {
        if (ty_begin < 0 || ty_begin > ty_end || ty_end > p.TY)
            return fail(ctx, FLOD_E_INVALID_ARG, "render_rows: need 0 <= ty_begin <= ty_end <= ceil(height / 16)");
        p.ty_begin = ty_begin; p.ty_end = ty_end;
        p.out_row0 = ty_begin * kTile;
        p.out_rows = std::min(p.H, ty_end * kTile) - p.out_row0;
        if (p.out_rows < 0) p.out_rows = 0;
    }
    return enqueue_frame(ctx, ctx->scene, p, out_rgb_dev, (cudaStream_t)stream);
}

}  // namespace

extern "C" {

int flod_render(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma, float *out_rgb_dev, void *stream)
{
    return render_impl(ctx, cam, mode, gamma, 0, -1, out_rgb_dev, stream);
}

int flod_render_rows(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma, int ty_begin, int ty_end,
                     float *out_strip_dev, void *stream)
{
    if (ty_end < 0) return ctx ? fail(ctx, FLOD_E_INVALID_ARG, "render_rows: ty_end < 0") : FLOD_E_INVALID_ARG;
    return render_impl(ctx, cam, mode, gamma, ty_begin, ty_end, out_strip_dev, stream);
}

}  // extern "C"

namespace {

// after a frame rendered into ws.image[i] on `s`: copy the image and the frame's overflow word out on `cs`
int enqueue_copy_out(flod_ctx *ctx, int i, const flod_camera *cam, float *out_rgb_host, cudaStream_t s, cudaStream_t cs)
{
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev_rendered[i], s));
    CUDA_TRY(ctx, cudaStreamWaitEvent(cs, ctx->ev_rendered[i], 0));
    CUDA_TRY(ctx, cudaMemcpyAsync(out_rgb_host, ctx->ws.image[i], (size_t)3 * cam->width * cam->height * sizeof(float),
                                  cudaMemcpyDeviceToHost, cs));
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->sub_n_host + 1 + i, ctx->ws.ovf_slots + i, sizeof(unsigned int), cudaMemcpyDeviceToHost, cs));
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev_copied[i], cs));
    ctx->copy_pending[i] = true;
    ctx->last_copy_stream = cs;
    ctx->img_turn = i ^ 1;
    return FLOD_OK;
}

}  // namespace

extern "C" {

int flod_render_to_host_async(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma, float *out_rgb_host,
                              void *stream, void *copy_stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!out_rgb_host) return fail(ctx, FLOD_E_INVALID_ARG, "render_to_host: null pointer");
    if (!ctx->has_ws) return fail(ctx, FLOD_E_NO_WORKSPACE, "render_to_host: no workspace set");
    cudaStream_t s = (cudaStream_t)stream, cs = (cudaStream_t)copy_stream;
    const int i = ctx->img_turn;
    // image[i] may still be on its way out (frame k - 2): the kernels of this frame wait for that copy only
    if (ctx->copy_pending[i]) CUDA_TRY(ctx, cudaStreamWaitEvent(s, ctx->ev_copied[i], 0));
    ctx->ws.ovf_out = ctx->ws.ovf_slots + i;               // the tile scan reports this frame's overflow word here
    const int rc = flod_render(ctx, cam, mode, gamma, ctx->ws.image[i], stream);
    ctx->ws.ovf_out = ctx->ws.ovf_slots + 2;
    if (rc != FLOD_OK) return rc;
    return enqueue_copy_out(ctx, i, cam, out_rgb_host, s, cs);
}

int flod_wait_host(flod_ctx *ctx)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    unsigned int ovf = 0;
    for (int i = 0; i < 2; ++i)
        if (ctx->copy_pending[i]) {
            CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_copied[i]));
            ctx->copy_pending[i] = false;
            ovf |= ctx->sub_n_host[1 + i];
            ctx->sub_n_host[1 + i] = 0;
        }
    if (ovf) return fail(ctx, FLOD_E_CAPACITY, overflow_text(ovf));
    return FLOD_OK;
}

int flod_render_to_host(flod_ctx *ctx, const flod_camera *cam, flod_level_mode mode, float gamma, float *out_rgb_host, void *stream)
{
    int rc = flod_render_to_host_async(ctx, cam, mode, gamma, out_rgb_host, stream, stream);
    if (rc != FLOD_OK) return rc;
    return flod_wait_host(ctx);
}

// ---------------------------------------------------------------- materialised G_sel (subset.cu)
}  // extern "C"

namespace {

struct SubLayout { SnapshotDev snap[2]; unsigned int *blk; size_t bytes; };

// two snapshots of up to n_range Gaussians + the per-block counters of the rebuild
SubLayout carve_subset(unsigned char *base, int64_t n_range)
{
    SubLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return (unsigned char *)((uintptr_t)base + o); };
    const size_t cap = (size_t)std::max<int64_t>(n_range, 1) + 8;       // k_geometry loads whole quads
    for (int i = 0; i < 2; ++i) {
        L.snap[i].n_sel = (unsigned int *)take(sizeof(unsigned int));
        for (int a = 0; a < 13; ++a) L.snap[i].plane[a] = (float *)take(cap * sizeof(float));
        L.snap[i].src_gid = (unsigned int *)take(cap * sizeof(unsigned int));
        L.snap[i].rec = (float4 *)take(cap * 8 * sizeof(float));
    }
    L.blk = (unsigned int *)take(((size_t)n_range / kGeoBlock + 4) * sizeof(unsigned int));
    L.bytes = off;
    return L;
}

bool subset_range(const flod_ctx *ctx, flod_level_mode mode, int *i0, int *i1)
{
    if (!ctx || !ctx->uploaded) return false;
    const int last_level = ctx->first_level + ctx->n_levels - 1;
    if (mode.l_start < ctx->first_level || mode.l_end > last_level || mode.l_start > mode.l_end) return false;
    *i0 = mode.l_start - ctx->first_level; *i1 = mode.l_end - ctx->first_level;
    return true;
}

}  // namespace

extern "C" {

size_t flod_subset_bytes(const flod_ctx *ctx, flod_level_mode mode)
{
    int i0, i1;
    if (!subset_range(ctx, mode, &i0, &i1)) return 0;
    return carve_subset(nullptr, ctx->level_off[i1 + 1] - ctx->level_off[i0]).bytes;
}

int flod_subset_set_arena(flod_ctx *ctx, void *arena_dev, size_t bytes, flod_level_mode mode)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ctx->uploaded) return fail(ctx, FLOD_E_NOT_UPLOADED, "subset_set_arena: no scene uploaded");
    int i0, i1;
    if (!subset_range(ctx, mode, &i0, &i1))
        return fail(ctx, FLOD_E_LEVEL_RANGE, "subset_set_arena: need first_level <= l_start <= l_end <= last_level");
    if (!arena_dev || (uintptr_t)arena_dev % 256) return fail(ctx, FLOD_E_INVALID_ARG, "subset_set_arena: null or unaligned pointer");
    SubLayout L = carve_subset((unsigned char *)arena_dev, ctx->level_off[i1 + 1] - ctx->level_off[i0]);
    if (bytes < L.bytes) return fail(ctx, FLOD_E_ARENA_TOO_SMALL, "subset_set_arena: arena too small");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if (ctx->sub_build_pending) cudaEventSynchronize(ctx->ev_sub_built);
    ctx->snap[0] = L.snap[0]; ctx->snap[1] = L.snap[1]; ctx->sub_blk = L.blk;
    ctx->sub_i0 = i0; ctx->sub_i1 = i1;
    ctx->sub_front = 0; ctx->sub_front_valid = false; ctx->sub_build_pending = false;
    ctx->sub_read_pending[0] = ctx->sub_read_pending[1] = false;
    ctx->has_subset = true;
    return FLOD_OK;
}

int flod_subset_build(flod_ctx *ctx, const float ref_pos[3], float fx, float gamma, void *stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ctx->has_subset) return fail(ctx, FLOD_E_NO_WORKSPACE, "subset_build: no subset arena set");
    if (!ref_pos) return fail(ctx, FLOD_E_INVALID_ARG, "subset_build: null reference position");
    for (int i = 0; i < 3; ++i)
        if (!isfinite(ref_pos[i]) || fabsf(ref_pos[i]) > 1e15f) return fail(ctx, FLOD_E_INVALID_ARG, "subset_build: reference must be finite, |x| <= 1e15");
    if (!(fx > 0.0f) || !isfinite(fx) || !(gamma > 0.0f) || !isfinite(gamma))
        return fail(ctx, FLOD_E_INVALID_ARG, "subset_build: fx and gamma must be finite and > 0");
    if (ctx->sub_build_pending) return fail(ctx, FLOD_E_INVALID_ARG, "subset_build: a rebuild is already enqueued (swap first)");
    cudaStream_t s = (cudaStream_t)stream;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    const int back = ctx->sub_front_valid ? ctx->sub_front ^ 1 : ctx->sub_front;
    // frames that still read the back snapshot (it was the front one before the last swap) come first
    if (ctx->sub_read_pending[back]) { CUDA_TRY(ctx, cudaStreamWaitEvent(s, ctx->ev_sub_read[back], 0)); ctx->sub_read_pending[back] = false; }
    SubsetParams q{};
    memcpy(q.ref, ref_pos, sizeof(q.ref));
    const int i0 = ctx->sub_i0, i1 = ctx->sub_i1;
    q.first_gid = ctx->level_off[i0];
    q.n_scan = (int)(ctx->level_off[i1 + 1] - ctx->level_off[i0]);
    q.n_levels = i1 - i0 + 1;
    band_params(ctx, i0, i1, fx, gamma, q.level_end, q.lo2, q.hi2);
    q.n_blocks = (int)((q.first_gid - (q.first_gid & ~3ll) + q.n_scan + kGeoBlock - 1) / kGeoBlock);
    launch_subset_build(*ctx, ctx->snap[back], q, s);
    CUDA_TRY(ctx, cudaGetLastError());
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->sub_n_host, ctx->snap[back].n_sel, sizeof(unsigned int), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev_sub_built, s));
    ctx->sub_build_pending = true;
    return FLOD_OK;
}

int flod_subset_ready(flod_ctx *ctx)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ctx->sub_build_pending) return 0;
    const cudaError_t e = cudaEventQuery(ctx->ev_sub_built);
    if (e == cudaSuccess) return 1;
    if (e == cudaErrorNotReady) return 0;
    return fail(ctx, FLOD_E_CUDA, cudaGetErrorString(e));
}

int flod_subset_swap(flod_ctx *ctx, int64_t *n_selected)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!ctx->sub_build_pending) return fail(ctx, FLOD_E_INVALID_ARG, "subset_swap: no rebuild enqueued");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev_sub_built));
    const int back = ctx->sub_front_valid ? ctx->sub_front ^ 1 : ctx->sub_front;
    ctx->sub_n[back] = (int64_t)*ctx->sub_n_host;
    ctx->sub_front = back; ctx->sub_front_valid = true; ctx->sub_build_pending = false;
    if (n_selected) *n_selected = ctx->sub_n[back];
    return FLOD_OK;
}

int flod_render_subset(flod_ctx *ctx, const flod_camera *cam, float *out_rgb_dev, void *stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (int rc = check_frame_args(ctx, cam, out_rgb_dev)) return rc;
    if (!ctx->has_subset || !ctx->sub_front_valid) return fail(ctx, FLOD_E_INVALID_ARG, "render_subset: no snapshot built and swapped in");
    const int f = ctx->sub_front;
    const SnapshotDev &sn = ctx->snap[f];
    SceneDev sc = ctx->scene;                                 // SH rows stay in the scene arena (read by gid)
    sc.mx = sn.plane[0]; sc.my = sn.plane[1]; sc.mz = sn.plane[2]; sc.rho2 = sn.plane[3]; sc.kappa = sn.plane[4];
    for (int k = 0; k < 6; ++k) sc.cov[k] = sn.plane[5 + k];
    sc.l2o = sn.plane[11]; sc.opacity = sn.plane[12];
    sc.src_gid = sn.src_gid; sc.rec = sn.rec;
    FrameParams p{};
    camera_params(p, cam);
    for (int i = 0; i < 3; ++i) p.ref[i] = p.centre[i];      // every entry of a snapshot is selected: one band [0, inf)
    p.n_levels = 1; p.first_gid = 0; p.n_scan = (int)ctx->sub_n[f];
    p.level_end[0] = p.n_scan; p.lo2[0] = 0.0f; p.hi2[0] = INFINITY;
    cudaStream_t s = (cudaStream_t)stream;
    const int rc = enqueue_frame(ctx, sc, p, out_rgb_dev, s);
    if (rc != FLOD_OK) return rc;
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev_sub_read[f], s));
    ctx->sub_read_pending[f] = true;
    return FLOD_OK;
}

size_t flod_backward_workspace_bytes(const flod_ctx *ctx)
{
    if (!ctx || !ctx->uploaded) return 0;
    return align_up(((size_t)std::max<int64_t>(ctx->n_total, 1) + 2 * kGeoBlock) * 9 * sizeof(float));
}

int flod_render_backward(flod_ctx *ctx, const flod_camera *cam, const float *dL_dimage_dev, const flod_grads *grads,
                         void *workspace_dev, size_t workspace_bytes, void *stream)
{
    if (!ctx) return FLOD_E_INVALID_ARG;
    if (!cam || !dL_dimage_dev || !grads || !workspace_dev) return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: null pointer");
    if (!grads->d_mean || !grads->d_log_scale || !grads->d_quat || !grads->d_opacity_logit || !grads->d_sh)
        return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: null gradient array");
    if (!ctx->rendered || !ctx->last_full_scene)
        return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: the last frame must come from flod_render");
    if ((uintptr_t)workspace_dev % 256 || workspace_bytes < flod_backward_workspace_bytes(ctx))
        return fail(ctx, FLOD_E_ARENA_TOO_SMALL, "render_backward: workspace unaligned or too small");
    const FrameParams &p = ctx->last_params;
    // the contract: the inputs of the forward pass that left its lists in the workspace
    FrameParams q{};
    camera_params(q, cam);
    if (memcmp(q.R, p.R, sizeof(q.R)) || memcmp(q.t, p.t, sizeof(q.t)) || memcmp(q.bg, p.bg, sizeof(q.bg)) || q.fx != p.fx ||
        q.fy != p.fy || q.cx != p.cx || q.cy != p.cy || q.W != p.W || q.H != p.H || q.z_near != p.z_near)
        return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: the camera is not the one of the last flod_render");
    if (p.ty_begin != 0 || p.ty_end != p.TY)
        return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: the last frame was a strip (flod_render_rows)");
    if (p.lazy_sort)
        return fail(ctx, FLOD_E_INVALID_ARG, "render_backward: render the frame with FLOD_OPT_FULL_SORT (its lists must be in their final order throughout)");
    cudaStream_t s = (cudaStream_t)stream;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    // gradients are indexed by gid over the whole scene: zero, then the drawn Gaussians add theirs
    const size_t n = (size_t)std::max<int64_t>(ctx->n_total, 1), K = (size_t)(ctx->sh_degree + 1) * (ctx->sh_degree + 1);
    CUDA_TRY(ctx, cudaMemsetAsync(grads->d_mean, 0, n * 3 * sizeof(float), s));
    CUDA_TRY(ctx, cudaMemsetAsync(grads->d_log_scale, 0, n * 3 * sizeof(float), s));
    CUDA_TRY(ctx, cudaMemsetAsync(grads->d_quat, 0, n * 4 * sizeof(float), s));
    CUDA_TRY(ctx, cudaMemsetAsync(grads->d_opacity_logit, 0, n * sizeof(float), s));
    CUDA_TRY(ctx, cudaMemsetAsync(grads->d_sh, 0, n * K * 3 * sizeof(float), s));
    CUDA_TRY(ctx, cudaMemsetAsync(workspace_dev, 0, flod_backward_workspace_bytes(ctx), s));
    launch_backward(*ctx, p, dL_dimage_dev, (float *)workspace_dev, *grads, s);
    CUDA_TRY(ctx, cudaGetLastError());
    return FLOD_OK;
}

int flod_get_stats(flod_ctx *ctx, flod_stats *out)
{
    if (!ctx || !out) return FLOD_E_INVALID_ARG;
    if (!ctx->rendered) return fail(ctx, FLOD_E_INVALID_ARG, "get_stats: nothing rendered yet");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->last_stream));
    FrameHeader h;
    CUDA_TRY(ctx, cudaMemcpy(&h, ctx->ws.hdr, sizeof(FrameHeader), cudaMemcpyDeviceToHost));
    memset(out, 0, sizeof(*out));
    out->n_sel = (int64_t)h.n_sel; out->n_front = (int64_t)h.n_front; out->n_vis = (int64_t)h.n_vis32;
    out->n_pairs = (int64_t)h.n_pairs; out->max_pairs = ctx->max_pairs; out->overflow = (int)h.overflow;
    out->evals = (int64_t)h.evals; out->blends = (int64_t)h.blends;
    out->n_scan = ctx->last_n_scan;
    if (ctx->ev_valid) {
        for (int i = 0; i < FLOD_N_STAGES; ++i) cudaEventElapsedTime(&out->ms_stage[i], ctx->ev[i], ctx->ev[i + 1]);
        cudaEventElapsedTime(&out->ms_total, ctx->ev[0], ctx->ev[FLOD_N_STAGES]);
    }
    if (h.overflow) return fail(ctx, FLOD_E_CAPACITY, overflow_text(h.overflow));
    return FLOD_OK;
}

int flod_debug_copy(flod_ctx *ctx, int what, void *host_dst, size_t bytes)
{
    if (!ctx || !host_dst) return FLOD_E_INVALID_ARG;
    if (what == FLOD_DBG_ACTIVATED) {
        if (!ctx->uploaded) return fail(ctx, FLOD_E_NOT_UPLOADED, "debug_copy: no scene uploaded");
        const size_t n = (size_t)ctx->n_total;
        if (bytes < n * 8 * sizeof(float)) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: buffer too small");
        std::vector<float> tmp(std::max<size_t>(n, 1));
        float *dst = (float *)host_dst;
        const float *planes[8] = {ctx->scene.cov[0], ctx->scene.cov[1], ctx->scene.cov[2], ctx->scene.cov[3],
                                  ctx->scene.cov[4], ctx->scene.cov[5], ctx->scene.opacity, ctx->scene.kappa};
        for (int k = 0; k < 8; ++k) {
            CUDA_TRY(ctx, cudaMemcpy(tmp.data(), planes[k], n * sizeof(float), cudaMemcpyDeviceToHost));
            for (size_t i = 0; i < n; ++i) dst[i * 8 + k] = tmp[i];
        }
        return FLOD_OK;
    }
    if (!ctx->rendered) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: nothing rendered yet");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->last_stream));
    FrameHeader h;
    CUDA_TRY(ctx, cudaMemcpy(&h, ctx->ws.hdr, sizeof(FrameHeader), cudaMemcpyDeviceToHost));
    switch (what) {
        case FLOD_DBG_MASK: {
            if (!(ctx->flags & FLOD_OPT_DEBUG)) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: MASK needs FLOD_OPT_DEBUG");
            if (bytes < (size_t)ctx->n_total) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: buffer too small");
            CUDA_TRY(ctx, cudaMemcpy(host_dst, ctx->ws.mask, (size_t)ctx->n_total, cudaMemcpyDeviceToHost));
            return FLOD_OK;
        }
        case FLOD_DBG_TILE_COUNTS: {
            const size_t tiles = (size_t)ctx->last_tx * ctx->last_ty;
            if (bytes < tiles * 4) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: buffer too small");
            std::vector<uint2> r(tiles);
            CUDA_TRY(ctx, cudaMemcpy(r.data(), ctx->ws.ranges, tiles * sizeof(uint2), cudaMemcpyDeviceToHost));
            uint32_t *dst = (uint32_t *)host_dst;
            for (size_t i = 0; i < tiles; ++i) dst[i] = r[i].y - r[i].x;
            return FLOD_OK;
        }
        case FLOD_DBG_PROJECTED: {
            if (!(ctx->flags & FLOD_OPT_DEBUG)) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: PROJECTED needs FLOD_OPT_DEBUG");
            const size_t nv = (size_t)h.n_vis32, nseg = (size_t)ctx->last_n_segs;
            if (bytes < nv * sizeof(flod_dbg_projected)) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: buffer too small");
            // segment s holds seg_count[s] records at positions s * kGeoBlock ..: concatenated they are in ascending gid
            std::vector<unsigned int> cnt(std::max<size_t>(nseg, 1));
            CUDA_TRY(ctx, cudaMemcpy(cnt.data(), ctx->ws.seg_count, nseg * 4, cudaMemcpyDeviceToHost));
            flod_dbg_projected *dst = (flod_dbg_projected *)host_dst;
            size_t k = 0;
            for (size_t sgm = 0; sgm < nseg && k < nv; ++sgm) {
                const size_t m = std::min<size_t>(cnt[sgm], nv - k);
                if (m) CUDA_TRY(ctx, cudaMemcpy(dst + k, ctx->ws.dbg + sgm * kGeoBlock, m * sizeof(flod_dbg_projected), cudaMemcpyDeviceToHost));
                k += m;
            }
            return FLOD_OK;
        }
        case FLOD_DBG_SORTED_PAIRS: {
            const size_t np = (size_t)h.n_pairs_clamped, ns = (size_t)ctx->last_n_segs * kGeoBlock;
            if (bytes < np * sizeof(flod_dbg_pair)) return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: buffer too small");
            const size_t tiles = (size_t)ctx->last_tx * ctx->last_ty;
            std::vector<uint2> r(std::max<size_t>(tiles, 1));
            std::vector<uint32_t> v(std::max<size_t>(np, 1)), dz(std::max<size_t>(ns, 1));
            std::vector<float4> dg(std::max<size_t>(ns, 1));
            CUDA_TRY(ctx, cudaMemcpy(dg.data(), ctx->ws.dirgid, ns * sizeof(float4), cudaMemcpyDeviceToHost));
            CUDA_TRY(ctx, cudaMemcpy(r.data(), ctx->ws.ranges, tiles * sizeof(uint2), cudaMemcpyDeviceToHost));
            CUDA_TRY(ctx, cudaMemcpy(v.data(), ctx->ws.vals, np * 4, cudaMemcpyDeviceToHost));
            CUDA_TRY(ctx, cudaMemcpy(dz.data(), ctx->ws.depth, ns * 4, cudaMemcpyDeviceToHost));
            flod_dbg_pair *dst = (flod_dbg_pair *)host_dst;
            for (size_t t = 0; t < tiles; ++t)
                for (size_t i = r[t].x; i < r[t].y && i < np; ++i) {
                    dst[i].tile = (uint32_t)t;
                    const uint32_t si = v[i];
                    const uint32_t bits = si < ns ? dz[si] : 0u;
                    memcpy(&dst[i].depth, &bits, 4);
                    uint32_t gid = 0xffffffffu;
                    if (si < ns) memcpy(&gid, &dg[si].w, 4);
                    dst[i].gid = gid;
                }
            return FLOD_OK;
        }
        default:
            return fail(ctx, FLOD_E_INVALID_ARG, "debug_copy: unknown selector");
    }
}

}  // extern "C"
