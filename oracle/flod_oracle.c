/*
 * oracle/flod_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow CPU oracle for the forward rasterizer of FLoD (arXiv 2408.12894), written from
 * PAPER.md and the readings listed in DESIGN.md §3.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * or constant generator with paper_2408_12894_b200/ (the CUDA path).
 *
 * What it computes, in the paper's order (P:n = /root/reference/PAPER.md line n):
 *   O0  activation          Sigma = R S S^T R^T                         Eq. 1
 *   O1  level selection     G_sel by distance bands, d_proj = s_min f / gamma   Eq. 6-7
 *   O2  cull + projection   "projected to 2D screenspace", mu'
 *   O3  EWA covariance      Sigma' (+0.3 px^2 dilation), conic = Sigma'^-1     P:110; DESIGN R8,R9
 *   O4  footprint rect      box of the alpha = 1/255 contour, 16x16 tiles      DESIGN R13
 *   O5  colour              spherical harmonics -> RGB                        P:97; DESIGN R16
 *   O6  pairs, order        per tile, ascending (depth, gid)                   P:111; DESIGN R15
 *   O7  compositing         alpha = o exp(-1/2 d^T Sigma'^-1 d), front to back  Eq. 2
 *
 * Arithmetic: O1-O4 are "canonical fp32": every operation below is one correctly rounded IEEE
 * binary32 operation in exactly the written order; compile with -ffp-contract=off and without
 * -ffast-math so that gcc neither fuses nor reorders (x86-64 SSE: no excess precision).  Per-frame
 * constants are computed once in fp64 and rounded to fp32.  O0, O5 and O7 are fp64 on fp32 inputs.
 *
 * Pins (tests/test_oracle_*.py, all run with -m "not gpu"): worked values of SPEC.md, closed form
 * of one isotropic Gaussian's footprint, two-layer compositing example, invariants on T and alpha,
 * band partition, tiled == brute force bit-exactly, numerical Jacobian of the pinhole map, SH
 * orthonormality by quadrature, SH basis == real combinations of scipy's complex harmonics.
 * parity unpinned: the inherited constants 0.3, 1.3, 1e-4, 0.5 and which SH sign convention a
 * trained model would use -- nothing in the paper fixes them.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_LEVELS 16
#define ORC_TILE 16

typedef struct {
    int64_t n; int level; float s_min;
    const float *mean, *log_scale, *quat, *opacity_logit, *sh;
} orc_level_desc;

typedef struct {
    float R[9], t[3];
    float fx, fy, cx, cy;
    int width, height;
    float z_near;
    float bg[3];
} orc_camera;

typedef struct {
    int L, sh_degree, K;
    int64_t n_total;
    int64_t offset[ORC_MAX_LEVELS + 1];
    int level_id[ORC_MAX_LEVELS];
    float s_min[ORC_MAX_LEVELS];
    float *mean;      /* [n][3] */
    float *cov;       /* [n][6] xx,xy,xz,yy,yz,zz */
    float *opacity;   /* [n] */
    float *kappa;     /* [n] 2 ln(255 o) */
    uint8_t *dead;    /* [n] o < 1/255 */
    float *sh;        /* [n][K][3] */
    float *raw_ls, *raw_q, *raw_logit;   /* [n][3], [n][4], [n]: the uploaded attributes (O64 activates from them) */
} orc_scene;

/* ---------------------------------------------------------------- small pins: Eq. 3, 4, 7 --- */

/* Eq. 3: s_min^(l) = tau * rho^(1-l) for l < L_max, 0 at L_max. */
double orc_scale_constraint(int level, double tau, double rho, int l_max)
{
    if (level < 1 || level > l_max) return NAN;
    if (level == l_max) return 0.0;
    return tau * pow(rho, 1.0 - (double)level);
}

/* Eq. 4: s^(l) = exp(s_opt) + s_min^(l). */
double orc_effective_scale(double s_opt, double s_min) { return exp(s_opt) + s_min; }

/* Eq. 7: d_proj^(l) = s_min^(l) / gamma * f. */
double orc_d_proj(double s_min, double gamma, double f) { return s_min / gamma * f; }

/* ------------------------------------------------------------------------ O0 activation --- */

/* Eq. 1: Sigma = R S S^T R^T, S = diag(s), R from the normalised quaternion (w,x,y,z).
 * fp64 from the fp32 inputs, each output rounded once to fp32.  Operation order is the one of
 * DESIGN.md §3 "O0" so that the library's upload, which restates it, rounds identically. */
void orc_activate_one(const float ls[3], const float q[4], float logit,
                      float cov[6], float *opacity, float *kappa, uint8_t *dead)
{
    double s0 = exp((double)ls[0]), s1 = exp((double)ls[1]), s2 = exp((double)ls[2]);
    double w = q[0], x = q[1], y = q[2], z = q[3];
    double nrm = sqrt(((w * w + x * x) + y * y) + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    double R[3][3];
    R[0][0] = 1.0 - 2.0 * (y * y + z * z); R[0][1] = 2.0 * (x * y - w * z); R[0][2] = 2.0 * (x * z + w * y);
    R[1][0] = 2.0 * (x * y + w * z); R[1][1] = 1.0 - 2.0 * (x * x + z * z); R[1][2] = 2.0 * (y * z - w * x);
    R[2][0] = 2.0 * (x * z - w * y); R[2][1] = 2.0 * (y * z + w * x); R[2][2] = 1.0 - 2.0 * (x * x + y * y);
    double v0 = s0 * s0, v1 = s1 * s1, v2 = s2 * s2;
    int k = 0;
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j)
            cov[k++] = (float)((R[i][0] * v0 * R[j][0] + R[i][1] * v1 * R[j][1]) + R[i][2] * v2 * R[j][2]);
    float o = (float)(1.0 / (1.0 + exp(-(double)logit)));
    *opacity = o;
    *kappa = (float)(2.0 * log(255.0 * (double)o));
    *dead = (uint8_t)(o < (float)(1.0 / 255.0));
}

orc_scene *orc_scene_create(int n_levels, const orc_level_desc *lv, int sh_degree)
{
    if (n_levels < 1 || n_levels > ORC_MAX_LEVELS || sh_degree < 0 || sh_degree > 3) return NULL;
    orc_scene *sc = (orc_scene *)calloc(1, sizeof(orc_scene));
    sc->L = n_levels; sc->sh_degree = sh_degree; sc->K = (sh_degree + 1) * (sh_degree + 1);
    for (int l = 0; l < n_levels; ++l) {
        sc->offset[l + 1] = sc->offset[l] + lv[l].n;
        sc->s_min[l] = lv[l].s_min;
        sc->level_id[l] = lv[l].level;
    }
    int64_t n = sc->n_total = sc->offset[n_levels];
    int64_t na = n > 0 ? n : 1;
    sc->mean = (float *)malloc(sizeof(float) * 3 * na);
    sc->cov = (float *)malloc(sizeof(float) * 6 * na);
    sc->opacity = (float *)malloc(sizeof(float) * na);
    sc->kappa = (float *)malloc(sizeof(float) * na);
    sc->dead = (uint8_t *)malloc(na);
    sc->sh = (float *)malloc(sizeof(float) * 3 * sc->K * na);
    sc->raw_ls = (float *)malloc(sizeof(float) * 3 * na);
    sc->raw_q = (float *)malloc(sizeof(float) * 4 * na);
    sc->raw_logit = (float *)malloc(sizeof(float) * na);
    for (int l = 0; l < n_levels; ++l) {
        int64_t base = sc->offset[l];
        memcpy(sc->mean + 3 * base, lv[l].mean, sizeof(float) * 3 * lv[l].n);
        memcpy(sc->sh + 3 * sc->K * base, lv[l].sh, sizeof(float) * 3 * sc->K * lv[l].n);
        memcpy(sc->raw_ls + 3 * base, lv[l].log_scale, sizeof(float) * 3 * lv[l].n);
        memcpy(sc->raw_q + 4 * base, lv[l].quat, sizeof(float) * 4 * lv[l].n);
        memcpy(sc->raw_logit + base, lv[l].opacity_logit, sizeof(float) * lv[l].n);
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < lv[l].n; ++i)
            orc_activate_one(lv[l].log_scale + 3 * i, lv[l].quat + 4 * i, lv[l].opacity_logit[i],
                             sc->cov + 6 * (base + i), sc->opacity + base + i, sc->kappa + base + i,
                             sc->dead + base + i);
    }
    return sc;
}

void orc_scene_destroy(orc_scene *sc)
{
    if (!sc) return;
    free(sc->mean); free(sc->cov); free(sc->opacity); free(sc->kappa); free(sc->dead); free(sc->sh);
    free(sc->raw_ls); free(sc->raw_q); free(sc->raw_logit);
    free(sc);
}

int64_t orc_scene_n_total(const orc_scene *sc) { return sc->n_total; }
const float *orc_scene_cov(const orc_scene *sc) { return sc->cov; }
const float *orc_scene_opacity(const orc_scene *sc) { return sc->opacity; }
const float *orc_scene_kappa(const orc_scene *sc) { return sc->kappa; }
const uint8_t *orc_scene_dead(const orc_scene *sc) { return sc->dead; }

/* -------------------------------------------------------------------------------- O5 SH --- */

/* Real orthonormal spherical harmonics up to degree 3 in the order (l, m = -l..l), sign
 * convention of DESIGN.md R16.  d must be a unit vector. */
void orc_sh_basis(int degree, const double d[3], double Y[16])
{
    const double PI = 3.14159265358979323846;
    double x = d[0], y = d[1], z = d[2];
    Y[0] = 0.5 * sqrt(1.0 / PI);
    if (degree < 1) return;
    double c1 = sqrt(3.0 / (4.0 * PI));
    Y[1] = -c1 * y; Y[2] = c1 * z; Y[3] = -c1 * x;
    if (degree < 2) return;
    double xx = x * x, yy = y * y, zz = z * z;
    Y[4] = 0.5 * sqrt(15.0 / PI) * x * y;
    Y[5] = -0.5 * sqrt(15.0 / PI) * y * z;
    Y[6] = 0.25 * sqrt(5.0 / PI) * (2.0 * zz - xx - yy);
    Y[7] = -0.5 * sqrt(15.0 / PI) * x * z;
    Y[8] = 0.25 * sqrt(15.0 / PI) * (xx - yy);
    if (degree < 3) return;
    Y[9] = -0.25 * sqrt(35.0 / (2.0 * PI)) * y * (3.0 * xx - yy);
    Y[10] = 0.5 * sqrt(105.0 / PI) * x * y * z;
    Y[11] = -0.25 * sqrt(21.0 / (2.0 * PI)) * y * (4.0 * zz - xx - yy);
    Y[12] = 0.25 * sqrt(7.0 / PI) * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);
    Y[13] = -0.25 * sqrt(21.0 / (2.0 * PI)) * x * (4.0 * zz - xx - yy);
    Y[14] = 0.5 * sqrt(105.0 / PI) * 0.5 * z * (xx - yy);
    Y[15] = -0.25 * sqrt(35.0 / (2.0 * PI)) * x * (xx - 3.0 * yy);
}

/* O5: colour of one Gaussian seen from camera centre c: max(0, 0.5 + sum_k Y_k(dir) sh[k][ch]). */
void orc_sh_color(int degree, const float mean[3], const float cam_centre[3], const float *sh, double rgb[3])
{
    double d[3] = { (double)mean[0] - (double)cam_centre[0], (double)mean[1] - (double)cam_centre[1],
                    (double)mean[2] - (double)cam_centre[2] };
    double n = sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
    d[0] /= n; d[1] /= n; d[2] /= n;
    double Y[16];
    orc_sh_basis(degree, d, Y);
    int K = (degree + 1) * (degree + 1);
    for (int ch = 0; ch < 3; ++ch) {
        double acc = 0.0;
        for (int k = 0; k < K; ++k) acc += Y[k] * (double)sh[3 * k + ch];
        acc += 0.5;
        rgb[ch] = acc > 0.0 ? acc : 0.0;
    }
}

/* ------------------------------------------------------------------------------- frame --- */

enum { ST_UNSELECTED = 0, ST_CULL_NEAR = 1, ST_CULL_DEAD = 2, ST_CULL_DET = 3, ST_EMPTY_RECT = 4, ST_VISIBLE = 5 };

typedef struct { uint32_t tile; float depth; uint32_t gid; } orc_pair;

typedef struct {
    const orc_scene *sc;
    orc_camera cam;
    int l_start, l_end;          /* 1-based positions in the uploaded ladder */
    float gamma;
    int TX, TY;
    float centre[3], ref[3], limx, limy;
    float lo2[ORC_MAX_LEVELS], hi2[ORC_MAX_LEVELS];
    uint8_t *mask;               /* [n_total] Eq. 6 membership */
    uint8_t *state;              /* [n_total] ST_* */
    float *mu2d;                 /* [n][2] */
    float *depth;                /* [n] */
    float *cov2d;                /* [n][3] a,b,c (dilated) */
    float *conic;                /* [n][3] A,B,C */
    int32_t *rect;               /* [n][4] tx0,ty0,tx1,ty1 */
    uint32_t *n_tiles;           /* [n] */
    double *rgb;                 /* [n][3] */
    int64_t n_scan, n_sel, n_front, n_vis, n_pairs, n_bf;
    orc_pair *pairs;             /* [n_pairs] sorted by (tile, depth, gid) */
    uint32_t *tile_start;        /* [T_n + 1] */
    uint32_t *bf_list;           /* [n_bf] all gaussians with state >= ST_EMPTY_RECT, (depth,gid) order */
    int bf_sorted;               /* bf_list is ordered on first brute-force use */
    int what;                    /* ORC_WITH_* : which of the optional products were built */
    /* variant O64 (ORC_FP64): the same steps with every operation in fp64 and nothing rounded to fp32 on the way */
    double *mu2d64, *depth64, *conic64, *opacity64;
} orc_frame;

enum { ORC_WITH_COLOUR = 1, ORC_WITH_PAIRS = 2, ORC_FP64 = 4, ORC_RULE_ELLIPSE = 8 };

/* Eq. 7 with the two boundary overrides, squared and rounded once to fp32.
 * Bands are half-open [d_proj^(l), d_proj^(l-1)) (DESIGN R1).  f = fx (DESIGN R4). */
void orc_band_thresholds(int L, const float *s_min, int l_start, int l_end, float fx, float gamma,
                         float *lo2, float *hi2)
{
    for (int l = 1; l <= L; ++l) { lo2[l - 1] = 0.0f; hi2[l - 1] = 0.0f; }
    for (int l = l_start; l <= l_end; ++l) {
        if (l == l_end) lo2[l - 1] = 0.0f;
        else {
            double d = (double)s_min[l - 1] * (double)fx / (double)gamma;
            lo2[l - 1] = (float)(d * d);
        }
    }
    for (int l = l_start; l <= l_end; ++l)
        hi2[l - 1] = (l == l_start) ? INFINITY : lo2[l - 2];
}

/* O1 predicate, canonical fp32 (Eq. 6; Euclidean distance to the reference, DESIGN R2,R3). */
static inline int select_one(const float m[3], const float ref[3], float lo2, float hi2)
{
    float dx = m[0] - ref[0], dy = m[1] - ref[1], dz = m[2] - ref[2];
    float d2 = (dx * dx + dy * dy) + dz * dz;
    return (d2 >= lo2) && (d2 < hi2);
}

/* O2-O4 for one Gaussian, canonical fp32.  Returns an ST_* state (never ST_UNSELECTED). */
static int project_one(const orc_frame *fr, int64_t g)
{
    const orc_scene *sc = fr->sc;
    const orc_camera *cm = &fr->cam;
    const float *R = cm->R, *t = cm->t;
    const float *m = sc->mean + 3 * g;
    const float *S = sc->cov + 6 * g;
    /* O2: p = R mu + t */
    float px = ((R[0] * m[0] + R[1] * m[1]) + R[2] * m[2]) + t[0];
    float py = ((R[3] * m[0] + R[4] * m[1]) + R[5] * m[2]) + t[1];
    float pz = ((R[6] * m[0] + R[7] * m[1]) + R[8] * m[2]) + t[2];
    if (pz <= cm->z_near) return ST_CULL_NEAR;
    if (sc->dead[g]) return ST_CULL_DEAD;
    float ix = px / pz, iy = py / pz;
    float mx = cm->fx * ix + cm->cx;
    float my = cm->fy * iy + cm->cy;
    /* O3: Jacobian at the clamped point (DESIGN R8), M = J R_cam, Sigma' = M Sigma M^T + 0.3 I */
    float u = fminf(fmaxf(ix, -fr->limx), fr->limx);
    float v = fminf(fmaxf(iy, -fr->limy), fr->limy);
    float j00 = cm->fx / pz;
    float j02 = -((cm->fx * u) / pz);
    float j11 = cm->fy / pz;
    float j12 = -((cm->fy * v) / pz);
    float m00 = j00 * R[0] + j02 * R[6], m01 = j00 * R[1] + j02 * R[7], m02 = j00 * R[2] + j02 * R[8];
    float m10 = j11 * R[3] + j12 * R[6], m11 = j11 * R[4] + j12 * R[7], m12 = j11 * R[5] + j12 * R[8];
    float v0x = (S[0] * m00 + S[1] * m01) + S[2] * m02;
    float v0y = (S[1] * m00 + S[3] * m01) + S[4] * m02;
    float v0z = (S[2] * m00 + S[4] * m01) + S[5] * m02;
    float v1x = (S[0] * m10 + S[1] * m11) + S[2] * m12;
    float v1y = (S[1] * m10 + S[3] * m11) + S[4] * m12;
    float v1z = (S[2] * m10 + S[4] * m11) + S[5] * m12;
    float a = ((m00 * v0x + m01 * v0y) + m02 * v0z) + 0.3f;
    float b = (m10 * v0x + m11 * v0y) + m12 * v0z;
    float c = ((m10 * v1x + m11 * v1y) + m12 * v1z) + 0.3f;
    float det = a * c - b * b;
    fr->mu2d[2 * g] = mx; fr->mu2d[2 * g + 1] = my; fr->depth[g] = pz;
    fr->cov2d[3 * g] = a; fr->cov2d[3 * g + 1] = b; fr->cov2d[3 * g + 2] = c;
    if (!(det > 0.0f)) return ST_CULL_DET;
    fr->conic[3 * g] = c / det;
    fr->conic[3 * g + 1] = -(b / det);
    fr->conic[3 * g + 2] = a / det;
    /* O4: axis-aligned box of the alpha = 1/255 contour, padded (DESIGN R13) */
    float kap = sc->kappa[g];
    float hx = sqrtf(kap * a) * 1.0009765625f + 0.015625f;
    float hy = sqrtf(kap * c) * 1.0009765625f + 0.015625f;
    float fTX = (float)fr->TX, fTY = (float)fr->TY;
    float x0 = fminf(fmaxf(floorf((mx - hx) * 0.0625f), 0.0f), fTX);
    float x1 = fminf(fmaxf(floorf((mx + hx) * 0.0625f) + 1.0f, 0.0f), fTX);
    float y0 = fminf(fmaxf(floorf((my - hy) * 0.0625f), 0.0f), fTY);
    float y1 = fminf(fmaxf(floorf((my + hy) * 0.0625f) + 1.0f, 0.0f), fTY);
    int32_t tx0 = (int32_t)x0, tx1 = (int32_t)x1, ty0 = (int32_t)y0, ty1 = (int32_t)y1;
    fr->rect[4 * g] = tx0; fr->rect[4 * g + 1] = ty0; fr->rect[4 * g + 2] = tx1; fr->rect[4 * g + 3] = ty1;
    uint32_t nt = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
    fr->n_tiles[g] = nt;
    return nt ? ST_VISIBLE : ST_EMPTY_RECT;
}

/* ---- variant O64 (SURVEY 8(c) "Oracle variants"): steps O0-O4 with every operation in fp64 on the fp32 inputs and
 * no intermediate rounding -- the mathematical result the canonical-fp32 sequence approximates.  NOT a parity target:
 * it exists to report how many masks / rects differ between the two and how far the images are apart.  The fp32
 * copies it leaves in mu2d / depth / conic / rect are for reporting; compositing reads the fp64 arrays. */
static int project_one_f64(const orc_frame *fr, int64_t g, const double centre[3], double limx, double limy)
{
    const orc_scene *sc = fr->sc;
    const orc_camera *cm = &fr->cam;
    const float *R = cm->R, *t = cm->t;
    const float *m = sc->mean + 3 * g;
    /* O0 in fp64 (Eq. 1), unrounded */
    const float *ls = sc->raw_ls + 3 * g, *q = sc->raw_q + 4 * g;
    double s0 = exp((double)ls[0]), s1 = exp((double)ls[1]), s2 = exp((double)ls[2]);
    double w = q[0], x = q[1], y = q[2], z = q[3];
    double nrm = sqrt(((w * w + x * x) + y * y) + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    double Rg[3][3] = {
        { 1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z), 2.0 * (x * z + w * y) },
        { 2.0 * (x * y + w * z), 1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x) },
        { 2.0 * (x * z - w * y), 2.0 * (y * z + w * x), 1.0 - 2.0 * (x * x + y * y) } };
    double v[3] = { s0 * s0, s1 * s1, s2 * s2 }, S[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            S[i][j] = (Rg[i][0] * v[0] * Rg[j][0] + Rg[i][1] * v[1] * Rg[j][1]) + Rg[i][2] * v[2] * Rg[j][2];
    double o = 1.0 / (1.0 + exp(-(double)sc->raw_logit[g]));
    /* O2 */
    double px = ((double)R[0] * m[0] + (double)R[1] * m[1] + (double)R[2] * m[2]) + t[0];
    double py = ((double)R[3] * m[0] + (double)R[4] * m[1] + (double)R[5] * m[2]) + t[1];
    double pz = ((double)R[6] * m[0] + (double)R[7] * m[1] + (double)R[8] * m[2]) + t[2];
    if (pz <= (double)cm->z_near) return ST_CULL_NEAR;
    if (o < 1.0 / 255.0) return ST_CULL_DEAD;
    double ix = px / pz, iy = py / pz;
    double mx = (double)cm->fx * ix + cm->cx, my = (double)cm->fy * iy + cm->cy;
    /* O3 */
    double u = fmin(fmax(ix, -limx), limx), vv = fmin(fmax(iy, -limy), limy);
    double J[2][3] = { { cm->fx / pz, 0.0, -((double)cm->fx * u) / pz }, { 0.0, cm->fy / pz, -((double)cm->fy * vv) / pz } };
    double M[2][3];
    for (int i = 0; i < 2; ++i)
        for (int k = 0; k < 3; ++k) M[i][k] = J[i][0] * R[k] + J[i][1] * R[3 + k] + J[i][2] * R[6 + k];
    double c2[2][2];
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) {
            double acc = 0.0;
            for (int k = 0; k < 3; ++k)
                for (int l = 0; l < 3; ++l) acc += M[i][k] * S[k][l] * M[j][l];
            c2[i][j] = acc;
        }
    double a = c2[0][0] + 0.3, b = c2[0][1], c = c2[1][1] + 0.3;
    double det = a * c - b * b;
    fr->mu2d64[2 * g] = mx; fr->mu2d64[2 * g + 1] = my; fr->depth64[g] = pz; fr->opacity64[g] = o;
    fr->mu2d[2 * g] = (float)mx; fr->mu2d[2 * g + 1] = (float)my; fr->depth[g] = (float)pz;
    fr->cov2d[3 * g] = (float)a; fr->cov2d[3 * g + 1] = (float)b; fr->cov2d[3 * g + 2] = (float)c;
    if (!(det > 0.0)) return ST_CULL_DET;
    fr->conic64[3 * g] = c / det; fr->conic64[3 * g + 1] = -(b / det); fr->conic64[3 * g + 2] = a / det;
    for (int k = 0; k < 3; ++k) fr->conic[3 * g + k] = (float)fr->conic64[3 * g + k];
    /* O4: the exact box of the alpha = 1/255 contour (no pad: the pad of the fp32 sequence covers ITS rounding) */
    double kap = 2.0 * log(255.0 * o);
    double hx = sqrt(kap * a), hy = sqrt(kap * c);
    double TXd = fr->TX, TYd = fr->TY;
    int32_t tx0 = (int32_t)fmin(fmax(floor((mx - hx) / 16.0), 0.0), TXd), tx1 = (int32_t)fmin(fmax(floor((mx + hx) / 16.0) + 1.0, 0.0), TXd);
    int32_t ty0 = (int32_t)fmin(fmax(floor((my - hy) / 16.0), 0.0), TYd), ty1 = (int32_t)fmin(fmax(floor((my + hy) / 16.0) + 1.0, 0.0), TYd);
    fr->rect[4 * g] = tx0; fr->rect[4 * g + 1] = ty0; fr->rect[4 * g + 2] = tx1; fr->rect[4 * g + 3] = ty1;
    uint32_t nt = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
    fr->n_tiles[g] = nt;
    return nt ? ST_VISIBLE : ST_EMPTY_RECT;
}

static const orc_frame *g_sort_frame;   /* qsort has no context argument; frames are built serially */
static int cmp_pair64(const void *pa, const void *pb)
{
    const orc_pair *a = (const orc_pair *)pa, *b = (const orc_pair *)pb;
    if (a->tile != b->tile) return a->tile < b->tile ? -1 : 1;
    double da = g_sort_frame->depth64[a->gid], db = g_sort_frame->depth64[b->gid];
    if (da != db) return da < db ? -1 : 1;
    if (a->gid != b->gid) return a->gid < b->gid ? -1 : 1;
    return 0;
}

/* ---- O6, pair rule 2 "ellipse" (DESIGN R26).  Pair rule 1 "box" lists a visible Gaussian in EVERY tile of
 * its rect (O4).  Rule 2 lists it, inside that rect, only in the tiles that hold a pixel centre of the (padded) contour
 * alpha = 1/255 of Eq. 2.  With the exponent of Eq. 2 in its factorised form (DESIGN R25),
 *     log2 alpha = log2 o - a w^2 - d dy^2,   w = dx + k dy,   k = B/A,  a = A log2(e)/2,  d = (C - B^2/A) log2(e)/2,
 * the contour is  a w^2 + d dy^2 = E = log2 o + log2 255.  The pixel centres of tile row ty are the band
 * y in [16 ty + .5, 16 ty + 15.5]; the ellipse cut by a band is convex, so the listed tiles of a row are ONE span
 * [ta, tb].  For a fixed dy = y - mu'y the ellipse is x - mu'x in [sl dy - s(dy), sl dy + s(dy)], sl = -k,
 * s(dy)^2 = KA - DA dy^2, KA = E/a, DA = d/a; the right end is concave in dy with its maximum at the ellipse's rightmost
 * point dy = dyt = -k sqrt(KA / (DA (DA + k^2))), so over the band it is largest at clamp(dyt, band) (the left end
 * smallest at clamp(-dyt, band)).  A tile column holds pixel centres x in [16 tx + .5, 16 tx + 15.5].
 * Arithmetic: k, a, d are derived from the ROUNDED fp32 conic (A, B, C) that O7 evaluates, in fp64 (C - B^2/A cancels
 * for thin diagonal footprints), each rounded once to fp32; everything after that is canonical fp32, like O1-O4:
 * one IEEE binary32 operation per written operation.  In this parametrisation nothing cancels except s^2 near the
 * ellipse's tips, where an error e in s^2 moves s by up to sqrt(e): the ends are padded by 2^-8 sqrt(KA) + 2^-6 pixels
 * plus 2^-20 of the magnitudes that were added, E by 2^-9 E + 2^-16.
 * Returns the number of tiles of row ty (0: none) and the span in *ta, *tb (inclusive). */
static int ellipse_row_span(float mx, float my, float cA, float cB, float cC, float opacity,
                            int tx0, int tx1, int ty, int *ta_out, int *tb_out)
{
    const double LOG2E = 1.4426950408889634;
    const double dA = (double)cA, dB = (double)cB, dC = (double)cC;
    const double rA = 1.0 / dA;
    const float k = (float)(dB * rA);
    const float a = -(float)((-0.5 * LOG2E) * dA);
    const float d = -fminf((float)((-0.5 * LOG2E) * (dC - (dB * dB) * rA)), 0.0f);
    const float l2o = (float)log2((double)opacity);
    *ta_out = tx0; *tb_out = tx1 - 1;
    if (!(a > 0.0f)) return tx1 - tx0;                       /* not an ellipse after rounding: the box rule */
    const float E = (l2o + 7.994353436858858f) * 1.001953125f + 0.0000152587890625f;
    const float sl = -k;
    const float ra = 1.0f / a;
    const float KA = E * ra;
    const float DA = d * ra;
    float dyt;
    if (DA > 0.0f) dyt = -(k * sqrtf(KA / (DA * (DA + k * k))));
    else dyt = k < 0.0f ? INFINITY : (k > 0.0f ? -INFINITY : 0.0f);      /* a strip: the ends are linear in dy */
    const float pad = sqrtf(KA) * 0.00390625f + 0.015625f;
    const float y0 = ((float)(16 * ty) + 0.5f) - my, y1 = y0 + 15.0f;
    const float dn = fminf(fmaxf(0.0f, y0), y1);
    if (DA * (dn * dn) > KA * 1.001953125f) return 0;        /* the band misses the ellipse */
    const float dh = fminf(fmaxf(dyt, y0), y1), dl = fminf(fmaxf(-dyt, y0), y1);
    const float sh = sqrtf(fmaxf(0.0f, KA - DA * (dh * dh))), sq = sqrtf(fmaxf(0.0f, KA - DA * (dl * dl)));
    const float ch = sl * dh, cl = sl * dl;
    const float padr = pad + ((fabsf(mx) + fabsf(ch)) + fabsf(cl)) * 9.5367431640625e-7f;
    const float xh = (mx + (ch + sh)) + padr;
    const float xl = (mx + (cl - sq)) - padr;
    const float ta = fmaxf(ceilf((xl - 15.5f) * 0.0625f), (float)tx0);
    const float tb = fminf(floorf((xh - 0.5f) * 0.0625f), (float)(tx1 - 1));
    if (!(tb >= ta)) return 0;
    *ta_out = (int)ta; *tb_out = (int)tb;
    return (int)tb - (int)ta + 1;
}

/* the tiles of row ty of Gaussian g's rect under the frame's pair rule */
static inline int row_span(const orc_frame *fr, int64_t g, int ty, int *ta, int *tb)
{
    const int32_t *r = fr->rect + 4 * g;
    if (!(fr->what & ORC_RULE_ELLIPSE)) { *ta = r[0]; *tb = r[2] - 1; return r[2] - r[0]; }
    return ellipse_row_span(fr->mu2d[2 * g], fr->mu2d[2 * g + 1], fr->conic[3 * g], fr->conic[3 * g + 1], fr->conic[3 * g + 2],
                            fr->sc->opacity[g], r[0], r[2], ty, ta, tb);
}

static int cmp_pair(const void *pa, const void *pb)
{
    const orc_pair *a = (const orc_pair *)pa, *b = (const orc_pair *)pb;
    if (a->tile != b->tile) return a->tile < b->tile ? -1 : 1;
    if (a->depth != b->depth) return a->depth < b->depth ? -1 : 1;
    if (a->gid != b->gid) return a->gid < b->gid ? -1 : 1;
    return 0;
}

static int cmp_bf(const void *pa, const void *pb)
{
    uint32_t a = *(const uint32_t *)pa, b = *(const uint32_t *)pb;
    if (g_sort_frame->what & ORC_FP64) {
        double da = g_sort_frame->depth64[a], db = g_sort_frame->depth64[b];
        if (da != db) return da < db ? -1 : 1;
        return a < b ? -1 : (a > b ? 1 : 0);
    }
    float da = g_sort_frame->depth[a], db = g_sort_frame->depth[b];
    if (da != db) return da < db ? -1 : 1;
    return a < b ? -1 : (a > b ? 1 : 0);
}

void orc_frame_destroy(orc_frame *fr)
{
    if (!fr) return;
    free(fr->mask); free(fr->state); free(fr->mu2d); free(fr->depth); free(fr->cov2d); free(fr->conic);
    free(fr->rect); free(fr->n_tiles); free(fr->rgb); free(fr->pairs); free(fr->tile_start); free(fr->bf_list);
    free(fr->mu2d64); free(fr->depth64); free(fr->conic64); free(fr->opacity64);
    free(fr);
}

/* Steps O1-O6 for one camera and mode.  ref_pos NULL = camera centre (DESIGN R2).  `what` (ORC_WITH_*) only leaves
 * products out: without ORC_WITH_COLOUR step O5 is skipped, without ORC_WITH_PAIRS the lists of O6 are counted
 * (tile_start is complete) but not stored -- masks, states, geometry and per-tile counts never depend on it. */
orc_frame *orc_frame_create_ex(const orc_scene *sc, const orc_camera *cam, int l_start, int l_end,
                               float gamma, const float *ref_pos, int what)
{
    if (!sc || !cam || l_start < 1 || l_end > sc->L || l_start > l_end || !(gamma > 0.0f)) return NULL;
    orc_frame *fr = (orc_frame *)calloc(1, sizeof(orc_frame));
    fr->sc = sc; fr->cam = *cam; fr->l_start = l_start; fr->l_end = l_end; fr->gamma = gamma; fr->what = what;
    fr->TX = (cam->width + ORC_TILE - 1) / ORC_TILE;
    fr->TY = (cam->height + ORC_TILE - 1) / ORC_TILE;
    const float *R = cam->R, *t = cam->t;
    /* camera centre c = -R^T t, fp64, rounded once */
    for (int i = 0; i < 3; ++i)
        fr->centre[i] = (float)(-(((double)R[i] * (double)t[0] + (double)R[3 + i] * (double)t[1])
                                  + (double)R[6 + i] * (double)t[2]));
    for (int i = 0; i < 3; ++i) fr->ref[i] = ref_pos ? ref_pos[i] : fr->centre[i];
    fr->limx = (float)(1.3 * (double)cam->width / (2.0 * (double)cam->fx));
    fr->limy = (float)(1.3 * (double)cam->height / (2.0 * (double)cam->fy));
    orc_band_thresholds(sc->L, sc->s_min, l_start, l_end, cam->fx, gamma, fr->lo2, fr->hi2);

    int64_t n = sc->n_total, na = n > 0 ? n : 1;
    fr->mask = (uint8_t *)calloc(na, 1);
    fr->state = (uint8_t *)calloc(na, 1);
    fr->mu2d = (float *)calloc(2 * na, sizeof(float));
    fr->depth = (float *)calloc(na, sizeof(float));
    fr->cov2d = (float *)calloc(3 * na, sizeof(float));
    fr->conic = (float *)calloc(3 * na, sizeof(float));
    fr->rect = (int32_t *)calloc(4 * na, sizeof(int32_t));
    fr->n_tiles = (uint32_t *)calloc(na, sizeof(uint32_t));
    fr->rgb = (double *)calloc(3 * na, sizeof(double));
    const int f64 = (what & ORC_FP64) != 0;
    double centre64[3], limx64 = 1.3 * (double)cam->width / (2.0 * (double)cam->fx), limy64 = 1.3 * (double)cam->height / (2.0 * (double)cam->fy);
    for (int i = 0; i < 3; ++i)
        centre64[i] = -(((double)R[i] * (double)t[0] + (double)R[3 + i] * (double)t[1]) + (double)R[6 + i] * (double)t[2]);
    if (f64) {
        fr->mu2d64 = (double *)calloc(2 * na, sizeof(double));
        fr->depth64 = (double *)calloc(na, sizeof(double));
        fr->conic64 = (double *)calloc(3 * na, sizeof(double));
        fr->opacity64 = (double *)calloc(na, sizeof(double));
    }

    int64_t n_sel = 0, n_front = 0, n_vis = 0, n_pairs = 0, n_bf = 0;
    for (int l = l_start; l <= l_end; ++l) {
        int64_t b = sc->offset[l - 1], e = sc->offset[l];
        float lo2 = fr->lo2[l - 1], hi2 = fr->hi2[l - 1];
        fr->n_scan += e - b;
#pragma omp parallel for schedule(static) reduction(+ : n_sel, n_front, n_vis, n_pairs, n_bf)
        for (int64_t g = b; g < e; ++g) {
            if (f64) {      /* O1 in fp64: unrounded thresholds d_proj^2, unrounded camera centre (or the given reference) */
                double dl = (l == l_end) ? 0.0 : (double)sc->s_min[l - 1] * (double)cam->fx / (double)gamma;
                double dh = (l == l_start) ? INFINITY : (double)sc->s_min[l - 2] * (double)cam->fx / (double)gamma;
                double d2 = 0.0;
                for (int i = 0; i < 3; ++i) {
                    double d = (double)sc->mean[3 * g + i] - (ref_pos ? (double)ref_pos[i] : centre64[i]);
                    d2 += d * d;
                }
                if (!(d2 >= dl * dl && d2 < dh * dh)) continue;
            } else if (!select_one(sc->mean + 3 * g, fr->ref, lo2, hi2)) continue;
            fr->mask[g] = 1; n_sel++;
            int st = f64 ? project_one_f64(fr, g, centre64, limx64, limy64) : project_one(fr, g);
            fr->state[g] = (uint8_t)st;
            if (st != ST_CULL_NEAR) n_front++;
            if (st >= ST_EMPTY_RECT) {
                n_bf++;
                if (what & ORC_WITH_COLOUR) orc_sh_color(sc->sh_degree, sc->mean + 3 * g, fr->centre,
                             sc->sh + 3 * (int64_t)sc->K * g, fr->rgb + 3 * g);
            }
            if (st == ST_VISIBLE) { n_vis++; n_pairs += fr->n_tiles[g]; }
        }
    }
    fr->n_sel = n_sel; fr->n_front = n_front; fr->n_vis = n_vis; fr->n_pairs = n_pairs; fr->n_bf = n_bf;

    /* O6: every tile's list = the visible Gaussians whose rect holds the tile, appended in ascending gid, then ordered
     * by (depth, gid) ("in depth order"; DESIGN R15).  The lists are stored tile after tile, so the whole array
     * is in (tile, depth, gid) order -- the same unique sequence one sort of all pairs by that triple gives (the
     * first version of this function did exactly that; per-tile lists sort in parallel and are what O7 walks). */
    fr->pairs = (orc_pair *)malloc(sizeof(orc_pair) * (size_t)(n_pairs > 0 ? n_pairs : 1));
    fr->bf_list = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(n_bf > 0 ? n_bf : 1));
    int T_n = fr->TX * fr->TY;
    fr->tile_start = (uint32_t *)calloc((size_t)T_n + 1, sizeof(uint32_t));
    int64_t q = 0;
    for (int64_t g = 0; g < n; ++g) {
        if (fr->state[g] >= ST_EMPTY_RECT) fr->bf_list[q++] = (uint32_t)g;
        if (fr->state[g] != ST_VISIBLE) continue;
        const int32_t *r = fr->rect + 4 * g;
        uint32_t np = 0;
        for (int ty = r[1]; ty < r[3]; ++ty) {
            int ta, tb;
            if (!row_span(fr, g, ty, &ta, &tb)) continue;
            for (int tx = ta; tx <= tb; ++tx) { fr->tile_start[ty * fr->TX + tx + 1]++; ++np; }
        }
        fr->n_tiles[g] = np;                /* pairs of g (= its rect's area under pair rule 1) */
    }
    for (int tI = 0; tI < T_n; ++tI) fr->tile_start[tI + 1] += fr->tile_start[tI];
    fr->n_pairs = n_pairs = fr->tile_start[T_n];
    if (!(what & ORC_WITH_PAIRS)) return fr;
    uint32_t *fill = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(T_n > 0 ? T_n : 1));
    memcpy(fill, fr->tile_start, sizeof(uint32_t) * (size_t)T_n);
    for (int64_t g = 0; g < n; ++g) {
        if (fr->state[g] != ST_VISIBLE) continue;
        const int32_t *r = fr->rect + 4 * g;
        for (int ty = r[1]; ty < r[3]; ++ty) {
            int ta, tb;
            if (!row_span(fr, g, ty, &ta, &tb)) continue;
            for (int tx = ta; tx <= tb; ++tx) {
                uint32_t tile = (uint32_t)(ty * fr->TX + tx);
                orc_pair *pp = fr->pairs + fill[tile]++;
                pp->tile = tile; pp->depth = fr->depth[g]; pp->gid = (uint32_t)g;
            }
        }
    }
    free(fill);
    g_sort_frame = fr;
#pragma omp parallel for schedule(dynamic, 8)
    for (int tI = 0; tI < T_n; ++tI)
        qsort(fr->pairs + fr->tile_start[tI], (size_t)(fr->tile_start[tI + 1] - fr->tile_start[tI]), sizeof(orc_pair),
              f64 ? cmp_pair64 : cmp_pair);
    return fr;
}

orc_frame *orc_frame_create(const orc_scene *sc, const orc_camera *cam, int l_start, int l_end,
                            float gamma, const float *ref_pos)
{
    return orc_frame_create_ex(sc, cam, l_start, l_end, gamma, ref_pos, ORC_WITH_COLOUR | ORC_WITH_PAIRS);
}

/* accessors */
int orc_frame_tx(const orc_frame *f) { return f->TX; }
int orc_frame_ty(const orc_frame *f) { return f->TY; }
void orc_frame_counts(const orc_frame *f, int64_t out[6])
{
    out[0] = f->n_scan; out[1] = f->n_sel; out[2] = f->n_front; out[3] = f->n_vis; out[4] = f->n_pairs; out[5] = f->n_bf;
}
const uint8_t *orc_frame_mask(const orc_frame *f) { return f->mask; }
const uint8_t *orc_frame_state(const orc_frame *f) { return f->state; }
const float *orc_frame_mu2d(const orc_frame *f) { return f->mu2d; }
const float *orc_frame_depth(const orc_frame *f) { return f->depth; }
const float *orc_frame_cov2d(const orc_frame *f) { return f->cov2d; }
const float *orc_frame_conic(const orc_frame *f) { return f->conic; }
const int32_t *orc_frame_rect(const orc_frame *f) { return f->rect; }
const uint32_t *orc_frame_n_tiles(const orc_frame *f) { return f->n_tiles; }
const double *orc_frame_rgb(const orc_frame *f) { return f->rgb; }
const uint32_t *orc_frame_tile_start(const orc_frame *f) { return f->tile_start; }
const float *orc_frame_thresholds(const orc_frame *f, int which) { return which ? f->hi2 : f->lo2; }
const float *orc_frame_centre(const orc_frame *f) { return f->centre; }
void orc_frame_sorted_pairs(const orc_frame *f, uint32_t *tile, float *depth, uint32_t *gid)
{
    for (int64_t i = 0; i < f->n_pairs; ++i) {
        tile[i] = f->pairs[i].tile; depth[i] = f->pairs[i].depth; gid[i] = f->pairs[i].gid;
    }
}

/* ------------------------------------------------------------------------ O7 compositing --- */

typedef struct { double T, C[3]; uint32_t E, B; int stopped; } pix_state;

/* One Gaussian into one pixel: Eq. 2 with the clamp / skip / stop rules (DESIGN R11,R12).
 * Pixel centre (i+.5, j+.5) (DESIGN R14).  Returns 1 when the pixel has terminated. */
static inline int blend_one(const orc_frame *fr, uint32_t g, double pxc, double pyc,
                            double skip_thr, double stop_thr, pix_state *ps)
{
    double dx, dy, A, B, C, o;
    if (fr->what & ORC_FP64) {
        dx = fr->mu2d64[2 * g] - pxc; dy = fr->mu2d64[2 * g + 1] - pyc;
        A = fr->conic64[3 * g]; B = fr->conic64[3 * g + 1]; C = fr->conic64[3 * g + 2]; o = fr->opacity64[g];
    } else {
        dx = (double)fr->mu2d[2 * g] - pxc; dy = (double)fr->mu2d[2 * g + 1] - pyc;
        A = fr->conic[3 * g]; B = fr->conic[3 * g + 1]; C = fr->conic[3 * g + 2]; o = (double)fr->sc->opacity[g];
    }
    double q = 0.5 * (A * dx * dx + C * dy * dy) + B * dx * dy;
    if (q < 0.0) q = 0.0;
    double alpha = o * exp(-q);
    if (alpha > 0.99) alpha = 0.99;
    ps->E++;
    if (alpha < skip_thr) return 0;
    const double *col = fr->rgb + 3 * (int64_t)g;
    double w = ps->T * alpha;
    ps->C[0] += w * col[0]; ps->C[1] += w * col[1]; ps->C[2] += w * col[2];
    ps->T = ps->T * (1.0 - alpha);
    ps->B++;
    if (ps->T < stop_thr) { ps->stopped = 1; return 1; }
    return 0;
}

/*
 * Composite the frame.  out_rgb is planar [3][H][W] fp64.  skip_thr: alpha below it is skipped
 * (nominal (float)(1/255)); stop_thr: compositing stops after the blend that takes T below it
 * (nominal 1e-4; pass a negative value to never stop).  brute != 0: every pixel visits every
 * Gaussian that survived the z / dead / det culls in global (depth, gid) order, ignoring tile
 * rects; brute == 0: every pixel visits its tile's list.  E, B, Tfin ([H][W]) may be NULL.
 */
void orc_frame_composite(const orc_frame *fr, double skip_thr, double stop_thr, int brute,
                         double *out_rgb, uint32_t *E, uint32_t *Bc, double *Tfin)
{
    int W = fr->cam.width, H = fr->cam.height;
    int T_n = fr->TX * fr->TY;
    if ((fr->what & (ORC_WITH_COLOUR | ORC_WITH_PAIRS)) != (ORC_WITH_COLOUR | ORC_WITH_PAIRS)) {
        for (int64_t i = 0; i < (int64_t)3 * W * H; ++i) out_rgb[i] = NAN;     /* a geometry-only frame has no image */
        return;
    }
    if (brute && !fr->bf_sorted) {            /* global (depth, gid) order, built on first use */
        orc_frame *mf = (orc_frame *)fr;
        g_sort_frame = fr;
        qsort(mf->bf_list, (size_t)mf->n_bf, sizeof(uint32_t), cmp_bf);
        mf->bf_sorted = 1;
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int tile = 0; tile < T_n; ++tile) {
        int tx = tile % fr->TX, ty = tile / fr->TX;
        uint32_t s = fr->tile_start[tile], e = fr->tile_start[tile + 1];
        for (int j = ty * ORC_TILE; j < (ty + 1) * ORC_TILE && j < H; ++j)
            for (int i = tx * ORC_TILE; i < (tx + 1) * ORC_TILE && i < W; ++i) {
                pix_state ps = { 1.0, { 0.0, 0.0, 0.0 }, 0, 0, 0 };
                double pxc = (double)i + 0.5, pyc = (double)j + 0.5;
                if (brute) {
                    for (int64_t k = 0; k < fr->n_bf; ++k)
                        if (blend_one(fr, fr->bf_list[k], pxc, pyc, skip_thr, stop_thr, &ps)) break;
                } else {
                    for (uint32_t k = s; k < e; ++k)
                        if (blend_one(fr, fr->pairs[k].gid, pxc, pyc, skip_thr, stop_thr, &ps)) break;
                }
                int64_t o = (int64_t)j * W + i;
                for (int ch = 0; ch < 3; ++ch)
                    out_rgb[(int64_t)ch * W * H + o] = ps.C[ch] + ps.T * (double)fr->cam.bg[ch];
                if (E) E[o] = ps.E;
                if (Bc) Bc[o] = ps.B;
                if (Tfin) Tfin[o] = ps.T;
            }
    }
}

/* Per-pixel trace of (alpha, T-before) for invariant tests: visits the pixel's tile list and
 * records up to cap blended entries.  Returns the number recorded. */
int orc_frame_trace_pixel(const orc_frame *fr, int i, int j, double skip_thr, double stop_thr,
                          double *alpha_out, double *T_out, int cap)
{
    int tile = (j / ORC_TILE) * fr->TX + (i / ORC_TILE);
    uint32_t s = fr->tile_start[tile], e = fr->tile_start[tile + 1];
    double T = 1.0; int n = 0;
    for (uint32_t k = s; k < e; ++k) {
        uint32_t g = fr->pairs[k].gid;
        double dx = (double)fr->mu2d[2 * g] - ((double)i + 0.5), dy = (double)fr->mu2d[2 * g + 1] - ((double)j + 0.5);
        double A = fr->conic[3 * g], B = fr->conic[3 * g + 1], C = fr->conic[3 * g + 2];
        double q = 0.5 * (A * dx * dx + C * dy * dy) + B * dx * dy;
        if (q < 0.0) q = 0.0;
        double alpha = (double)fr->sc->opacity[g] * exp(-q);
        if (alpha > 0.99) alpha = 0.99;
        if (alpha < skip_thr) continue;
        if (n < cap) { alpha_out[n] = alpha; T_out[n] = T; }
        ++n;
        T *= (1.0 - alpha);
        if (T < stop_thr) break;
    }
    return n;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
