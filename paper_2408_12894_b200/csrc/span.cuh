// Pair rule 2 "ellipse" (DESIGN R26): inside its tile rect a visible Gaussian is listed only in the tiles
// that hold a pixel centre of the padded alpha = 1/255 contour of Eq. 2.  The contour is taken from the
// factorised exponent the blend evaluates (DESIGN R25; the per-Gaussian blend features gA, gB of flod_internal.cuh):
//     log2 alpha = log2 o + a2 w^2 + d2 dy^2,   w = dx + k dy,   a2, d2 <= 0      =>      a w^2 + d dy^2 = E,
//     a = -a2,  d = -d2,  E = log2 o + log2 255.
// A tile row's pixel centres are the band y in [16 ty + .5, 16 ty + 15.5]; the ellipse cut by a band is convex, so the
// listed tiles of a row are ONE span [ta, tb].  For a fixed dy the ellipse is x - mu'x in [sl dy - s(dy), sl dy + s(dy)],
// sl = -k, s(dy)^2 = KA - DA dy^2, KA = E/a, DA = d/a; the right end is concave in dy with its maximum at the ellipse's
// rightmost point dy = dyt, so over the band it is largest at clamp(dyt, band), the left end smallest at clamp(-dyt, band).
// Arithmetic: canonical fp32, as in k_geometry -- every operation is one IEEE binary32 round-to-nearest operation in the
// written order (the *_rn intrinsics are never contracted), so the integer spans equal the oracle's bit for bit.  k, a2,
// d2 were derived from the rounded conic in fp64 (C - B^2/A cancels for thin diagonal footprints) and rounded once, so
// nothing cancels here except s^2 near the ellipse's tips: the ends are padded (DESIGN R26 has the estimate).
// No storage of its own: the inputs are the 24 bytes of blend features the duplication kernels read anyway.
#pragma once
#include <cuda_runtime.h>

namespace flod {

struct SpanCoef { float sl, KA, DA, dyt, pad, mx, my; bool box; };

__device__ __forceinline__ SpanCoef span_coefficients(float mx, float my, float k, float a2, float d2, float l2o)
{
    SpanCoef c;
    c.mx = mx; c.my = my;
    const float a = -a2, d = -d2;
    c.box = !(a > 0.0f);                                  // not an ellipse after rounding: every tile of the rect
    const float E = __fadd_rn(__fmul_rn(__fadd_rn(l2o, 7.994353436858858f), 1.001953125f), 0.0000152587890625f);
    c.sl = -k;
    const float ra = __fdiv_rn(1.0f, a);
    c.KA = __fmul_rn(E, ra);
    c.DA = __fmul_rn(d, ra);
    if (c.DA > 0.0f) c.dyt = -__fmul_rn(k, __fsqrt_rn(__fdiv_rn(c.KA, __fmul_rn(c.DA, __fadd_rn(c.DA, __fmul_rn(k, k))))));
    else c.dyt = k < 0.0f ? __int_as_float(0x7f800000) : (k > 0.0f ? __int_as_float(0xff800000) : 0.0f);   // a strip
    c.pad = __fadd_rn(__fmul_rn(__fsqrt_rn(c.KA), 0.00390625f), 0.015625f);
    return c;
}

// Tiles [ta, tb] (inclusive) of tile row ty that the Gaussian is listed in, clipped to the columns [tx0, tx1) of its
// rect; returns their number (0: none).
__device__ __forceinline__ int span_of_row(const SpanCoef &c, int tx0, int tx1, int ty, int *ta_out, int *tb_out)
{
    *ta_out = tx0; *tb_out = tx1 - 1;
    if (c.box) return tx1 - tx0;
    const float y0 = __fsub_rn(__fadd_rn((float)(16 * ty), 0.5f), c.my), y1 = __fadd_rn(y0, 15.0f);
    const float dn = fminf(fmaxf(0.0f, y0), y1);
    if (__fmul_rn(c.DA, __fmul_rn(dn, dn)) > __fmul_rn(c.KA, 1.001953125f)) return 0;      // the band misses the ellipse
    const float dh = fminf(fmaxf(c.dyt, y0), y1), dl = fminf(fmaxf(-c.dyt, y0), y1);
    const float sh = __fsqrt_rn(fmaxf(0.0f, __fsub_rn(c.KA, __fmul_rn(c.DA, __fmul_rn(dh, dh)))));
    const float sq = __fsqrt_rn(fmaxf(0.0f, __fsub_rn(c.KA, __fmul_rn(c.DA, __fmul_rn(dl, dl)))));
    const float ch = __fmul_rn(c.sl, dh), cl = __fmul_rn(c.sl, dl);
    const float padr = __fadd_rn(c.pad, __fmul_rn(__fadd_rn(__fadd_rn(fabsf(c.mx), fabsf(ch)), fabsf(cl)), 9.5367431640625e-7f));
    const float xh = __fadd_rn(__fadd_rn(c.mx, __fadd_rn(ch, sh)), padr);
    const float xl = __fsub_rn(__fadd_rn(c.mx, __fsub_rn(cl, sq)), padr);
    const float ta = fmaxf(ceilf(__fmul_rn(__fsub_rn(xl, 15.5f), 0.0625f)), (float)tx0);
    const float tb = fminf(floorf(__fmul_rn(__fsub_rn(xh, 0.5f), 0.0625f)), (float)(tx1 - 1));
    if (!(tb >= ta)) return 0;
    *ta_out = (int)ta; *tb_out = (int)tb;
    return (int)tb - (int)ta + 1;
}

}  // namespace flod
