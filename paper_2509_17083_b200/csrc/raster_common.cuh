// raster_common.cuh — pieces shared by the forward rasterizers (raster.cu, raster_warp.cu) and the backward of S5
// (raster_backward.cu): the reach test of a list entry against a pixel box and the MUFU exp2 of D10.
#pragma once
#include "common.cuh"

// Can list entry (mean (u, v), conic (A, B, C), opacity o) reach alpha >= 1/255 at ANY pixel of the tile
// [X0, X1] x [Y0, Y1]? The quadratic form q = A dx^2 + 2 B dx dy + C dy^2 is convex, so its minimum over the pixel box
// is 0 when the mean lies inside, else it sits on a face whose plane separates the mean from the box: at most two
// one-dimensional minimisations. alpha <= o exp(-q_min / 2) everywhere in the tile; entries below the threshold
// would be skipped by every pixel, so dropping them changes no output bit — PROVIDED the comparison allows for the
// rounding of both sides: this q_min and every pixel's own `power` are binary32 sums of three terms that cancel on
// long thin splats (near-degenerate conic: A ex^2 ~ 1e5-1e6 against q ~ 10), each off by a few ulp of its largest
// term. hy_q_slack bounds the terms over the whole box (any pixel's |dx| <= max(|X0-u|, |X1-u|), same for dy) and
// allows 16 ulp of that sum, on top of a fixed 1 % margin on alpha (0.02 in q) for the MUFU exp / log.
__device__ __forceinline__ float hy_q_slack(float u, float v, float A, float B, float C, float X0, float X1, float Y0,
                                            float Y1) {
    const float mx = fmaxf(fabsf(X0 - u), fabsf(X1 - u)), my = fmaxf(fabsf(Y0 - v), fabsf(Y1 - v));
    return 2.0e-6f * (A * mx * mx + 2.0f * fabsf(B) * mx * my + C * my * my);
}

__device__ __forceinline__ bool entry_reaches_tile(float u, float v, float A, float B, float C, float o, float X0,
                                                   float X1, float Y0, float Y1) {
    const float ex = fminf(fmaxf(u, X0), X1) - u, ey = fminf(fmaxf(v, Y0), Y1) - v;
    if (ex == 0.0f && ey == 0.0f) return true;
    float qmin = 3.0e38f;
    if (ex != 0.0f) {
        const float dy = fminf(fmaxf(__fdividef(-B * ex, C), Y0 - v), Y1 - v);
        qmin = A * ex * ex + 2.0f * B * ex * dy + C * dy * dy;
    }
    if (ey != 0.0f) {
        const float dx = fminf(fmaxf(__fdividef(-B * ey, A), X0 - u), X1 - u);
        qmin = fminf(qmin, A * dx * dx + 2.0f * B * dx * ey + C * ey * ey);
    }
    qmin -= hy_q_slack(u, v, A, B, C, X0, X1, Y0, Y1);
    return !(o * __expf(-0.5f * qmin) < 0.99f / 255.0f);   // NaN keeps the entry
}

// The same test for a sub-rectangle of the tile, with the per-entry work hoisted: iA = 1 / A, iC = 1 / C,
// qthr = 2 ln(o * 255 / 0.99) + the tile's hy_q_slack (alpha >= 0.99 / 255  <=>  q <= 2 ln(o 255 / 0.99)). NaN keeps the entry.
__device__ __forceinline__ bool entry_reaches_block(float u, float v, float A, float B, float C, float iA, float iC,
                                                    float qthr, float X0, float X1, float Y0, float Y1) {
    const float ex = fminf(fmaxf(u, X0), X1) - u, ey = fminf(fmaxf(v, Y0), Y1) - v;
    if (ex == 0.0f && ey == 0.0f) return true;
    float qmin = 3.0e38f;
    if (ex != 0.0f) {
        const float dy = fminf(fmaxf(-B * ex * iC, Y0 - v), Y1 - v);
        qmin = A * ex * ex + 2.0f * B * ex * dy + C * dy * dy;
    }
    if (ey != 0.0f) {
        const float dx = fminf(fmaxf(-B * ey * iA, X0 - u), X1 - u);
        qmin = fminf(qmin, A * dx * dx + 2.0f * B * dx * ey + C * ey * ey);
    }
    return !(qmin > qthr);
}

// exp2 on the MUFU, flushing subnormal results to 0 (they are far below the 1/255 skip threshold anyway)
__device__ __forceinline__ float ex2_ftz(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Which of the eight 8 x 4 pixel blocks (block w: columns (w & 1) * 8 .., rows (w >> 1) * 4 ..) of the 16 x 16 tile at
// (X0, Y0) can the entry reach with alpha >= 1/255? Blocks outside the W x H image are never set (nobody blends there).
__device__ __forceinline__ uint32_t entry_block_mask(float u, float v, float A, float B, float C, float o, float X0,
                                                     float Y0, int W, int H) {
    const float iA = __fdividef(1.0f, A), iC = __fdividef(1.0f, C);
    const float qthr = 2.0f * __logf(o * (255.0f / 0.99f)) +
                       hy_q_slack(u, v, A, B, C, X0, fminf(X0 + 15.0f, (float)(W - 1)), Y0, fminf(Y0 + 15.0f, (float)(H - 1)));
    uint32_t m = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) {
        const float bx0 = X0 + (float)((w & 1) * 8), by0 = Y0 + (float)((w >> 1) * 4);
        const float bx1 = fminf(bx0 + 7.0f, (float)(W - 1)), by1 = fminf(by0 + 3.0f, (float)(H - 1));
        const bool in_img = bx0 <= (float)(W - 1) && by0 <= (float)(H - 1);
        if (in_img && entry_reaches_block(u, v, A, B, C, iA, iC, qthr, bx0, bx1, by0, by1)) m |= 1u << w;
    }
    return m;
}

// The same for the four 8 x 8 pixel blocks of the tile (block w: columns (w & 1) * 8 .., rows (w >> 1) * 8 ..): what the
// two-pixels-per-lane rasterizer (raster_pair.cu) needs, at half the tests.
__device__ __forceinline__ uint32_t entry_block_mask4(float u, float v, float A, float B, float C, float o, float X0,
                                                      float Y0, int W, int H) {
    const float iA = __fdividef(1.0f, A), iC = __fdividef(1.0f, C);
    const float qthr = 2.0f * __logf(o * (255.0f / 0.99f)) +
                       hy_q_slack(u, v, A, B, C, X0, fminf(X0 + 15.0f, (float)(W - 1)), Y0, fminf(Y0 + 15.0f, (float)(H - 1)));
    uint32_t m = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const float bx0 = X0 + (float)((w & 1) * 8), by0 = Y0 + (float)((w >> 1) * 8);
        const float bx1 = fminf(bx0 + 7.0f, (float)(W - 1)), by1 = fminf(by0 + 7.0f, (float)(H - 1));
        const bool in_img = bx0 <= (float)(W - 1) && by0 <= (float)(H - 1);
        if (in_img && entry_reaches_block(u, v, A, B, C, iA, iC, qthr, bx0, bx1, by0, by1)) m |= 1u << w;
    }
    return m;
}
