// common.cuh — device-side definitions shared by the HyRF kernels (sm_100a).
// Written from DESIGN.md §2 (which restates PAPER.md §3.2–3.3, A.1–A.2). Shares nothing with oracle/.
// Compile with -fmad=false: every fused multiply-add below is explicit, so rounding points are the documented ones.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#define HY_MAX_LEVELS 16
#define HY_TILE 16
#ifndef HY_MACRO_SHIFT
#define HY_MACRO_SHIFT 2                  // binning granularity: 4 x 4 tiles (64 x 64 pixels) per macro tile
#endif
#define HY_MACRO (1 << HY_MACRO_SHIFT)
#define HY_REC_F4 3  // projected record = 3 x float4: (u, v, A, B) (C, opacity, r, g) (b, depth, radius, tiles)

// One multi-resolution grid as the kernels see it (DESIGN.md §2 D3).
struct GridDev {
    const void* table;               // [entries][2], float2, __half2 or uchar2 (8-bit min-max codes)
    uint32_t levels;
    uint32_t table_mask;             // T - 1
    uint32_t dense_mask;             // bit l set: level l is dense
    uint32_t res[HY_MAX_LEVELS];     // N_l
    uint32_t offset[HY_MAX_LEVELS];  // first entry of level l
    float2 q[HY_MAX_LEVELS][2];      // 8-bit tables only: (min, step) of level l, feature f (DESIGN.md §2 D3')
};

// Camera plus the per-frame constants derived from it on the host (DESIGN.md §2 "Camera", D1).
struct FrameDev {
    float R[9], t[3];
    float fx, fy, cx, cy;
    float o[3];         // camera centre -R^T t
    float limx, limy;   // (1 + tol) * W / (2 fx), (1 + tol) * H / (2 fy)
    float z_near, tau_T, bg_radius;
    float aabb_c[3], aabb_h[3];
    int32_t W, H, gx, gy;
    int32_t mshift;     // binning granularity of this frame: macro tile = 2^mshift x 2^mshift tiles (0 on small grids)
    int32_t mgx, mgy;   // macro-tile grid
    uint32_t ablation;  // hyrf_ablation bits (include/hyrf.h)
    int32_t ty0, ty1;   // tile rows [ty0, ty1) this device bins, rasterises and composites (hyrf_set_strip); 0, gy = the whole image
};

// D6 soft exponential: the one exp behind every sigmoid, so geometry decisions are bit-reproducible.
__device__ __forceinline__ float hy_softexp(float x) {
    x = fminf(fmaxf(x, -87.0f), 88.0f);
    float n = rintf(__fmul_rn(x, 1.44269504f));
    float r = __fmaf_rn(n, -0.693145752f, x);
    r = __fmaf_rn(n, -1.42860677e-6f, r);
    float p = 1.98412701e-4f;
    p = __fmaf_rn(p, r, 1.38888892e-3f);
    p = __fmaf_rn(p, r, 8.33333377e-3f);
    p = __fmaf_rn(p, r, 4.16666679e-2f);
    p = __fmaf_rn(p, r, 1.66666672e-1f);
    p = __fmaf_rn(p, r, 0.5f);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    int ni = (int)n;
    float s = __int_as_float((ni + 127) << 23);
    return __fmul_rn(p, s);
}

__device__ __forceinline__ float hy_sigmoid(float v) {
    return __fdiv_rn(1.0f, __fadd_rn(1.0f, hy_softexp(-v)));
}

// D1: world point -> camera space.
__device__ __forceinline__ void hy_to_camera(const FrameDev& f, float px, float py, float pz, float& X, float& Y,
                                             float& Z) {
    X = __fmaf_rn(f.R[2], pz, __fmaf_rn(f.R[1], py, __fmaf_rn(f.R[0], px, f.t[0])));
    Y = __fmaf_rn(f.R[5], pz, __fmaf_rn(f.R[4], py, __fmaf_rn(f.R[3], px, f.t[1])));
    Z = __fmaf_rn(f.R[8], pz, __fmaf_rn(f.R[7], py, __fmaf_rn(f.R[6], px, f.t[2])));
}

// D2 contraction into [0,1]^3 (Eq. 2 / 14 with the 0.5 offset of reading A1).
__device__ __forceinline__ void hy_contract(const FrameDev& f, float px, float py, float pz, float x[3]) {
    float q0 = __fdiv_rn(__fsub_rn(px, f.aabb_c[0]), f.aabb_h[0]);
    float q1 = __fdiv_rn(__fsub_rn(py, f.aabb_c[1]), f.aabb_h[1]);
    float q2 = __fdiv_rn(__fsub_rn(pz, f.aabb_c[2]), f.aabb_h[2]);
    float n2 = __fmaf_rn(q2, q2, __fmaf_rn(q1, q1, __fmul_rn(q0, q0)));
    float n = __fsqrt_rn(n2);
    if (!(n <= 1.0f)) {
        float inv = __fdiv_rn(1.0f, n);
        float sc = __fmul_rn(__fsub_rn(2.0f, inv), inv);
        q0 = __fmul_rn(sc, q0);
        q1 = __fmul_rn(sc, q1);
        q2 = __fmul_rn(sc, q2);
    }
    x[0] = fminf(fmaxf(__fmaf_rn(0.25f, q0, 0.5f), 0.0f), 1.0f);
    x[1] = fminf(fmaxf(__fmaf_rn(0.25f, q1, 0.5f), 0.0f), 1.0f);
    x[2] = fminf(fmaxf(__fmaf_rn(0.25f, q2, 0.5f), 0.0f), 1.0f);
}

// Table entry types: DT 0 = fp32, 1 = fp16, 2 = 8-bit min-max codes (decoders fp16).
#define HY_DT_F32 0
#define HY_DT_F16 1
#define HY_DT_U8 2

// D3: one level of one grid at contracted position x -> two features (fp32, not yet rounded to half).
template <int DT>
__device__ __forceinline__ void hy_grid_level(const GridDev& g, uint32_t l, const float x[3], float& f0, float& f1) {
    const uint32_t N = g.res[l];
    const float Nf = (float)N;
    uint32_t ci[3];
    float w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float u = __fmul_rn(x[a], Nf);
        int i = (int)floorf(u);
        i = min(i, (int)N - 1);
        ci[a] = (uint32_t)i;
        w[a] = __fsub_rn(u, (float)i);
    }
    const bool dense = (g.dense_mask >> l) & 1u;
    const uint32_t n1 = N + 1u;
    uint32_t idx[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        uint32_t vx = ci[0] + (k & 1), vy = ci[1] + ((k >> 1) & 1), vz = ci[2] + ((k >> 2) & 1);
        uint32_t e = dense ? (vx + n1 * (vy + n1 * vz))
                           : ((vx ^ (vy * 2654435761u) ^ (vz * 805459861u)) & g.table_mask);
        idx[k] = g.offset[l] + e;
    }
    float v0[8], v1[8];
    if (DT == HY_DT_U8) {   // D3': value = fma(code, step, min)
        const uchar2* tab = reinterpret_cast<const uchar2*>(g.table);
        const float2 q0 = g.q[l][0], q1 = g.q[l][1];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uchar2 c = __ldg(tab + idx[k]);
            v0[k] = __fmaf_rn((float)c.x, q0.y, q0.x);
            v1[k] = __fmaf_rn((float)c.y, q1.y, q1.x);
        }
    } else if (DT == HY_DT_F16) {
        const __half2* tab = reinterpret_cast<const __half2*>(g.table);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float2 v = __half22float2(__ldg(tab + idx[k]));
            v0[k] = v.x;
            v1[k] = v.y;
        }
    } else {
        const float2* tab = reinterpret_cast<const float2*>(g.table);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            float2 v = __ldg(tab + idx[k]);
            v0[k] = v.x;
            v1[k] = v.y;
        }
    }
    const float wx1 = w[0], wx0 = __fsub_rn(1.0f, w[0]);
    const float wy1 = w[1], wy0 = __fsub_rn(1.0f, w[1]);
    const float wz1 = w[2], wz0 = __fsub_rn(1.0f, w[2]);
    float a0 = 0.0f, a1 = 0.0f;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float wt = __fmul_rn(__fmul_rn((k & 1) ? wx1 : wx0, (k & 2) ? wy1 : wy0), (k & 4) ? wz1 : wz0);
        a0 = __fmaf_rn(wt, v0[k], a0);
        a1 = __fmaf_rn(wt, v1[k], a1);
    }
    f0 = a0;
    f1 = a1;
}

__device__ __forceinline__ float hy_round_half(float v) { return __half2float(__float2half_rn(v)); }

// D4: direction encoding of a unit vector, 6 values per octave: sin(pi 2^k d_a) then cos(pi 2^k d_a).
template <bool FP16>
__device__ __forceinline__ void hy_dir_pe(const float d[3], int octaves, float* out) {
    for (int k = 0; k < octaves; ++k) {
        float sc = (float)(1u << k);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float s, c;
            sincospif(__fmul_rn(sc, d[a]), &s, &c);
            out[6 * k + a] = FP16 ? hy_round_half(s) : s;
            out[6 * k + 3 + a] = FP16 ? hy_round_half(c) : c;
        }
    }
}

#define HY_CUDA_OK(expr)                                  \
    do {                                                  \
        cudaError_t _e = (expr);                          \
        if (_e != cudaSuccess) return hy_cuda_fail(_e, #expr); \
    } while (0)
