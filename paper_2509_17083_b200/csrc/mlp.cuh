// mlp.cuh — the tiny decoder MLP on CUDA cores (DESIGN.md §2 D5; "2 hidden layers, 64 neurons").
#pragma once
#include "common.cuh"

// One neuron: acc = fma(w[k], h[k], acc), k ascending (D5's order). VEC: the row is 16-byte aligned and a multiple of
// 4 long (compile-time shapes: rows of 32 / 40 / 56 / 64 floats in a 16-byte aligned block), so the weights come as
// broadcast LDS.128 — a quarter of the shared-memory instructions of the scalar form, same arithmetic.
template <bool VEC>
__device__ __forceinline__ float mlp_dot(const float* __restrict__ w, const float* h, int n) {
    float acc = 0.0f;
    if (VEC) {
        const float4* w4 = reinterpret_cast<const float4*>(w);
#pragma unroll
        for (int k = 0; k < n / 4; ++k) {
            const float4 q = w4[k];
            acc = __fmaf_rn(q.x, h[4 * k], acc);
            acc = __fmaf_rn(q.y, h[4 * k + 1], acc);
            acc = __fmaf_rn(q.z, h[4 * k + 2], acc);
            acc = __fmaf_rn(q.w, h[4 * k + 3], acc);
        }
    } else {
#pragma unroll
        for (int k = 0; k < n; ++k) acc = __fmaf_rn(w[k], h[k], acc);
    }
    return acc;
}

// One decoder: in[IN] -> hidden x NH (ReLU) -> out[OUT]. Weights in shared memory as fp32, row-major [out][in].
// CIN/CHID/CNH > 0: compile-time shapes, fully unrolled, activations in registers. 0: run-time shapes.
template <int CIN, int CHID, int CNH, int OUT, bool FP16>
__device__ __forceinline__ void mlp_eval(const float* __restrict__ w, int rin, int rhid, int rnh, float* a,
                                         float* b, float* out) {
    if (CIN > 0 && CHID > 0 && CNH == 1) {
        // one hidden layer, compile-time shapes: each hidden activation is consumed by the output neurons as soon as
        // it exists, so the hidden vector never occupies registers. Every output still accumulates its inputs in
        // ascending order, one fma at a time: same bits as the layer-by-layer form below.
        const float* w2 = w + CHID * CIN;
        float acc[OUT];
#pragma unroll
        for (int c = 0; c < OUT; ++c) acc[c] = 0.0f;
        static_assert(CHID % 4 == 0 && CIN % 4 == 0, "compile-time decoder shapes are multiples of 4");
#pragma unroll
        for (int j = 0; j < CHID; j += 4) {
            // four hidden neurons at a time: four independent fma chains over the same activations hide the fma and
            // shared-memory latencies at the few warps per SM this kernel has; each chain is still k ascending
            const float4* r0 = reinterpret_cast<const float4*>(w + (j + 0) * CIN);
            const float4* r1 = reinterpret_cast<const float4*>(w + (j + 1) * CIN);
            const float4* r2 = reinterpret_cast<const float4*>(w + (j + 2) * CIN);
            const float4* r3 = reinterpret_cast<const float4*>(w + (j + 3) * CIN);
            float h[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
            for (int k = 0; k < CIN / 4; ++k) {
                const float4 q0 = r0[k], q1 = r1[k], q2 = r2[k], q3 = r3[k];
                const float x0 = a[4 * k], x1 = a[4 * k + 1], x2 = a[4 * k + 2], x3 = a[4 * k + 3];
                h[0] = __fmaf_rn(q0.x, x0, h[0]); h[1] = __fmaf_rn(q1.x, x0, h[1]); h[2] = __fmaf_rn(q2.x, x0, h[2]); h[3] = __fmaf_rn(q3.x, x0, h[3]);
                h[0] = __fmaf_rn(q0.y, x1, h[0]); h[1] = __fmaf_rn(q1.y, x1, h[1]); h[2] = __fmaf_rn(q2.y, x1, h[2]); h[3] = __fmaf_rn(q3.y, x1, h[3]);
                h[0] = __fmaf_rn(q0.z, x2, h[0]); h[1] = __fmaf_rn(q1.z, x2, h[1]); h[2] = __fmaf_rn(q2.z, x2, h[2]); h[3] = __fmaf_rn(q3.z, x2, h[3]);
                h[0] = __fmaf_rn(q0.w, x3, h[0]); h[1] = __fmaf_rn(q1.w, x3, h[1]); h[2] = __fmaf_rn(q2.w, x3, h[2]); h[3] = __fmaf_rn(q3.w, x3, h[3]);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                float v = fmaxf(h[i], 0.0f);
                if (FP16) v = hy_round_half(v);
#pragma unroll
                for (int c = 0; c < OUT; ++c) acc[c] = __fmaf_rn(w2[c * CHID + j + i], v, acc[c]);
            }
        }
#pragma unroll
        for (int c = 0; c < OUT; ++c) out[c] = acc[c];
        return;
    }
    const int IN = CIN > 0 ? CIN : rin;
    const int HID = CHID > 0 ? CHID : rhid;
    const int NH = CNH > 0 ? CNH : rnh;
    int cur = IN;
    float* src = a;
    float* dst = b;
#pragma unroll
    for (int layer = 0; layer < NH; ++layer) {
#pragma unroll
        for (int j = 0; j < HID; ++j) dst[j] = fmaxf(mlp_dot<(CIN > 0 && CHID > 0)>(w + j * cur, src, cur), 0.0f);
        if (FP16) {
#pragma unroll
            for (int j = 0; j < HID; ++j) dst[j] = hy_round_half(dst[j]);
        }
        w += HID * cur;
        cur = HID;
        float* t = src; src = dst; dst = t;
    }
#pragma unroll
    for (int j = 0; j < OUT; ++j) out[j] = mlp_dot<(CIN > 0 && CHID > 0)>(w + j * cur, src, cur);
}


// One dense layer with compile-time sizes as a LOOP over groups of four neurons (not unrolled over the neurons): the
// layer's inputs in registers, weight rows as 16-byte shared-memory loads, out[j] = act(sum_k w[j][k] in[k]) with k
// ascending — D5's order, the bits of mlp_dot. `in` / `out` may be local arrays (indexed by the neuron at run time).
// Unrolling a whole 64-wide decoder over its neurons (mlp_eval above with CNH = 2) makes ~20 k instructions of
// straight-line code: longer than the instruction cache, and with a dozen warps per SM at different places in it the
// kernel waits for instruction fetches (`no_instruction` 9.5 of 12 warps at config 2). This form is ~300 instructions
// per layer.
template <bool FP16, int NIN, bool RELU, int NJ>
__device__ __forceinline__ void mlp_dense_ct(const float* __restrict__ w, const float* in, float* out) {
    float x[NIN];
#pragma unroll
    for (int k = 0; k < NIN; ++k) x[k] = in[k];
    static_assert(NIN % 4 == 0, "rows are read 16 bytes at a time");
    constexpr int G = NJ % 4 == 0 ? 4 : 1;   // neurons per step
#pragma unroll 1
    for (int j = 0; j < NJ; j += G) {
        float h[G];
#pragma unroll
        for (int u = 0; u < G; ++u) h[u] = 0.0f;
#pragma unroll
        for (int k = 0; k < NIN / 4; ++k) {
#pragma unroll
            for (int u = 0; u < G; ++u) {
                const float4 q = reinterpret_cast<const float4*>(w + (j + u) * NIN)[k];
                h[u] = fmaf(q.x, x[4 * k], h[u]);
                h[u] = fmaf(q.y, x[4 * k + 1], h[u]);
                h[u] = fmaf(q.z, x[4 * k + 2], h[u]);
                h[u] = fmaf(q.w, x[4 * k + 3], h[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < G; ++u) {
            float v = h[u];
            if (RELU) { v = fmaxf(v, 0.0f); if (FP16) v = hy_round_half(v); }
            out[j + u] = v;
        }
    }
}

