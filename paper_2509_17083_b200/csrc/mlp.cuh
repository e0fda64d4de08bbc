// mlp.cuh — the tiny decoder MLP on CUDA cores (DESIGN.md §2 D5; "2 hidden layers, 64 neurons").
#pragma once
#include "common.cuh"

// One decoder: in[IN] -> hidden x NH (ReLU) -> out[OUT]. Weights in shared memory as fp32, row-major [out][in].
// CIN/CHID/CNH > 0: compile-time shapes, fully unrolled, activations in registers. 0: run-time shapes.
template <int CIN, int CHID, int CNH, int OUT, bool FP16>
__device__ __forceinline__ void mlp_eval(const float* __restrict__ w, int rin, int rhid, int rnh, float* a,
                                         float* b, float* out) {
    const int IN = CIN > 0 ? CIN : rin;
    const int HID = CHID > 0 ? CHID : rhid;
    const int NH = CNH > 0 ? CNH : rnh;
    int cur = IN;
    float* src = a;
    float* dst = b;
#pragma unroll
    for (int layer = 0; layer < NH; ++layer) {
#pragma unroll
        for (int j = 0; j < HID; ++j) {
            float acc = 0.0f;
#pragma unroll
            for (int k = 0; k < cur; ++k) acc = __fmaf_rn(w[j * cur + k], src[k], acc);
            acc = fmaxf(acc, 0.0f);
            dst[j] = FP16 ? hy_round_half(acc) : acc;
        }
        w += HID * cur;
        cur = HID;
        float* t = src; src = dst; dst = t;
    }
#pragma unroll
    for (int j = 0; j < OUT; ++j) {
        float acc = 0.0f;
#pragma unroll
        for (int k = 0; k < cur; ++k) acc = __fmaf_rn(w[j * cur + k], src[k], acc);
        out[j] = acc;
    }
}

