// field_common.cuh — argument block and the S3 + S4a tail (aggregation Eq. 7, EWA projection) shared by the two
// field kernels (field.cu: fp32 FMA decoders; field_mma.cu: fp16 tensor-core decoders). DESIGN.md §2 D7, D8.
#pragma once
#include "scene.h"

struct FieldArgs {
    GridDev geo, app;
    MlpDev geo_mlp, app_mlp;
    FrameDev f;
    const float4* gm;          // [N][2] Morton-ordered (pos.xyz, scale | opacity, rgb)
    const uint32_t* gm_id;     // [N] id of the m-th Morton record
    const uint32_t* vis_m;     // [V] Morton indices of the visible Gaussians, ascending
    const uint32_t* id_words;  // visibility bits by id
    const uint32_t* word_rank; // visible rank of the first bit of each id word
    uint32_t N;
    uint32_t pe_octaves;
    FrameCounters* counters;
    float4* rec;
    uint4* rect;
    uint32_t* tiles;
    uint32_t* mtiles;
    float* dbg_raw;
    float* dbg_attrs;
};

void hy_fill_field_args(hyrf_scene* s, const FrameDev& f, FieldArgs* out);

// One visible Gaussian of the work list: its explicit parameters (Morton record) and its visible rank j in id order,
// the slot of every per-Gaussian output (j = rank of the first bit of its id word + set bits below it).
struct Explicit { float px, py, pz, s_e, a_e, c_e0, c_e1, c_e2; uint32_t j; };

static __device__ __forceinline__ Explicit fetch_visible(const FieldArgs& A, uint32_t work_index) {
    const uint32_t m = __ldg(A.vis_m + work_index);
    const float4 a = __ldg(A.gm + 2ull * m), b = __ldg(A.gm + 2ull * m + 1);
    const uint32_t id = __ldg(A.gm_id + m);
    Explicit e;
    e.px = a.x; e.py = a.y; e.pz = a.z; e.s_e = a.w;
    e.a_e = b.x; e.c_e0 = b.y; e.c_e1 = b.z; e.c_e2 = b.w;
    if (A.f.ablation & HYRF_ABL_NO_EXPLICIT) e.s_e = e.a_e = e.c_e0 = e.c_e1 = e.c_e2 = 0.0f;
    e.j = __ldg(A.word_rank + (id >> 5)) + __popc(__ldg(A.id_words + (id >> 5)) & ((1u << (id & 31u)) - 1u));
    return e;
}

// sigmoid for the tensor-core path: MUFU exp2 + MUFU reciprocal (2-ulp class). That path is compared with the oracle
// by tolerance and its decoder outputs already carry ~1e-4 of accumulation-order noise, so the soft
// exponential and IEEE division of D6 — there for bit-reproducible geometry — buy nothing on it.
static __device__ __forceinline__ float sigmoid_fast(float v) {
    return __fdividef(1.0f, 1.0f + __expf(-v));
}

// D7 + D8 for one Gaussian. raw = (alpha_n, s_n[3], r_n[4], c_n[3]). FAST: tensor-core path arithmetic (see above).
template <bool FAST>
static __device__ __forceinline__ void aggregate_project(const FieldArgs& A, const Explicit& ex, const float* raw) {
    const FrameDev& f = A.f;
    const uint32_t j = ex.j;
    const float px = ex.px, py = ex.py, pz = ex.pz;
    const float s_e = ex.s_e, a_e = ex.a_e;
    const float c_e0 = ex.c_e0, c_e1 = ex.c_e1, c_e2 = ex.c_e2;
    // Eq. 7
    float s0, s1, s2, w, x, y, z, alpha, c0, c1, c2;
    if (FAST) {
        s0 = sigmoid_fast(raw[1] + s_e); s1 = sigmoid_fast(raw[2] + s_e); s2 = sigmoid_fast(raw[3] + s_e);
        const float m2 = raw[7] * raw[7] + raw[6] * raw[6] + raw[5] * raw[5] + raw[4] * raw[4];
        const float inv = rsqrtf(fmaxf(m2, 1e-24f));
        w = raw[4] * inv; x = raw[5] * inv; y = raw[6] * inv; z = raw[7] * inv;
        alpha = sigmoid_fast(raw[0] + a_e);
        c0 = sigmoid_fast(raw[8] + c_e0); c1 = sigmoid_fast(raw[9] + c_e1); c2 = sigmoid_fast(raw[10] + c_e2);
    } else {
        s0 = hy_sigmoid(__fadd_rn(raw[1], s_e));
        s1 = hy_sigmoid(__fadd_rn(raw[2], s_e));
        s2 = hy_sigmoid(__fadd_rn(raw[3], s_e));
        const float m = __fsqrt_rn(__fmaf_rn(raw[7], raw[7], __fmaf_rn(raw[6], raw[6], __fmaf_rn(raw[5], raw[5], __fmul_rn(raw[4], raw[4])))));
        const float den = fmaxf(m, 1e-12f);
        w = __fdiv_rn(raw[4], den); x = __fdiv_rn(raw[5], den); y = __fdiv_rn(raw[6], den); z = __fdiv_rn(raw[7], den);
        alpha = hy_sigmoid(__fadd_rn(raw[0], a_e));
        c0 = hy_sigmoid(__fadd_rn(raw[8], c_e0));
        c1 = hy_sigmoid(__fadd_rn(raw[9], c_e1));
        c2 = hy_sigmoid(__fadd_rn(raw[10], c_e2));
    }
    if (A.dbg_raw) {
        for (int k = 0; k < 11; ++k) A.dbg_raw[11ull * j + k] = raw[k];
    }
    if (A.dbg_attrs) {
        float* o = A.dbg_attrs + 11ull * j;
        o[0] = s0; o[1] = s1; o[2] = s2; o[3] = w; o[4] = x; o[5] = y; o[6] = z; o[7] = alpha; o[8] = c0; o[9] = c1; o[10] = c2;
    }
    // D8
    float M[9];
    M[0] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(y, y, __fmul_rn(z, z))));
    M[1] = __fmul_rn(2.0f, __fmaf_rn(x, y, -__fmul_rn(w, z)));
    M[2] = __fmul_rn(2.0f, __fmaf_rn(x, z, __fmul_rn(w, y)));
    M[3] = __fmul_rn(2.0f, __fmaf_rn(x, y, __fmul_rn(w, z)));
    M[4] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(x, x, __fmul_rn(z, z))));
    M[5] = __fmul_rn(2.0f, __fmaf_rn(y, z, -__fmul_rn(w, x)));
    M[6] = __fmul_rn(2.0f, __fmaf_rn(x, z, -__fmul_rn(w, y)));
    M[7] = __fmul_rn(2.0f, __fmaf_rn(y, z, __fmul_rn(w, x)));
    M[8] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(x, x, __fmul_rn(y, y))));
    float L[9];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        L[3 * i + 0] = __fmul_rn(M[3 * i + 0], s0);
        L[3 * i + 1] = __fmul_rn(M[3 * i + 1], s1);
        L[3 * i + 2] = __fmul_rn(M[3 * i + 2], s2);
    }
    float S[9];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 3; ++k)
            S[3 * i + k] = __fmaf_rn(L[3 * i + 2], L[3 * k + 2], __fmaf_rn(L[3 * i + 1], L[3 * k + 1], __fmul_rn(L[3 * i], L[3 * k])));
    float X, Y, Z;
    hy_to_camera(f, px, py, pz, X, Y, Z);
    const float iz = __fdiv_rn(1.0f, Z), xn = __fmul_rn(X, iz), yn = __fmul_rn(Y, iz);
    const float J00 = __fmul_rn(f.fx, iz), J02 = __fmul_rn(-__fmul_rn(f.fx, xn), iz);
    const float J11 = __fmul_rn(f.fy, iz), J12 = __fmul_rn(-__fmul_rn(f.fy, yn), iz);
    float T0[3], T1[3], U0[3], U1[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T0[k] = __fmaf_rn(J02, f.R[6 + k], __fmul_rn(J00, f.R[k]));
        T1[k] = __fmaf_rn(J12, f.R[6 + k], __fmul_rn(J11, f.R[3 + k]));
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        U0[k] = __fmaf_rn(T0[2], S[6 + k], __fmaf_rn(T0[1], S[3 + k], __fmul_rn(T0[0], S[k])));
        U1[k] = __fmaf_rn(T1[2], S[6 + k], __fmaf_rn(T1[1], S[3 + k], __fmul_rn(T1[0], S[k])));
    }
    const float a = __fadd_rn(__fmaf_rn(U0[2], T0[2], __fmaf_rn(U0[1], T0[1], __fmul_rn(U0[0], T0[0]))), 0.3f);
    const float b = __fmaf_rn(U0[2], T1[2], __fmaf_rn(U0[1], T1[1], __fmul_rn(U0[0], T1[0])));
    const float c = __fadd_rn(__fmaf_rn(U1[2], T1[2], __fmaf_rn(U1[1], T1[1], __fmul_rn(U1[0], T1[0]))), 0.3f);
    const float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
    const float u = __fmaf_rn(f.fx, xn, f.cx), v = __fmaf_rn(f.fy, yn, f.cy);
    float cA = 0.0f, cB = 0.0f, cC = 0.0f, radius = 0.0f;
    uint4 rc = make_uint4(0, 0, 0, 0);
    uint32_t nt = 0;
    // "w/o pre-culling" ablation: Eq. 9 is applied here instead of in S1 (D1's test on the same X, Y, Z)
    const bool dropped = (f.ablation & HYRF_ABL_NO_CULL) &&
                         !((Z > f.z_near) && (fabsf(X) <= __fmul_rn(f.limx, Z)) && (fabsf(Y) <= __fmul_rn(f.limy, Z)));
    if (!dropped && det != 0.0f && isfinite(det)) {
        const float di = __fdiv_rn(1.0f, det);
        cA = __fmul_rn(c, di);
        cB = __fmul_rn(-b, di);
        cC = __fmul_rn(a, di);
        const float mid = __fmul_rn(0.5f, __fadd_rn(a, c));
        const float lam = __fadd_rn(mid, __fsqrt_rn(fmaxf(0.1f, __fmaf_rn(mid, mid, -det))));
        radius = ceilf(__fmul_rn(3.0f, __fsqrt_rn(lam)));
        const float gx = (float)f.gx, gy = (float)f.gy;
        const float fx0 = fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(u, radius), 0.0625f)), 0.0f), gx);
        const float fx1 = fminf(fmaxf(floorf(__fmul_rn(__fadd_rn(__fadd_rn(u, radius), 15.0f), 0.0625f)), 0.0f), gx);
        const float fy0 = fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(v, radius), 0.0625f)), 0.0f), gy);
        const float fy1 = fminf(fmaxf(floorf(__fmul_rn(__fadd_rn(__fadd_rn(v, radius), 15.0f), 0.0625f)), 0.0f), gy);
        if (fx0 == fx0 && fx1 == fx1 && fy0 == fy0 && fy1 == fy1) {
            // (screen strips, hyrf_set_strip: only the tile rows of this device's strip are binned; a tile inside the strip
            // sees exactly the rectangles it would see in the whole image)
            rc = make_uint4((uint32_t)fx0, (uint32_t)fx1, max((uint32_t)fy0, (uint32_t)f.ty0), min((uint32_t)fy1, (uint32_t)f.ty1));
            if (rc.y > rc.x && rc.w > rc.z) nt = (rc.y - rc.x) * (rc.w - rc.z);
        }
    }
    // macro tiles (4 x 4 tile blocks) the rectangle touches: the unit the binning works in
    uint32_t mt = 0;
    if (nt) {
        const uint32_t sh = (uint32_t)f.mshift, r = (1u << sh) - 1u;
        mt = (((rc.y + r) >> sh) - (rc.x >> sh)) * (((rc.w + r) >> sh) - (rc.z >> sh));
    }
    {   // D = sum of tiles touched, Dm = sum of macro tiles touched: one atomic each per warp
        const unsigned am = __activemask();
        const uint32_t wsum = __reduce_add_sync(am, nt), msum = __reduce_add_sync(am, mt);
        if ((threadIdx.x & 31u) == (uint32_t)(__ffs(am) - 1) && wsum) {
            atomicAdd(&A.counters->D, (unsigned long long)wsum);
            atomicAdd(&A.counters->Dm, (unsigned long long)msum);
        }
    }
    if (dropped) {
        const float4 zero = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        A.rec[3ull * j + 0] = zero; A.rec[3ull * j + 1] = zero; A.rec[3ull * j + 2] = zero;
    } else {
        A.rec[3ull * j + 0] = make_float4(u, v, cA, cB);
        A.rec[3ull * j + 1] = make_float4(cC, alpha, c0, c1);
        A.rec[3ull * j + 2] = make_float4(c2, Z, radius, __uint_as_float(nt));
    }
    // (the key of the depth sort S4c, the bits of this same Z, is written by the cull's compaction: the sort runs
    // beside this kernel on a second stream)
    A.rect[j] = rc;
    A.tiles[j] = nt;
    A.mtiles[j] = mt;
}

