// backward.cu — the backward pass of the hybrid render (§3.4): given dL/d out of
// the LAST rendered frame, gradients with respect to every parameter of the scene — explicit Gaussians (position,
// s_e, alpha_e, c_e), the geometry / appearance / background tables, the three decoders — and the loss of Eq. 12.
// Arithmetic: DESIGN.md §2 D13. The forward's decisions (visible set, cells, lists, blended prefixes, background
// mask, ReLU masks, clamps) are frozen; everything smooth in between is differentiated in binary32:
//
//   background_backward_kernel   S6: out = C_fg + T c_s  ->  dL/dT per background pixel, bg table (atomics), bg decoder
//   raster_backward_kernel       S5: (raster_backward.cu)  ->  dL/d(u, v, A, B, C, o, r, g, b) per visible Gaussian
//   field_backward_kernel        S4a-S2: projection, Eq. 7, both decoders, direction encoding, both grid encodes,
//                                contraction  ->  explicit parameters (one thread owns a Gaussian: plain adds), tables
//                                (atomics), decoder weights
//   loss kernels                 Eq. 12: (1 - lambda) L1 + lambda (1 - SSIM), value and dL/d image
//
// A thread owns one Gaussian (or background pixel), recomputes its forward activations with the decoders' fp32 weights
// in shared memory, and back-propagates on CUDA cores (for the paper's decoder shapes through routines with
// compile-time sizes). Decoder weight gradients are sums over ALL Gaussians of outer products delta x activation:
// per warp a 32-Gaussian slice of dW = Delta^T H on the tensor cores (mma.sync tf32, accumulate_dw_mma) — or, for
// other decoder shapes, a transposing butterfly (accumulate_dw) — into one shared-memory accumulator block per
// persistent CTA; the CTAs add their blocks to global memory once at the end. (Activations and deltas as tensor-core
// tiles too, as in the forward kernel, is the next step: DESIGN.md §12.)
#include <mutex>

#include "field_common.cuh"
#include "mlp.cuh"
#include "raster_common.cuh"

namespace {

constexpr int kBwdThreads = 128;
constexpr int kMaxW = HYRF_MAX_WIDTH;   // 64

// sum over the warp's lanes of v[i], delivered to lane i: a butterfly in which every lane keeps one half of its values
// and hands the other half to its partner (16 + 8 + 4 + 2 + 1 = 31 shuffles for 32 values)
__device__ __forceinline__ float warp_transpose_sum32(float (&v)[32], uint32_t lane) {
#pragma unroll
    for (int off = 16, n = 32; off >= 1; off >>= 1, n >>= 1) {
        const bool up = lane & off;
#pragma unroll
        for (int i = 0; i < n / 2; ++i) {
            const float send = up ? v[i] : v[i + n / 2];
            const float keep = up ? v[i + n / 2] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
    }
    return v[0];
}

// dW[j][k] += sum over the warp's lanes of delta[j] * h[k]   (dW: shared memory, row-major [n_out][n_in])
__device__ __forceinline__ void accumulate_dw(float* dW, const float* delta, const float* h, int n_out, int n_in, uint32_t lane) {
    for (int j = 0; j < n_out; ++j) {
        const float dj = delta[j];
        for (int k0 = 0; k0 < n_in; k0 += 32) {
            float v[32];
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = (k0 + i < n_in) ? dj * h[k0 + i] : 0.0f;
            const float s = warp_transpose_sum32(v, lane);
            if (k0 + (int)lane < n_in && s != 0.0f) atomicAdd(&dW[j * n_in + k0 + lane], s);
        }
    }
}

// Decoder forward keeping what the backward needs. w: fp32 weights in shared memory. act[0] = input (n_in), act[1..nh] =
// hidden activations after ReLU (rounded to fp16 when FP16, as the forward pass does), out = linear outputs.
template <bool FP16>
__device__ __forceinline__ void mlp_forward_keep(const float* w, int n_in, int hid, int nh, int n_out,
                                                 float (*act)[kMaxW], float* out) {
    const float* wl = w;
    int nin = n_in;
    for (int l = 0; l < nh; ++l) {
        for (int j = 0; j < hid; ++j) {
            float acc = 0.0f;
            for (int k = 0; k < nin; ++k) acc = fmaf(wl[j * nin + k], act[l][k], acc);
            acc = fmaxf(acc, 0.0f);
            act[l + 1][j] = FP16 ? hy_round_half(acc) : acc;
        }
        wl += hid * nin;
        nin = hid;
    }
    for (int j = 0; j < n_out; ++j) {
        float acc = 0.0f;
        for (int k = 0; k < nin; ++k) acc = fmaf(wl[j * nin + k], act[nh][k], acc);
        out[j] = acc;
    }
}

// Decoder backward: g_out (n_out) -> g_in (n_in), weight gradients into dW (shared memory, same layout as w).
// `active`: lanes without work pass zeros (every lane of the warp takes part in the reductions).
__device__ __forceinline__ void mlp_backward(const float* w, float* dW, int n_in, int hid, int nh, int n_out,
                                             float (*act)[kMaxW], const float* g_out, float* g_in, uint32_t lane) {
    // offsets of the layers
    int offs[6];
    int nin = n_in, o = 0;
    for (int l = 0; l < nh; ++l) { offs[l] = o; o += hid * nin; nin = hid; }
    offs[nh] = o;
    float delta[kMaxW], prev[kMaxW];
    // output layer
    accumulate_dw(dW + offs[nh], g_out, act[nh], n_out, hid, lane);
    for (int k = 0; k < hid; ++k) {
        float acc = 0.0f;
        for (int j = 0; j < n_out; ++j) acc = fmaf(w[offs[nh] + j * hid + k], g_out[j], acc);
        delta[k] = act[nh][k] > 0.0f ? acc : 0.0f;      // ReLU mask of the forward pass
    }
    for (int l = nh - 1; l >= 0; --l) {
        const int li = l == 0 ? n_in : hid;
        accumulate_dw(dW + offs[l], delta, act[l], hid, li, lane);
        for (int k = 0; k < li; ++k) {
            float acc = 0.0f;
            for (int j = 0; j < hid; ++j) acc = fmaf(w[offs[l] + j * li + k], delta[j], acc);
            prev[k] = (l > 0) ? (act[l][k] > 0.0f ? acc : 0.0f) : acc;
        }
        for (int k = 0; k < li; ++k) delta[k] = prev[k];
    }
    for (int k = 0; k < n_in; ++k) g_in[k] = delta[k];
}

// dW[j][k] += sum over the warp's 32 Gaussians of delta[j] * h[k] on the tensor cores: D = Delta^T H as 16 x 8 tiles of
// mma.m16n8k8 (tf32 x tf32 -> fp32), K = the 32 lanes in four steps. A lane holds ITS Gaussian's delta and h; the
// fragments need other lanes' values (A: row j = 16 jt + lane / 4 (+ 8), column g = 8 ks + lane % 4 (+ 4); B: row g,
// column k = 8 kt + lane / 4), so they are assembled with shuffles: for r = 0 .. 7 every lane offers element r of the
// current row block and the lanes with lane / 4 == r keep what the owner of their column's Gaussian offered. ~1.3
// shuffle + select pairs per weight instead of the butterfly's 6 instructions; the products are rounded to tf32
// (10-bit mantissa, round to nearest: relative 2^-11 per factor, unbiased), the sums are fp32.
__device__ __forceinline__ uint32_t to_tf32(float v) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
    return r;
}

template <int NOUT, int NIN>
__device__ __forceinline__ void accumulate_dw_mma(float* dW, const float* delta, const float* h, uint32_t lane) {
    static_assert(NIN % 8 == 0, "column tiles of 8");
    constexpr int JT = (NOUT + 15) / 16, KT = NIN / 8;
    constexpr bool HI = NOUT > 8;   // rows 8 .. 15 of a row block exist
    const uint32_t gid = lane >> 2, tig = lane & 3u;
#pragma unroll 1
    for (int jt = 0; jt < JT; ++jt) {
        // A fragments of this row block for the four k-steps
        uint32_t a[4][4];
        {
            float lo[8], hi8[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                lo[r] = (jt * 16 + r < NOUT) ? delta[jt * 16 + r] : 0.0f;
                hi8[r] = (HI && jt * 16 + 8 + r < NOUT) ? delta[jt * 16 + 8 + r] : 0.0f;
            }
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                float f0 = 0.0f, f1 = 0.0f, f2 = 0.0f, f3 = 0.0f;
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const float u0 = __shfl_sync(0xffffffffu, lo[r], 8 * ks + tig), u2 = __shfl_sync(0xffffffffu, lo[r], 8 * ks + tig + 4);
                    if (gid == (uint32_t)r) { f0 = u0; f2 = u2; }
                    if (HI) {
                        const float u1 = __shfl_sync(0xffffffffu, hi8[r], 8 * ks + tig), u3 = __shfl_sync(0xffffffffu, hi8[r], 8 * ks + tig + 4);
                        if (gid == (uint32_t)r) { f1 = u1; f3 = u3; }
                    }
                }
                a[ks][0] = to_tf32(f0); a[ks][1] = to_tf32(f1); a[ks][2] = to_tf32(f2); a[ks][3] = to_tf32(f3);
            }
        }
#pragma unroll 1
        for (int kt = 0; kt < KT; ++kt) {
            float hv[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) hv[r] = h[kt * 8 + r];
            float c0 = 0.0f, c1 = 0.0f, c2 = 0.0f, c3 = 0.0f;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                float g0 = 0.0f, g1 = 0.0f;
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const float u0 = __shfl_sync(0xffffffffu, hv[r], 8 * ks + tig), u1 = __shfl_sync(0xffffffffu, hv[r], 8 * ks + tig + 4);
                    if (gid == (uint32_t)r) { g0 = u0; g1 = u1; }
                }
                const uint32_t b0 = to_tf32(g0), b1 = to_tf32(g1);
                asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                             : "+f"(c0), "+f"(c1), "+f"(c2), "+f"(c3)
                             : "r"(a[ks][0]), "r"(a[ks][1]), "r"(a[ks][2]), "r"(a[ks][3]), "r"(b0), "r"(b1));
            }
            const int j0 = jt * 16 + (int)gid, k0 = kt * 8 + 2 * (int)tig;
            if (j0 < NOUT) {
                if (c0 != 0.0f) atomicAdd(&dW[j0 * NIN + k0], c0);
                if (c1 != 0.0f) atomicAdd(&dW[j0 * NIN + k0 + 1], c1);
            }
            if (HI && j0 + 8 < NOUT) {
                if (c2 != 0.0f) atomicAdd(&dW[(j0 + 8) * NIN + k0], c2);
                if (c3 != 0.0f) atomicAdd(&dW[(j0 + 8) * NIN + k0 + 1], c3);
            }
        }
    }
}

// ---- the same two routines for the paper's decoder shapes (NIN -> 64 -> 64 -> NOUT), sizes known at compile
// time: inputs of a layer in registers, weight rows as 16-byte shared-memory loads, four neurons (forward) or one row of
// 64 accumulators (backward) at a time. Every sum keeps the order of the run-time versions above (and of D5), so the
// values are the same bits; the run-time versions cost ~4.5 issued instructions per multiply-add, these ~1.3.
template <bool FP16, int NIN, int NOUT>
__device__ __forceinline__ void mlp_forward_keep_ct(const float* w, float (*act)[kMaxW], float* out) {
    mlp_dense_ct<FP16, NIN, true, 64>(w, act[0], act[1]);
    mlp_dense_ct<FP16, 64, true, 64>(w + 64 * NIN, act[1], act[2]);
    mlp_dense_ct<FP16, 64, false, NOUT>(w + 64 * NIN + 64 * 64, act[2], out);
}

// prev[k] = sum_j w[j][k] d[j] (j ascending for every k), k < NK
template <int NK, int NJ>
__device__ __forceinline__ void backprop_ct(const float* __restrict__ w, const float* d, float (&acc)[NK]) {
#pragma unroll
    for (int k = 0; k < NK; ++k) acc[k] = 0.0f;
#pragma unroll 1
    for (int j = 0; j < NJ; ++j) {
        const float dj = d[j];
        const float4* row = reinterpret_cast<const float4*>(w + j * NK);
#pragma unroll
        for (int k = 0; k < NK / 4; ++k) {
            const float4 q = row[k];
            acc[4 * k] = fmaf(q.x, dj, acc[4 * k]);
            acc[4 * k + 1] = fmaf(q.y, dj, acc[4 * k + 1]);
            acc[4 * k + 2] = fmaf(q.z, dj, acc[4 * k + 2]);
            acc[4 * k + 3] = fmaf(q.w, dj, acc[4 * k + 3]);
        }
    }
}

template <int NIN, int NOUT>
__device__ __forceinline__ void mlp_backward_ct(const float* w, float* dW, float (*act)[kMaxW], const float* g_out, float* g_in,
                                                uint32_t lane) {
    constexpr int o1 = 64 * NIN, o2 = o1 + 64 * 64;
    float delta[kMaxW];
    {
        accumulate_dw_mma<NOUT, 64>(dW + o2, g_out, act[2], lane);
        float acc[64];
        backprop_ct<64, NOUT>(w + o2, g_out, acc);
#pragma unroll
        for (int k = 0; k < 64; ++k) delta[k] = act[2][k] > 0.0f ? acc[k] : 0.0f;      // ReLU mask of the forward pass
    }
    {
        accumulate_dw_mma<64, 64>(dW + o1, delta, act[1], lane);
        float acc[64];
        backprop_ct<64, 64>(w + o1, delta, acc);
#pragma unroll
        for (int k = 0; k < 64; ++k) delta[k] = act[1][k] > 0.0f ? acc[k] : 0.0f;
    }
    {
        accumulate_dw_mma<64, NIN>(dW, delta, act[0], lane);
        float acc[NIN];
        backprop_ct<NIN, 64>(w, delta, acc);
#pragma unroll
        for (int k = 0; k < NIN; ++k) g_in[k] = acc[k];
    }
}

// the background decoder's shape (NIN -> 64 -> 3, one hidden layer)
template <bool FP16, int NIN>
__device__ __forceinline__ void mlp_forward_keep_ct1(const float* w, float (*act)[kMaxW], float* out) {
    mlp_dense_ct<FP16, NIN, true, 64>(w, act[0], act[1]);
    mlp_dense_ct<FP16, 64, false, 3>(w + 64 * NIN, act[1], out);
}

template <int NIN>
__device__ __forceinline__ void mlp_backward_ct1(const float* w, float* dW, float (*act)[kMaxW], const float* g_out, float* g_in,
                                                 uint32_t lane) {
    constexpr int o1 = 64 * NIN;
    float delta[kMaxW];
    {
        accumulate_dw_mma<3, 64>(dW + o1, g_out, act[1], lane);
        float acc[64];
        backprop_ct<64, 3>(w + o1, g_out, acc);
#pragma unroll
        for (int k = 0; k < 64; ++k) delta[k] = act[1][k] > 0.0f ? acc[k] : 0.0f;      // ReLU mask of the forward pass
    }
    {
        accumulate_dw_mma<64, NIN>(dW, delta, act[0], lane);
        float acc[NIN];
        backprop_ct<NIN, 64>(w, delta, acc);
#pragma unroll
        for (int k = 0; k < NIN; ++k) g_in[k] = acc[k];
    }
}

// One level of one grid, forward and backward in one corner loop: the feature gradient g (2 values) is scattered to the
// eight entries (atomics on the fp32 gradient table, [entry][2]) and its derivative with respect to the contracted
// position accumulated in gx. The cell is the forward's (frozen).
template <int DT>
__device__ __forceinline__ void grid_level_backward(const GridDev& g, uint32_t l, const float x[3], float g0, float g1,
                                                    float* __restrict__ gtab, float gx[3]) {
    const uint32_t N = g.res[l];
    const float Nf = (float)N;
    uint32_t ci[3];
    float w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float u = x[a] * Nf;
        int i = (int)floorf(u);
        i = min(i, (int)N - 1);
        ci[a] = (uint32_t)i;
        w[a] = u - (float)i;
    }
    const bool dense = (g.dense_mask >> l) & 1u;
    const uint32_t n1 = N + 1u;
    float dwa[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const uint32_t bx = k & 1, by = (k >> 1) & 1, bz = (k >> 2) & 1;
        const uint32_t vx = ci[0] + bx, vy = ci[1] + by, vz = ci[2] + bz;
        const uint32_t e = g.offset[l] + (dense ? (vx + n1 * (vy + n1 * vz)) : ((vx ^ (vy * 2654435761u) ^ (vz * 805459861u)) & g.table_mask));
        const float ax = bx ? w[0] : 1.0f - w[0], ay = by ? w[1] : 1.0f - w[1], az = bz ? w[2] : 1.0f - w[2];
        const float wt = ax * ay * az;
        if (gtab) {
            if (g0 != 0.0f) atomicAdd(gtab + 2ull * e, wt * g0);
            if (g1 != 0.0f) atomicAdd(gtab + 2ull * e + 1, wt * g1);
        }
        float v0, v1;
        if (DT == HY_DT_U8) {
            const uchar2 c = __ldg(reinterpret_cast<const uchar2*>(g.table) + e);
            v0 = fmaf((float)c.x, g.q[l][0].y, g.q[l][0].x); v1 = fmaf((float)c.y, g.q[l][1].y, g.q[l][1].x);
        } else if (DT == HY_DT_F16) {
            const float2 v = __half22float2(__ldg(reinterpret_cast<const __half2*>(g.table) + e));
            v0 = v.x; v1 = v.y;
        } else {
            const float2 v = __ldg(reinterpret_cast<const float2*>(g.table) + e);
            v0 = v.x; v1 = v.y;
        }
        const float vg = v0 * g0 + v1 * g1;
        dwa[0] += (bx ? 1.0f : -1.0f) * ay * az * vg;
        dwa[1] += (by ? 1.0f : -1.0f) * ax * az * vg;
        dwa[2] += (bz ? 1.0f : -1.0f) * ax * ay * vg;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) gx[a] += Nf * dwa[a];
}

// D2 backward: g_x (gradient on the contracted position) -> g_p (world position). Clamped coordinates pass nothing.
__device__ __forceinline__ void contract_backward(const FrameDev& f, const float p[3], const float x[3], const float gx[3], float gp[3]) {
    float q[3], gq[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        q[a] = (p[a] - f.aabb_c[a]) / f.aabb_h[a];
        gq[a] = (x[a] > 0.0f && x[a] < 1.0f) ? 0.25f * gx[a] : 0.0f;
    }
    const float n = sqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
    if (n > 1.0f) {   // q' = s(n) q,  s = 2 / n - 1 / n^2
        const float inv = 1.0f / n, s = (2.0f - inv) * inv, ds = (-2.0f + 2.0f * inv) * inv * inv;
        const float dot = q[0] * gq[0] + q[1] * gq[1] + q[2] * gq[2];
#pragma unroll
        for (int a = 0; a < 3; ++a) gq[a] = s * gq[a] + ds * inv * dot * q[a];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) gp[a] = gq[a] / f.aabb_h[a];
}

// D4 forward values (fp32) and backward: g_pe (6 K) -> g_d (3)
__device__ __forceinline__ void dir_pe_backward(const float d[3], int octaves, const float* g_pe, float gd[3]) {
    gd[0] = gd[1] = gd[2] = 0.0f;
    for (int k = 0; k < octaves; ++k) {
        const float sc = (float)(1u << k);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float sn, cs;
            sincospif(sc * d[a], &sn, &cs);
            gd[a] += 3.14159265358979f * sc * (g_pe[6 * k + a] * cs - g_pe[6 * k + 3 + a] * sn);
        }
    }
}


struct BwdArgs {
    FieldArgs F;                 // the forward's argument block of the same frame (grids, decoders, camera, work list)
    GridDev bg_grid;
    MlpDev bg_mlp;
    const float* g_rec;          // [V][9] dL/d(u, v, A, B, C, o, r, g, b), row = visible rank
    const uint32_t* tiles;       // [V] tiles touched (0: the Gaussian was in no list)
    // outputs (any may be null)
    float *g_pos, *g_rgb, *g_scale, *g_opac;   // [3][N], [3][N], [N], [N]
    float *g_geo_table, *g_app_table, *g_bg_table;
    float *g_geo_w, *g_app_w, *g_bg_w;
    // background
    const float* g_out;          // [H][W][3]
    const float* finalT;
    const uint32_t* bg_list;
    float* g_T;                  // [H][W], written for the background pixels (zeroed before)
    uint32_t fp16;               // activations rounded to fp16 in the forward pass
};

__device__ __forceinline__ int mlp_weight_count(const MlpDev& m) {
    return (int)(m.in_dim * m.hidden + (m.n_hidden - 1) * m.hidden * m.hidden + m.hidden * m.out_dim);
}

template <typename T>
__device__ __forceinline__ void load_weights(float* dst, const void* src, int n) {
    const T* w = reinterpret_cast<const T*>(src);
    for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = (float)w[i];
}

// ---- S4a .. S2 ------------------------------------------------------------------------------------------------------
constexpr int kFieldBwdThreads = 512;   // one CTA per SM (116 KB of weights + accumulators): 16 warps hide the local-memory and shared-memory latencies

// STD: the decoders have the paper's shapes (geometry 32 -> 64 -> 64 -> 8, appearance 56 -> 64 -> 64 -> 3)
template <int DT, bool STD>
__global__ void __launch_bounds__(kFieldBwdThreads)
field_backward_kernel(const BwdArgs B) {
    extern __shared__ __align__(16) float sm[];
    constexpr bool FP16 = DT != HY_DT_F32;
    const FieldArgs& A = B.F;
    const FrameDev& f = A.f;
    const int nwg = mlp_weight_count(A.geo_mlp), nwa = mlp_weight_count(A.app_mlp);
    float *wg = sm, *wa = sm + nwg, *dwg = wa + nwa, *dwa = dwg + nwg;
    if (FP16) { load_weights<__half>(wg, A.geo_mlp.w, nwg); load_weights<__half>(wa, A.app_mlp.w, nwa); }
    else { load_weights<float>(wg, A.geo_mlp.w, nwg); load_weights<float>(wa, A.app_mlp.w, nwa); }
    for (int i = threadIdx.x; i < nwg + nwa; i += blockDim.x) dwg[i] = 0.0f;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t V = A.counters->V;
    const int Lg = (int)A.geo.levels, La = (int)A.app.levels, oct = (int)A.pe_octaves;
    const int gin = (int)A.geo_mlp.in_dim, ain = (int)A.app_mlp.in_dim;
    const int hg = (int)A.geo_mlp.hidden, ha = (int)A.app_mlp.hidden, nhg = (int)A.geo_mlp.n_hidden, nha = (int)A.app_mlp.n_hidden;
    const bool neural = !(f.ablation & HYRF_ABL_NO_NEURAL);
    const uint32_t per_pass = gridDim.x * blockDim.x;
    for (uint32_t base = blockIdx.x * blockDim.x; base < V; base += per_pass) {   // warps stay together: the reductions need every lane
        if (STD) __syncthreads();
        const uint32_t wi = base + threadIdx.x;
        const bool have = wi < V;
        Explicit ex{};
        uint32_t id = 0;
        if (have) {
            ex = fetch_visible(A, wi);
            id = __ldg(A.gm_id + __ldg(A.vis_m + wi));
        }
        const bool live = have && B.tiles[ex.j] > 0;     // in no list: no gradient (and no finite conic)
        float gr[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) gr[k] = live ? B.g_rec[9ull * ex.j + k] : 0.0f;
        const float p[3] = {ex.px, ex.py, ex.pz};
        float x[3] = {0.5f, 0.5f, 0.5f};
        if (have) hy_contract(f, p[0], p[1], p[2], x);
        // ---- forward recompute (fp32, the exact path's arithmetic) ----
        constexpr int kRows = STD ? 3 : 5;   // input + hidden layers kept (the paper's decoders have two hidden layers)
        float act_g[kRows][kMaxW], act_a[kRows][kMaxW], raw[11];
        float dvec[3] = {0.0f, 0.0f, 1.0f}, dn = 1.0f;
#pragma unroll
        for (int k = 0; k < 11; ++k) raw[k] = 0.0f;
        if (neural) {
            for (int k = 0; k < kMaxW; ++k) { act_g[0][k] = 0.0f; act_a[0][k] = 0.0f; }
            if (have) {
                for (int l = 0; l < Lg; ++l) {
                    float f0, f1;
                    hy_grid_level<DT>(A.geo, l, x, f0, f1);
                    act_g[0][2 * l] = FP16 ? hy_round_half(f0) : f0; act_g[0][2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
                }
                for (int l = 0; l < La; ++l) {
                    float f0, f1;
                    hy_grid_level<DT>(A.app, l, x, f0, f1);
                    act_a[0][2 * l] = FP16 ? hy_round_half(f0) : f0; act_a[0][2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
                }
                const float dx = p[0] - f.o[0], dy = p[1] - f.o[1], dz = p[2] - f.o[2];
                dn = sqrtf(dx * dx + dy * dy + dz * dz);
                dvec[0] = dx / dn; dvec[1] = dy / dn; dvec[2] = dz / dn;
                float pe[36];
                if (FP16) hy_dir_pe<true>(dvec, oct, pe); else hy_dir_pe<false>(dvec, oct, pe);
                for (int k = 0; k < 6 * oct; ++k) act_a[0][2 * La + k] = pe[k];
            }
            if (STD) { mlp_forward_keep_ct<FP16, 32, 8>(wg, act_g, raw); mlp_forward_keep_ct<FP16, 56, 3>(wa, act_a, raw + 8); }
            else { mlp_forward_keep<FP16>(wg, gin, hg, nhg, 8, act_g, raw); mlp_forward_keep<FP16>(wa, ain, ha, nha, 3, act_a, raw + 8); }
        }
        // Eq. 7
        const float s0 = hy_sigmoid(raw[1] + ex.s_e), s1 = hy_sigmoid(raw[2] + ex.s_e), s2 = hy_sigmoid(raw[3] + ex.s_e);
        const float qm = sqrtf(raw[4] * raw[4] + raw[5] * raw[5] + raw[6] * raw[6] + raw[7] * raw[7]);
        const float qd = fmaxf(qm, 1e-12f);
        const float qw = raw[4] / qd, qx = raw[5] / qd, qy = raw[6] / qd, qz = raw[7] / qd;
        const float alpha = hy_sigmoid(raw[0] + ex.a_e);
        const float c0 = hy_sigmoid(raw[8] + ex.c_e0), c1 = hy_sigmoid(raw[9] + ex.c_e1), c2 = hy_sigmoid(raw[10] + ex.c_e2);
        // ---- D8 backward ----
        float g_raw[11], gp[3] = {0.0f, 0.0f, 0.0f}, g_se = 0.0f;
#pragma unroll
        for (int k = 0; k < 11; ++k) g_raw[k] = 0.0f;
        if (live) {
            const float M[9] = {1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy),
                                2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx),
                                2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)};
            const float sv[3] = {s0, s1, s2};
            float L[9], S[9];
            for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) L[3 * i + k] = M[3 * i + k] * sv[k];
            for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) S[3 * i + k] = L[3 * i] * L[3 * k] + L[3 * i + 1] * L[3 * k + 1] + L[3 * i + 2] * L[3 * k + 2];
            float X, Y, Z;
            hy_to_camera(f, p[0], p[1], p[2], X, Y, Z);
            const float iz = 1.0f / Z, iz2 = iz * iz;
            const float J00 = f.fx * iz, J02 = -f.fx * X * iz2, J11 = f.fy * iz, J12 = -f.fy * Y * iz2;
            float T0[3], T1[3];
            for (int k = 0; k < 3; ++k) { T0[k] = J00 * f.R[k] + J02 * f.R[6 + k]; T1[k] = J11 * f.R[3 + k] + J12 * f.R[6 + k]; }
            float U0[3], U1[3];
            for (int k = 0; k < 3; ++k) { U0[k] = T0[0] * S[k] + T0[1] * S[3 + k] + T0[2] * S[6 + k]; U1[k] = T1[0] * S[k] + T1[1] * S[3 + k] + T1[2] * S[6 + k]; }
            const float a = U0[0] * T0[0] + U0[1] * T0[1] + U0[2] * T0[2] + 0.3f;
            const float b = U0[0] * T1[0] + U0[1] * T1[1] + U0[2] * T1[2];
            const float c = U1[0] * T1[0] + U1[1] * T1[1] + U1[2] * T1[2] + 0.3f;
            const float det = a * c - b * b, id2 = 1.0f / (det * det), idet = 1.0f / det;
            const float gA = gr[2], gB = gr[3], gC = gr[4];
            const float ga = gA * (-c * c * id2) + gB * (b * c * id2) + gC * (-b * b * id2);
            const float gb = gA * (2 * b * c * id2) + gB * (-idet - 2 * b * b * id2) + gC * (2 * a * b * id2);
            const float gc = gA * (-b * b * id2) + gB * (a * b * id2) + gC * (-a * a * id2);
            // G = [[ga, gb/2], [gb/2, gc]];  dL/dSigma = Tm^T G Tm,  dL/dTm = 2 G Tm Sigma = 2 G [U0; U1]
            const float G00 = ga, G01 = 0.5f * gb, G11 = gc;
            float gS[9];
            for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k)
                gS[3 * i + k] = T0[i] * (G00 * T0[k] + G01 * T1[k]) + T1[i] * (G01 * T0[k] + G11 * T1[k]);
            float gT0[3], gT1[3];
            for (int k = 0; k < 3; ++k) { gT0[k] = 2.0f * (G00 * U0[k] + G01 * U1[k]); gT1[k] = 2.0f * (G01 * U0[k] + G11 * U1[k]); }
            // Tm = J R  ->  dL/dJ = dL/dTm R^T
            const float gJ00 = gT0[0] * f.R[0] + gT0[1] * f.R[1] + gT0[2] * f.R[2];
            const float gJ02 = gT0[0] * f.R[6] + gT0[1] * f.R[7] + gT0[2] * f.R[8];
            const float gJ11 = gT1[0] * f.R[3] + gT1[1] * f.R[4] + gT1[2] * f.R[5];
            const float gJ12 = gT1[0] * f.R[6] + gT1[1] * f.R[7] + gT1[2] * f.R[8];
            const float gu = gr[0], gv = gr[1], iz3 = iz2 * iz;
            const float gX = gJ02 * (-f.fx * iz2) + gu * f.fx * iz;
            const float gY = gJ12 * (-f.fy * iz2) + gv * f.fy * iz;
            const float gZ = gJ00 * (-f.fx * iz2) + gJ02 * (2 * f.fx * X * iz3) + gJ11 * (-f.fy * iz2) + gJ12 * (2 * f.fy * Y * iz3) +
                             gu * (-f.fx * X * iz2) + gv * (-f.fy * Y * iz2);
            for (int k = 0; k < 3; ++k) gp[k] = f.R[k] * gX + f.R[3 + k] * gY + f.R[6 + k] * gZ;
            // Sigma = L L^T  ->  dL/dL = 2 gS L (gS symmetric);  L = M diag(s)
            float gL[9], gs[3] = {0.0f, 0.0f, 0.0f}, gM[9];
            for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) gL[3 * i + k] = 2.0f * (gS[3 * i] * L[k] + gS[3 * i + 1] * L[3 + k] + gS[3 * i + 2] * L[6 + k]);
            for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) { gs[k] += gL[3 * i + k] * M[3 * i + k]; gM[3 * i + k] = gL[3 * i + k] * sv[k]; }
            const float gqw = 2 * (-qz * gM[1] + qy * gM[2] + qz * gM[3] - qx * gM[5] - qy * gM[6] + qx * gM[7]);
            const float gqx = 2 * (qy * gM[1] + qz * gM[2] + qy * gM[3] - 2 * qx * gM[4] - qw * gM[5] + qz * gM[6] + qw * gM[7] - 2 * qx * gM[8]);
            const float gqy = 2 * (-2 * qy * gM[0] + qx * gM[1] + qw * gM[2] + qx * gM[3] + qz * gM[5] - qw * gM[6] + qz * gM[7] - 2 * qy * gM[8]);
            const float gqz = 2 * (-2 * qz * gM[0] - qw * gM[1] + qx * gM[2] + qw * gM[3] - 2 * qz * gM[4] + qy * gM[5] + qx * gM[6] + qy * gM[7]);
            // Eq. 7 backward
            g_raw[1] = gs[0] * s0 * (1 - s0); g_raw[2] = gs[1] * s1 * (1 - s1); g_raw[3] = gs[2] * s2 * (1 - s2);
            g_se = g_raw[1] + g_raw[2] + g_raw[3];
            if (qm > 1e-12f) {
                const float dotq = qw * gqw + qx * gqx + qy * gqy + qz * gqz;
                g_raw[4] = (gqw - qw * dotq) / qd; g_raw[5] = (gqx - qx * dotq) / qd;
                g_raw[6] = (gqy - qy * dotq) / qd; g_raw[7] = (gqz - qz * dotq) / qd;
            }
            g_raw[0] = gr[5] * alpha * (1 - alpha);
            g_raw[8] = gr[6] * c0 * (1 - c0); g_raw[9] = gr[7] * c1 * (1 - c1); g_raw[10] = gr[8] * c2 * (1 - c2);
        }
        // explicit parameters: this thread owns the Gaussian
        if (live && !(f.ablation & HYRF_ABL_NO_EXPLICIT)) {
            if (B.g_scale) B.g_scale[id] += g_se;
            if (B.g_opac) B.g_opac[id] += g_raw[0];
            if (B.g_rgb) { B.g_rgb[id] += g_raw[8]; B.g_rgb[A.N + id] += g_raw[9]; B.g_rgb[2ull * A.N + id] += g_raw[10]; }
        }
        // ---- decoders, encodings, contraction ----
        if (neural) {
            float g_in_g[kMaxW], g_in_a[kMaxW];
            if (STD) {
                // (the barriers keep the CTA's 16 warps in the same stretch of this long kernel: without them the warps
                // spread over more code than the instruction cache holds and `no_instruction` is the first stall reason)
                __syncthreads();
                mlp_backward_ct<32, 8>(wg, dwg, act_g, g_raw, g_in_g, lane);
                __syncthreads();
                mlp_backward_ct<56, 3>(wa, dwa, act_a, g_raw + 8, g_in_a, lane);
                __syncthreads();
            } else {
                mlp_backward(wg, dwg, gin, hg, nhg, 8, act_g, g_raw, g_in_g, lane);
                mlp_backward(wa, dwa, ain, ha, nha, 3, act_a, g_raw + 8, g_in_a, lane);
            }
            if (live) {
                float gx[3] = {0.0f, 0.0f, 0.0f};
                for (int l = 0; l < Lg; ++l) grid_level_backward<DT>(A.geo, l, x, g_in_g[2 * l], g_in_g[2 * l + 1], B.g_geo_table, gx);
                for (int l = 0; l < La; ++l) grid_level_backward<DT>(A.app, l, x, g_in_a[2 * l], g_in_a[2 * l + 1], B.g_app_table, gx);
                float gpc[3];
                contract_backward(f, p, x, gx, gpc);
                float gd[3];
                dir_pe_backward(dvec, oct, g_in_a + 2 * La, gd);
                const float dotd = dvec[0] * gd[0] + dvec[1] * gd[1] + dvec[2] * gd[2];
                for (int k = 0; k < 3; ++k) gp[k] += gpc[k] + (gd[k] - dvec[k] * dotd) / dn;
            }
        }
        if (live && B.g_pos) { B.g_pos[id] += gp[0]; B.g_pos[A.N + id] += gp[1]; B.g_pos[2ull * A.N + id] += gp[2]; }
    }
    __syncthreads();
    if (B.g_geo_w) for (int i = threadIdx.x; i < nwg; i += blockDim.x) if (dwg[i] != 0.0f) atomicAdd(B.g_geo_w + i, dwg[i]);
    if (B.g_app_w) for (int i = threadIdx.x; i < nwa; i += blockDim.x) if (dwa[i] != 0.0f) atomicAdd(B.g_app_w + i, dwa[i]);
}


// ---- S6 ---------------------------------------------------------------------------------------------------------------
// out = C_fg + T c_s on the background pixels of the frame (the rasterizer's list): dL/dT = sum_c g_out c_s (the part of
// dL/dT that comes through the composite; raster_backward adds nothing else to it), dL/dc_s = T g_out -> sigmoid ->
// background decoder -> background table.
// STD: the background decoder has the paper's shape (40 -> 64 -> 3)
template <int DT, bool STD>
__global__ void __launch_bounds__(kBwdThreads)
background_backward_kernel(const BwdArgs B) {
    extern __shared__ __align__(16) float sm[];
    constexpr bool FP16 = DT != HY_DT_F32;
    const FrameDev& f = B.F.f;
    const int nw = mlp_weight_count(B.bg_mlp);
    float *w = sm, *dw = sm + nw;
    if (FP16) load_weights<__half>(w, B.bg_mlp.w, nw); else load_weights<float>(w, B.bg_mlp.w, nw);
    for (int i = threadIdx.x; i < nw; i += blockDim.x) dw[i] = 0.0f;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t n_bg = B.F.counters->n_bg;
    const int L = (int)B.bg_grid.levels, oct = (int)B.F.pe_octaves;
    const int nin = (int)B.bg_mlp.in_dim, hid = (int)B.bg_mlp.hidden, nh = (int)B.bg_mlp.n_hidden;
    const uint32_t per_pass = gridDim.x * blockDim.x;
    for (uint32_t base = blockIdx.x * blockDim.x; base < n_bg; base += per_pass) {
        const uint32_t q = base + threadIdx.x;
        const bool have = q < n_bg;
        float act[5][kMaxW], raw[3] = {0.0f, 0.0f, 0.0f}, x[3] = {0.5f, 0.5f, 0.5f}, T = 0.0f, g[3] = {0.0f, 0.0f, 0.0f};
        int pix = 0;
        for (int k = 0; k < kMaxW; ++k) act[0][k] = 0.0f;
        if (have) {
            pix = (int)B.bg_list[q];
            T = B.finalT[pix];
            g[0] = B.g_out[3ull * pix]; g[1] = B.g_out[3ull * pix + 1]; g[2] = B.g_out[3ull * pix + 2];
            const int pi = pix % f.W, pj = pix / f.W;
            const float dcx = ((float)pi - f.cx) / f.fx, dcy = ((float)pj - f.cy) / f.fy;
            float dwv[3], d[3], ps[3];
            for (int k = 0; k < 3; ++k) dwv[k] = f.R[k] * dcx + f.R[3 + k] * dcy + f.R[6 + k];
            const float n = sqrtf(dwv[0] * dwv[0] + dwv[1] * dwv[1] + dwv[2] * dwv[2]);
            for (int k = 0; k < 3; ++k) d[k] = dwv[k] / n;
            const float Bq = 2.0f * (f.o[0] * d[0] + f.o[1] * d[1] + f.o[2] * d[2]);
            const float Cq = f.o[0] * f.o[0] + f.o[1] * f.o[1] + f.o[2] * f.o[2] - f.bg_radius * f.bg_radius;
            const float t = 0.5f * (-Bq + sqrtf(Bq * Bq - 4.0f * Cq));
            for (int k = 0; k < 3; ++k) ps[k] = fmaf(t, d[k], f.o[k]);
            hy_contract(f, ps[0], ps[1], ps[2], x);
            for (int l = 0; l < L; ++l) {
                float f0, f1;
                hy_grid_level<DT>(B.bg_grid, l, x, f0, f1);
                act[0][2 * l] = FP16 ? hy_round_half(f0) : f0; act[0][2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
            }
            float pe[36];
            if (FP16) hy_dir_pe<true>(d, oct, pe); else hy_dir_pe<false>(d, oct, pe);
            for (int k = 0; k < 6 * oct; ++k) act[0][2 * L + k] = pe[k];
        }
        if (STD) mlp_forward_keep_ct1<FP16, 40>(w, act, raw); else mlp_forward_keep<FP16>(w, nin, hid, nh, 3, act, raw);
        float g_raw[3] = {0.0f, 0.0f, 0.0f}, gT = 0.0f;
        if (have) {
            for (int c = 0; c < 3; ++c) {
                const float cs = hy_sigmoid(raw[c]);
                gT += g[c] * cs;
                g_raw[c] = T * g[c] * cs * (1.0f - cs);
            }
            B.g_T[pix] = gT;
        }
        float g_in[kMaxW];
        if (STD) mlp_backward_ct1<40>(w, dw, act, g_raw, g_in, lane); else mlp_backward(w, dw, nin, hid, nh, 3, act, g_raw, g_in, lane);
        if (have && B.g_bg_table) {
            float gx[3] = {0.0f, 0.0f, 0.0f};
            for (int l = 0; l < L; ++l) grid_level_backward<DT>(B.bg_grid, l, x, g_in[2 * l], g_in[2 * l + 1], B.g_bg_table, gx);
        }
    }
    __syncthreads();
    if (B.g_bg_w) for (int i = threadIdx.x; i < nw; i += blockDim.x) if (dw[i] != 0.0f) atomicAdd(B.g_bg_w + i, dw[i]);
}

// ---- Eq. 12 -------------------------------------------------------------------------------------------------------------
// L = (1 - lambda) mean |a - b| + lambda (1 - mean SSIM(a, b)), SSIM with an 11 x 11 Gaussian window (sigma 1.5), zero
// padding, C1 = 0.01^2, C2 = 0.03^2 (reading A28). Pass 1 (per pixel and channel): window moments -> the SSIM map m and
// its partial derivatives with respect to mu_a, E[a^2], E[ab]; the loss terms are summed with one atomic per warp.
// Pass 2: dL/da_p = (1 - lambda) sign(a_p - b_p) / n - (lambda / n) sum_q w(q - p) (D1_q + 2 a_p D2_q + b_p D3_q).
__constant__ float c_win[11];

// The 11 x 11 window is an outer product, so both passes run it as 11 + 11 taps: a tile's inputs (16 x 16 pixels + a
// halo of 5, zeros outside the image) go to shared memory, the row pass leaves the horizontally filtered moments of
// the tile's 26 rows there, the column pass finishes them per pixel. 5 x fewer multiply-adds than the direct window.
constexpr int kSsimTile = 16, kSsimHalo = 5, kSsimIn = kSsimTile + 2 * kSsimHalo;   // 26

// NM maps in: src(m, y, x) for the tile with halo -> s_h[m][26][16]: sum over di of win[di + 5] * src(m, y, x0 + col + di)
template <int NM, typename F>
__device__ __forceinline__ void ssim_row_pass(F src, float (*s_in)[kSsimIn][kSsimIn], float (*s_h)[kSsimIn][kSsimTile], int x0, int y0) {
    for (int i = threadIdx.x; i < kSsimIn * kSsimIn; i += 256) {
        const int r = i / kSsimIn, c = i - r * kSsimIn;
        float v[NM];
        src(y0 + r - kSsimHalo, x0 + c - kSsimHalo, v);
#pragma unroll
        for (int m = 0; m < NM; ++m) s_in[m][r][c] = v[m];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kSsimIn * kSsimTile; i += 256) {
        const int r = i / kSsimTile, c = i - r * kSsimTile;
#pragma unroll
        for (int m = 0; m < NM; ++m) {
            float acc = 0.0f;
#pragma unroll
            for (int d = 0; d < 11; ++d) acc += c_win[d] * s_in[m][r][c + d];
            s_h[m][r][c] = acc;
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(256)
ssim_maps_kernel(const float* __restrict__ a, const float* __restrict__ b, int W, int H, float lam, float* __restrict__ D,
                 double* __restrict__ loss) {
    __shared__ float s_in[5][kSsimIn][kSsimIn];      // a, b, a a, b b, a b
    __shared__ float s_h[5][kSsimIn][kSsimTile];
    const int x0 = blockIdx.x * kSsimTile, y0 = blockIdx.y * kSsimTile, c = blockIdx.z;
    const int ti = threadIdx.x & 15, tj = threadIdx.x >> 4, i = x0 + ti, j = y0 + tj;
    ssim_row_pass<5>([&](int y, int x, float* v) {
        float av = 0.0f, bv = 0.0f;
        if (x >= 0 && x < W && y >= 0 && y < H) { av = a[3ull * ((size_t)y * W + x) + c]; bv = b[3ull * ((size_t)y * W + x) + c]; }
        v[0] = av; v[1] = bv; v[2] = av * av; v[3] = bv * bv; v[4] = av * bv;
    }, s_in, s_h, x0, y0);
    float l1 = 0.0f, ss = 0.0f;
    if (i < W && j < H) {
        float mo[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) {
            float acc = 0.0f;
#pragma unroll
            for (int d = 0; d < 11; ++d) acc += c_win[d] * s_h[m][tj + d][ti];
            mo[m] = acc;
        }
        const float ma = mo[0], mb = mo[1], saa = mo[2], sbb = mo[3], sab = mo[4];
        const float C1 = 1e-4f, C2 = 9e-4f;
        const float va = saa - ma * ma, vb = sbb - mb * mb, cab = sab - ma * mb;
        const float n1 = 2 * ma * mb + C1, n2 = 2 * cab + C2, d1 = ma * ma + mb * mb + C1, d2 = va + vb + C2;
        const float m = (n1 * n2) / (d1 * d2);
        // partial derivatives of m with respect to mu_a (at fixed E[a^2], E[ab]), E[a^2], E[ab]
        const float dm_dn1 = n2 / (d1 * d2), dm_dn2 = n1 / (d1 * d2), dm_dd1 = -m / d1, dm_dd2 = -m / d2;
        // n1 = 2 mu_a mu_b + C1; n2 = 2 (E[ab] - mu_a mu_b) + C2; d1 = mu_a^2 + mu_b^2 + C1; d2 = E[a^2] - mu_a^2 + vb + C2
        const size_t o = 3ull * ((size_t)j * W + i) + c, P3 = 3ull * W * H;
        D[o] = dm_dn1 * 2 * mb + dm_dn2 * (-2 * mb) + dm_dd1 * 2 * ma + dm_dd2 * (-2 * ma);
        D[P3 + o] = dm_dd2;
        D[2 * P3 + o] = 2 * dm_dn2;
        ss = m;
        l1 = fabsf(s_in[0][tj + kSsimHalo][ti + kSsimHalo] - s_in[1][tj + kSsimHalo][ti + kSsimHalo]);
    }
    const float n = 3.0f * W * H;
    float term = ((1.0f - lam) * l1 - lam * ss) / n;
    for (int off = 16; off >= 1; off >>= 1) term += __shfl_xor_sync(0xffffffffu, term, off);
    if ((threadIdx.x & 31) == 0 && term != 0.0f) atomicAdd(loss, (double)term);
}

__global__ void __launch_bounds__(256)
ssim_grad_kernel(const float* __restrict__ a, const float* __restrict__ b, int W, int H, float lam, const float* __restrict__ D,
                 float* __restrict__ g) {
    __shared__ float s_in[3][kSsimIn][kSsimIn];      // D1, D2, D3
    __shared__ float s_h[3][kSsimIn][kSsimTile];
    const int x0 = blockIdx.x * kSsimTile, y0 = blockIdx.y * kSsimTile, c = blockIdx.z;
    const int ti = threadIdx.x & 15, tj = threadIdx.x >> 4, i = x0 + ti, j = y0 + tj;
    const size_t P3 = 3ull * W * H;
    ssim_row_pass<3>([&](int y, int x, float* v) {
        v[0] = v[1] = v[2] = 0.0f;
        if (x >= 0 && x < W && y >= 0 && y < H) {
            const size_t q = 3ull * ((size_t)y * W + x) + c;
            v[0] = D[q]; v[1] = D[P3 + q]; v[2] = D[2 * P3 + q];
        }
    }, s_in, s_h, x0, y0);
    if (i >= W || j >= H) return;
    float sacc[3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
        float acc = 0.0f;
#pragma unroll
        for (int d = 0; d < 11; ++d) acc += c_win[d] * s_h[m][tj + d][ti];
        sacc[m] = acc;
    }
    const size_t o = 3ull * ((size_t)j * W + i) + c;
    const float n = 3.0f * W * H, av = a[o], bv = b[o];
    const float sgn = av > bv ? 1.0f : (av < bv ? -1.0f : 0.0f);
    g[o] = ((1.0f - lam) * sgn - lam * (sacc[0] + 2.0f * av * sacc[1] + bv * sacc[2])) / n;
}

}  // namespace

// ---- host side -----------------------------------------------------------------------------------------------------------
namespace {

hyrf_status bwd_alloc(hyrf_scene* s, float** p, size_t count) {
    if (*p) return HYRF_OK;
    void* q = nullptr;
    if (s->desc.alloc) q = s->desc.alloc(count * sizeof(float), s->desc.user);
    else if (cudaMalloc(&q, count * sizeof(float)) != cudaSuccess) { cudaGetLastError(); q = nullptr; }
    if (!q) return hy_fail(HYRF_ERR_OOM, "backward scratch of %zu floats", count);
    *p = static_cast<float*>(q);
    return HYRF_OK;
}

template <int DT>
hyrf_status launch_backward(hyrf_scene* s, const BwdArgs& B, uint32_t* launches) {
    const hyrf_mlp_desc &g = s->desc.geo_mlp, &a = s->desc.app_mlp, &b = s->desc.bg_mlp;
    auto nw = [](const hyrf_mlp_desc& m) { return (size_t)m.in_dim * m.hidden + (size_t)(m.n_hidden - 1) * m.hidden * m.hidden + (size_t)m.hidden * m.out_dim; };
    const size_t smem_bg = 2 * nw(b) * sizeof(float), smem_f = 2 * (nw(g) + nw(a)) * sizeof(float);
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(background_backward_kernel<DT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bg)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(background_backward_kernel<DT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bg)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(field_backward_kernel<DT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_f)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(field_backward_kernel<DT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_f)) != cudaSuccess)
        return hy_cuda_fail(e, "cudaFuncSetAttribute(backward)");
    const bool std_shapes = g.in_dim == 32 && g.hidden == 64 && g.n_hidden == 2 && g.out_dim == 8 &&
                            a.in_dim == 56 && a.hidden == 64 && a.n_hidden == 2 && a.out_dim == 3;
    const int P = s->lastW * s->lastH;
    if ((e = cudaMemsetAsync(B.g_T, 0, (size_t)P * sizeof(float), s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemsetAsync(g_T)");
    if (!(s->last_frame.ablation & HYRF_ABL_NO_BG)) {
        if (b.in_dim == 40 && b.hidden == 64 && b.n_hidden == 1 && b.out_dim == 3) background_backward_kernel<DT, true><<<s->sm_count * 4, kBwdThreads, smem_bg, s->stream>>>(B);
        else background_backward_kernel<DT, false><<<s->sm_count * 4, kBwdThreads, smem_bg, s->stream>>>(B);
        ++*launches;
    }
    hyrf_status st = hy_launch_raster_backward(s, B.g_out, B.g_T, const_cast<float*>(B.g_rec), launches);
    if (st != HYRF_OK) return st;
    if (std_shapes) field_backward_kernel<DT, true><<<s->sm_count, kFieldBwdThreads, smem_f, s->stream>>>(B);
    else field_backward_kernel<DT, false><<<s->sm_count, kFieldBwdThreads, smem_f, s->stream>>>(B);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return hy_cuda_fail(e, "backward kernels");
    return HYRF_OK;
}

}  // namespace

extern "C" hyrf_status hyrf_backward(hyrf_scene* s, const float* g_out, const hyrf_grads* grads) {
    if (!s || !g_out || !grads) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_backward: NULL argument");
    if (!s->rendered || !s->list_final)
        return hy_fail(HYRF_ERR_NOT_READY, "hyrf_backward: the last frame kept no per-tile lists (hyrf_set_retain_lists, or the debug export HYRF_DBG_TILE_LIST | HYRF_DBG_TILE_RANGES)");
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    hyrf_status st;
    if ((st = bwd_alloc(s, &s->bwd_gT, (size_t)s->desc.max_width * s->desc.max_height)) != HYRF_OK) return st;
    if ((st = bwd_alloc(s, &s->bwd_grec, 9ull * s->N)) != HYRF_OK) return st;
    BwdArgs B{};
    hy_fill_field_args(s, s->last_frame, &B.F);
    B.F.dbg_raw = nullptr; B.F.dbg_attrs = nullptr;
    B.bg_grid = s->bg_grid; B.bg_mlp = s->bg_mlp;
    B.g_rec = s->bwd_grec; B.tiles = s->tiles;
    B.g_pos = grads->pos; B.g_rgb = grads->rgb_logit; B.g_scale = grads->scale_logit; B.g_opac = grads->opacity_logit;
    B.g_geo_table = grads->geo_table; B.g_app_table = grads->app_table; B.g_bg_table = grads->bg_table;
    B.g_geo_w = grads->geo_w; B.g_app_w = grads->app_w; B.g_bg_w = grads->bg_w;
    B.g_out = g_out; B.finalT = s->finalT; B.bg_list = s->bg_list; B.g_T = s->bwd_gT;
    B.fp16 = s->fp16;
    uint32_t launches = 0;
    if (s->u8) st = launch_backward<HY_DT_U8>(s, B, &launches);
    else if (s->fp16) st = launch_backward<HY_DT_F16>(s, B, &launches);
    else st = launch_backward<HY_DT_F32>(s, B, &launches);
    s->last_backward_launches = launches;
    return st;
}

extern "C" hyrf_status hyrf_loss_l1_ssim(hyrf_scene* s, const float* image, const float* target, int32_t W, int32_t H,
                                         float lambda, double* loss_host, float* g_image) {
    if (!s || !image || !target || !loss_host) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim: NULL argument");
    if (W < 1 || H < 1 || (uint32_t)W > s->desc.max_width || (uint32_t)H > s->desc.max_height || !(lambda >= 0.0f) || !(lambda <= 1.0f))
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim: W x H = %d x %d, lambda = %g", W, H, (double)lambda);
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    hyrf_status st;
    const size_t P3 = 3ull * s->desc.max_width * s->desc.max_height;
    if ((st = bwd_alloc(s, &s->bwd_ssim, 3 * P3 + 4)) != HYRF_OK) return st;
    float win[11], sum = 0.0f;
    for (int k = 0; k < 11; ++k) { win[k] = expf(-(float)((k - 5) * (k - 5)) / (2.0f * 1.5f * 1.5f)); sum += win[k]; }
    for (int k = 0; k < 11; ++k) win[k] /= sum;
    if ((e = cudaMemcpyToSymbolAsync(c_win, win, sizeof(win), 0, cudaMemcpyHostToDevice, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyToSymbol");
    double* dloss = reinterpret_cast<double*>(s->bwd_ssim);   // [0, 2): the loss accumulator; the three maps follow
    float* maps = s->bwd_ssim + 2;
    if ((e = cudaMemsetAsync(dloss, 0, sizeof(double), s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemsetAsync(loss)");
    const dim3 grid((W + 15) / 16, (H + 15) / 16, 3);
    ssim_maps_kernel<<<grid, 256, 0, s->stream>>>(image, target, W, H, lambda, maps, dloss);
    if (g_image) ssim_grad_kernel<<<grid, 256, 0, s->stream>>>(image, target, W, H, lambda, maps, g_image);
    double l = 0.0;
    if ((e = cudaMemcpyAsync(&l, dloss, sizeof(double), cudaMemcpyDeviceToHost, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyAsync(loss)");
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(loss)");
    *loss_host = l + (double)lambda;   // the kernels summed (1 - lambda) L1 - lambda SSIM
    return HYRF_OK;
}

// ---- Eq. 12 once more, through an entry point that allocates nothing (include/hyrf.h hyrf_loss_l1_ssim_noalloc) ------------
// Same kernels, same arithmetic as hyrf_loss_l1_ssim; the scratch (the loss accumulator and the three derivative maps)
// is this file-scope array instead of a cudaMalloc'ed buffer of the scene. Every device that loads the library holds
// its own copy (37.7 MB) until the process exits. In HOST code the array's name is a host-side stand-in, not a device
// address: the kernels get the address cudaGetSymbolAddress returns, asked for once per device with that device
// current. All calls on a device share the array, and it keeps the last call's contents: the accumulator is cleared
// here before every use; the maps are completely rewritten by pass 1 (for the W x H of the call) before pass 2 reads them.
static __device__ __align__(256) float g_loss_scratch[4 + 9ull * HYRF_LOSS_NOALLOC_MAX_PIXELS];

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
float* g_noalloc_ptr[kNoAllocMaxDevices] = {};
}  // namespace

extern "C" hyrf_status hyrf_loss_l1_ssim_noalloc(int32_t device, void* cuda_stream, const float* image, const float* target,
                                                 int32_t W, int32_t H, float lambda, double* loss_host, float* g_image) {
    if (!image || !target || !loss_host) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim_noalloc: NULL argument");
    if (device < 0 || device >= kNoAllocMaxDevices) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim_noalloc: device %d", device);
    if (W < 1 || H < 1 || !(lambda >= 0.0f) || !(lambda <= 1.0f))
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim_noalloc: W x H = %d x %d, lambda = %g", W, H, (double)lambda);
    if ((uint64_t)W * (uint64_t)H > (uint64_t)HYRF_LOSS_NOALLOC_MAX_PIXELS)
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_loss_l1_ssim_noalloc: %d x %d = %llu pixels exceed the built-in scratch of %u pixels "
                       "(HYRF_LOSS_NOALLOC_MAX_PIXELS); use hyrf_loss_l1_ssim", W, H, (unsigned long long)W * (unsigned long long)H,
                       (unsigned)HYRF_LOSS_NOALLOC_MAX_PIXELS);
    cudaError_t e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    float* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mu);
        if (!g_noalloc_ptr[device]) {
            void* p = nullptr;
            if ((e = cudaGetSymbolAddress(&p, g_loss_scratch)) != cudaSuccess) return hy_cuda_fail(e, "cudaGetSymbolAddress(g_loss_scratch)");
            g_noalloc_ptr[device] = static_cast<float*>(p);
        }
        scratch = g_noalloc_ptr[device];
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    float win[11], sum = 0.0f;
    for (int k = 0; k < 11; ++k) { win[k] = expf(-(float)((k - 5) * (k - 5)) / (2.0f * 1.5f * 1.5f)); sum += win[k]; }
    for (int k = 0; k < 11; ++k) win[k] /= sum;
    if ((e = cudaMemcpyToSymbolAsync(c_win, win, sizeof(win), 0, cudaMemcpyHostToDevice, st)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyToSymbol");
    double* dloss = reinterpret_cast<double*>(scratch);   // [0, 4): the loss accumulator; the three maps follow
    float* maps = scratch + 4;
    if ((e = cudaMemsetAsync(dloss, 0, sizeof(double), st)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemsetAsync(loss)");
    const dim3 grid((W + 15) / 16, (H + 15) / 16, 3);
    ssim_maps_kernel<<<grid, 256, 0, st>>>(image, target, W, H, lambda, maps, dloss);
    if (g_image) ssim_grad_kernel<<<grid, 256, 0, st>>>(image, target, W, H, lambda, maps, g_image);
    if ((e = cudaGetLastError()) != cudaSuccess) return hy_cuda_fail(e, "ssim kernels");
    double l = 0.0;
    if ((e = cudaMemcpyAsync(&l, dloss, sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyAsync(loss)");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(loss)");
    *loss_host = l + (double)lambda;   // the kernels summed (1 - lambda) L1 - lambda SSIM
    return HYRF_OK;
}
