// raster_backward.cu — backward of S5 (DESIGN.md §2 D12, first piece): gradients of a loss with
// respect to the projected records (u, v, A, B, C, o, r, g, b) of the visible Gaussians, given dL/dC_fg and
// dL/dT_final per pixel, with the forward pass's decisions frozen. The training of PAPER.md:136-142 back-propagates
// through the 3DGS rasterizer the paper defers to (:108); this is that step for the pass of raster.cu.
//
// One CTA per tile, one thread per pixel, over the tile's own depth-ordered list (the per-tile lists the forward
// keeps under hyrf_set_retain_lists, or exports whole under HYRF_DBG_TILE_LIST | HYRF_DBG_TILE_RANGES). Phase 1 replays D10 with the forward's
// exact binary32 operations (same ex2.approx, same order, hence the same decisions) to find, per pixel, the end of its
// blended prefix and its final T. Phase 2 walks the list backwards in staged batches: alpha is recomputed, the
// transmittance in front of a pair is recovered as T_k = T_{k+1} / (1 - alpha_k) (alpha <= 0.99 bounds the
// amplification), the colour behind it is the running suffix sum. The nine per-pair contributions are reduced over
// the warp with 12 shuffles (halving exchange) and added to the Gaussian's row with one atomic per value and warp. HBM traffic is small
// (records re-read per tile, as in the forward); the kernel is bound by ALU issue and shuffles.
#include "raster_common.cuh"
#include "scene.h"

namespace {

constexpr int kBatch = HY_TILE * HY_TILE;

// D10 for one pair: returns false when the pair is skipped; alpha and e = exp(power) otherwise (operations and order of
// raster.cu's blend loop)
__device__ __forceinline__ bool pair_alpha(const float4 a0, float C, float o, float fi, float fj, float& alpha, float& e,
                                           float& dx, float& dy) {
    dx = __fsub_rn(a0.x, fi);
    dy = __fsub_rn(a0.y, fj);
    const float power = __fmaf_rn(-0.5f, __fmaf_rn(__fmul_rn(a0.z, dx), dx, __fmul_rn(__fmul_rn(C, dy), dy)),
                                  -__fmul_rn(__fmul_rn(a0.w, dx), dy));
    e = ex2_ftz(__fmul_rn(power, 1.44269504f));
    alpha = fminf(0.99f, __fmul_rn(o, e));
    return !(power > 0.0f) && !(alpha < 1.0f / 255.0f);
}

__global__ void __launch_bounds__(kBatch)
raster_backward_kernel(const uint2* __restrict__ ranges, const uint32_t* __restrict__ list_len, const uint32_t* __restrict__ list,
                       const float4* __restrict__ rec, int W, int H, int gx, const float* __restrict__ g_cfg,
                       const float* __restrict__ g_T, float* __restrict__ grad) {
    __shared__ float4 s_r0[kBatch];   // (u, v, A, B)
    __shared__ float4 s_r1[kBatch];   // (C, opacity, r, g)
    __shared__ float s_b[kBatch];
    __shared__ uint32_t s_id[kBatch];
    const int tile = (int)blockIdx.x;
    const int tx = tile % gx, ty = tile / gx;
    const uint32_t lane = threadIdx.x & 31u;
    // a warp owns an 8 x 4 pixel block (not 16 x 2 rows): more entries miss a whole block, and those cost it only the test
    const uint32_t warp = threadIdx.x >> 5;
    const int px = tx * HY_TILE + (int)(warp & 1u) * 8 + (int)(lane & 7u);
    const int py = ty * HY_TILE + (int)(warp >> 1) * 4 + (int)(lane >> 3);
    const bool inside = px < W && py < H;
    const float fi = (float)px, fj = (float)py;
    const uint2 rg = ranges[tile];
    // retained lists end where the forward's tile stopped walking (every pixel terminated): nothing behind that point was blended
    const uint32_t len = list_len ? min(rg.y - rg.x, list_len[tile]) : rg.y - rg.x;

    // phase 1: the forward's decisions -> n_mine = length of this pixel's blended prefix of the list, T = its final T
    float T = 1.0f;
    uint32_t n_mine = 0;
    bool done = !inside;
    for (uint32_t b0 = 0; b0 < len; b0 += kBatch) {
        if (__syncthreads_count(done) == kBatch) break;
        const uint32_t i = b0 + threadIdx.x;
        if (i < len) {
            const uint32_t g = list[rg.x + i];
            s_r0[threadIdx.x] = __ldg(rec + 3ull * g);
            s_r1[threadIdx.x] = __ldg(rec + 3ull * g + 1);
        }
        __syncthreads();
        const uint32_t nb = min((uint32_t)kBatch, len - b0);
        for (uint32_t k = 0; k < nb && !done; ++k) {
            float alpha, e, dx, dy;
            if (!pair_alpha(s_r0[k], s_r1[k].x, s_r1[k].y, fi, fj, alpha, e, dx, dy)) continue;
            const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
            if (Tn < 1e-4f) { done = true; break; }
            T = Tn;
            n_mine = b0 + k + 1;
        }
    }
    const float Tfin = T;
    float gc0 = 0.0f, gc1 = 0.0f, gc2 = 0.0f, gT = 0.0f;
    if (inside) {
        const size_t o = (size_t)py * W + px;
        gc0 = g_cfg[3 * o]; gc1 = g_cfg[3 * o + 1]; gc2 = g_cfg[3 * o + 2];
        gT = g_T[o];
    }
    // the longest prefix of the tile bounds the walk
    __shared__ uint32_t s_max;
    if (threadIdx.x == 0) s_max = 0;
    __syncthreads();
    atomicMax(&s_max, n_mine);
    __syncthreads();
    const uint32_t n_tile = s_max;

    // phase 2: back to front
    float S0 = 0.0f, S1 = 0.0f, S2 = 0.0f;   // colour behind the current pair
    const uint32_t n_batches = (n_tile + kBatch - 1) / kBatch;
    for (uint32_t bi = n_batches; bi-- > 0;) {
        const uint32_t b0 = bi * kBatch;
        __syncthreads();
        const uint32_t i = b0 + threadIdx.x;
        if (i < n_tile) {
            const uint32_t g = list[rg.x + i];
            s_id[threadIdx.x] = g;
            s_r0[threadIdx.x] = __ldg(rec + 3ull * g);
            s_r1[threadIdx.x] = __ldg(rec + 3ull * g + 1);
            s_b[threadIdx.x] = __ldg(reinterpret_cast<const float*>(rec + 3ull * g + 2));
        }
        __syncthreads();
        const uint32_t nb = min((uint32_t)kBatch, n_tile - b0);
        for (uint32_t k = nb; k-- > 0;) {
            const float4 a0 = s_r0[k];
            const float4 a1 = s_r1[k];
            const float cb = s_b[k];
            float alpha, e, dx, dy;
            const bool mine = (b0 + k < n_mine) && pair_alpha(a0, a1.x, a1.y, fi, fj, alpha, e, dx, dy);
            if (!__any_sync(0xffffffffu, mine)) continue;
            float v[9];
#pragma unroll
            for (int j = 0; j < 9; ++j) v[j] = 0.0f;
            if (mine) {
                const float iom = __frcp_rn(1.0f - alpha);   // one reciprocal serves the four quotients (1 - alpha >= 0.01)
                const float Tk = T * iom;                    // transmittance in front of this pair
                const float w = alpha * Tk;
                const float da = gc0 * (a1.z * Tk - S0 * iom) + gc1 * (a1.w * Tk - S1 * iom) + gc2 * (cb * Tk - S2 * iom) -
                                 gT * Tfin * iom;
                v[6] = w * gc0; v[7] = w * gc1; v[8] = w * gc2;
                S0 = fmaf(a1.z, w, S0); S1 = fmaf(a1.w, w, S1); S2 = fmaf(cb, w, S2);
                T = Tk;
                if (!(a1.y * e > 0.99f)) {        // not clamped
                    const float dP = alpha * da;
                    v[0] = -(a0.z * dx + a0.w * dy) * dP;
                    v[1] = -(a1.x * dy + a0.w * dx) * dP;
                    v[2] = -0.5f * dx * dx * dP;
                    v[3] = -dx * dy * dP;
                    v[4] = -0.5f * dy * dy * dP;
                    v[5] = e * da;
                }
            }
            // nine sums over the warp in 12 shuffles instead of 45: at every step a lane keeps one half of its values and
            // hands the other half to its partner (5 + 3 + 2 + 1 exchanges), then one plain step; the lane ends with value
            // number idx (padding slots are zero and dropped)
            const bool h16 = lane & 16u, h8 = lane & 8u, h4 = lane & 4u, h2 = lane & 2u;
            float a[5], b[3], c[2], d;
#pragma unroll
            for (int i = 0; i < 5; ++i) {
                const float hi = i < 4 ? v[5 + i] : 0.0f;
                a[i] = (h16 ? hi : v[i]) + __shfl_xor_sync(0xffffffffu, h16 ? v[i] : hi, 16);
            }
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const float hi = i < 2 ? a[3 + i] : 0.0f;
                b[i] = (h8 ? hi : a[i]) + __shfl_xor_sync(0xffffffffu, h8 ? a[i] : hi, 8);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const float hi = i < 1 ? b[2] : 0.0f;
                c[i] = (h4 ? hi : b[i]) + __shfl_xor_sync(0xffffffffu, h4 ? b[i] : hi, 4);
            }
            d = (h2 ? c[1] : c[0]) + __shfl_xor_sync(0xffffffffu, h2 ? c[0] : c[1], 2);
            d += __shfl_xor_sync(0xffffffffu, d, 1);
            const uint32_t idx = (h16 ? 5u : 0u) + (h8 ? 3u : 0u) + (h4 ? 2u : 0u) + (h2 ? 1u : 0u);
            const bool holds = !(lane & 1u) && !(h4 && h2) && !(h8 && h4) && idx < 9u;
            if (holds) atomicAdd(grad + 9ull * s_id[k] + idx, d);
        }
    }
}

}  // namespace

// Enqueues the backward of the last rendered frame on the scene's stream. grad: DEVICE float [V][9], zeroed here.
hyrf_status hy_launch_raster_backward(hyrf_scene* s, const float* g_cfg, const float* g_T, float* grad,
                                      uint32_t* launches) {
    const int W = s->lastW, H = s->lastH;
    const int gx = (W + HY_TILE - 1) / HY_TILE, gy = (H + HY_TILE - 1) / HY_TILE;
    cudaError_t e = cudaMemsetAsync(grad, 0, (size_t)s->lastV * 9 * sizeof(float), s->stream);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaMemsetAsync(grad)");
    raster_backward_kernel<<<(unsigned)(gx * gy), kBatch, 0, s->stream>>>(s->ranges, s->list_partial ? s->list_len : nullptr, s->list_final, s->rec, W, H, gx, g_cfg,
                                                                          g_T, grad);
    if ((e = cudaGetLastError()) != cudaSuccess) return hy_cuda_fail(e, "raster_backward_kernel");
    ++*launches;
    return HYRF_OK;
}
