// raster.cu — S5: front-to-back alpha blending, Eq. 1, per 16x16 tile over its depth-ordered list.
// Arithmetic DESIGN.md §2 D10 (constants of the 3DGS rasterizer the paper defers to).
// One CTA per tile, one thread per pixel; list entries are staged through shared memory in batches of 256 so each
// projected record is fetched once per tile; the CTA stops as soon as every pixel has terminated. Bound by plain
// fp32 ALU issue + one MUFU.EX2 per pair — no tensor cores (nothing here is a dense contraction).
#include "scene.h"

namespace {

constexpr int kBatch = HY_TILE * HY_TILE;

__global__ void __launch_bounds__(kBatch)
raster_kernel(const uint2* __restrict__ ranges, const uint32_t* __restrict__ list, const float4* __restrict__ rec,
              int W, int H, int gx, float tau_T, float* __restrict__ out_rgb, float* __restrict__ finalT,
              uint32_t* __restrict__ bg_list, FrameCounters* __restrict__ counters, uint8_t* __restrict__ bg_mask,
              float* __restrict__ dbg_fg) {
    __shared__ float4 s_r0[kBatch];
    __shared__ float4 s_r1[kBatch];
    __shared__ float s_b[kBatch];
    const int tile = blockIdx.y * gx + blockIdx.x;
    const int px = blockIdx.x * HY_TILE + (threadIdx.x & (HY_TILE - 1));
    const int py = blockIdx.y * HY_TILE + (threadIdx.x >> 4);
    const bool inside = px < W && py < H;
    const float fi = (float)px, fj = (float)py;
    const uint2 rg = ranges[tile];
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f;
    bool done = !inside;
    for (uint32_t b0 = rg.x; b0 < rg.y; b0 += kBatch) {
        if (__syncthreads_count(done) == kBatch) break;
        const uint32_t q = b0 + threadIdx.x;
        if (q < rg.y) {
            const uint32_t g = list[q];
            s_r0[threadIdx.x] = __ldg(rec + 3ull * g);
            s_r1[threadIdx.x] = __ldg(rec + 3ull * g + 1);
            s_b[threadIdx.x] = __ldg(reinterpret_cast<const float*>(rec + 3ull * g + 2));
        }
        __syncthreads();
        const int cnt = min((int)kBatch, (int)(rg.y - b0));
        if (!done) {
            for (int k = 0; k < cnt; ++k) {
                const float4 r0 = s_r0[k];
                const float4 r1 = s_r1[k];
                const float dx = __fsub_rn(r0.x, fi), dy = __fsub_rn(r0.y, fj);
                const float power = __fmaf_rn(-0.5f, __fmaf_rn(__fmul_rn(r0.z, dx), dx, __fmul_rn(__fmul_rn(r1.x, dy), dy)),
                                              -__fmul_rn(__fmul_rn(r0.w, dx), dy));
                if (power > 0.0f) continue;
                const float alpha = fminf(0.99f, __fmul_rn(r1.y, __expf(power)));
                if (alpha < 1.0f / 255.0f) continue;
                const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                if (Tn < 1e-4f) { done = true; break; }
                const float wgt = __fmul_rn(alpha, T);
                C0 = __fmaf_rn(r1.z, wgt, C0);
                C1 = __fmaf_rn(r1.w, wgt, C1);
                C2 = __fmaf_rn(s_b[k], wgt, C2);
                T = Tn;
            }
        }
    }
    if (inside) {
        const size_t o = (size_t)py * W + px;
        out_rgb[3 * o] = C0; out_rgb[3 * o + 1] = C1; out_rgb[3 * o + 2] = C2;
        finalT[o] = T;
        if (dbg_fg) { dbg_fg[3 * o] = C0; dbg_fg[3 * o + 1] = C1; dbg_fg[3 * o + 2] = C2; }
    }
    // S6 work list: pixels with T > tau_T, appended with one atomic per warp. The order of the list is
    // arbitrary; the background of a pixel does not depend on it.
    const bool want_bg = inside && T > tau_T;
    if (inside && bg_mask) bg_mask[(size_t)py * W + px] = want_bg ? 1 : 0;
    const uint32_t bal = __ballot_sync(0xffffffffu, want_bg);
    if (bal) {
        const uint32_t lane = threadIdx.x & 31u;
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&counters->n_bg, (uint32_t)__popc(bal));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (want_bg) bg_list[base + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)(py * W + px);
    }
}

}  // namespace

void hy_launch_raster(hyrf_scene* s, const FrameDev& f, const uint32_t* list, float* out_rgb, uint32_t* launches) {
    dim3 grid((unsigned)f.gx, (unsigned)f.gy);
    const bool want_fg = (s->debug_mask >> HYRF_DBG_FG) & 1u;
    const bool want_mask = (s->debug_mask >> HYRF_DBG_BG_MASK) & 1u;
    raster_kernel<<<grid, kBatch, 0, s->stream>>>(s->ranges, list, s->rec, f.W, f.H, f.gx, f.tau_T, out_rgb, s->finalT,
                                                  s->bg_list, s->counters, want_mask ? s->bg_mask : nullptr,
                                                  want_fg ? s->fg : nullptr);
    ++*launches;
}
