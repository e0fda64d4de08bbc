// raster.cu — S5: front-to-back alpha blending, Eq. 1, per 16x16 tile over its depth-ordered list.
// Arithmetic DESIGN.md §2 D10 (constants of the 3DGS rasterizer the paper defers to).
// One CTA per tile, one thread per pixel; list entries are staged through shared memory in batches of 256 so each
// projected record is fetched once per tile, and entries that cannot reach alpha >= 1/255 anywhere in the tile are
// dropped while staging (stable compaction, so the order is untouched). The per-pair body is branch-free
// (profiles/r1a: divergent skip/stop branches cost 45 issue slots per pair against ~30 predicated); warps stop
// when all of their pixels have terminated, the CTA when all warps have. Bound by plain fp32 ALU issue + one
// MUFU.EX2 per pair — no tensor cores (nothing here is a dense contraction).
#include "raster_common.cuh"
#include "scene.h"

namespace {

constexpr int kBatch = HY_TILE * HY_TILE;
constexpr int kWarps = kBatch / 32;

__global__ void __launch_bounds__(kBatch)
raster_kernel(const uint2* __restrict__ ranges, const uint32_t* __restrict__ list, const float4* __restrict__ rec,
              int W, int H, int gx, float tau_T, float* __restrict__ out_rgb, float* __restrict__ finalT,
              uint32_t* __restrict__ bg_list, FrameCounters* __restrict__ counters, uint8_t* __restrict__ bg_mask,
              float* __restrict__ dbg_fg, const uint32_t* __restrict__ tile_queue, const uint4* __restrict__ rect,
              int mshift, int mgx, uint32_t* __restrict__ dbg_list, const uint2* __restrict__ dbg_ranges, uint32_t* __restrict__ dbg_len,
        int ty0, int ty1) {
    __shared__ float4 s_r0[2 * kBatch + 8];   // (u, v, A, B)   (+ 8: padding to a multiple of 8)
    __shared__ float4 s_r1[2 * kBatch + 8];   // (C, opacity, r, g)
    __shared__ float s_b[2 * kBatch + 8];
    __shared__ uint32_t s_ids[2 * kBatch];    // ids waiting for stage B
    __shared__ uint32_t s_wcnt[kWarps];
    __shared__ uint32_t s_hcnt[kWarps];
    // tiles are taken longest list first (queue built by bin_ordered.cu), so the heavy tiles do not form the tail
    const int tile = tile_queue ? (int)tile_queue[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % gx, ty = tile / gx;
    if (ty < ty0 || ty >= ty1) return;   // screen strips (hyrf_set_strip): another device's tile rows
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const int px = tx * HY_TILE + (threadIdx.x & (HY_TILE - 1));
    const int py = ty * HY_TILE + (threadIdx.x >> 4);
    const bool inside = px < W && py < H;
    const float fi = (float)px, fj = (float)py;
    const float X0 = (float)(tx * HY_TILE), Y0 = (float)(ty * HY_TILE);
    const float X1 = fminf(X0 + (float)(HY_TILE - 1), (float)(W - 1)), Y1 = fminf(Y0 + (float)(HY_TILE - 1), (float)(H - 1));
    // mshift > 0: the lists are per MACRO tile (HY_MACRO x HY_MACRO tiles, depth-ordered); this tile's list is the
    // subsequence whose tile rectangle contains it, picked out while staging. mshift = 0: per-tile lists.
    const uint2 rg = ranges[mshift ? (ty >> mshift) * mgx + (tx >> mshift) : tile];
    uint32_t dbg_pos = dbg_list ? dbg_ranges[tile].x : 0u;   // debug export of the per-tile list this CTA consumed
    float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f;
    bool done = !inside;
    uint32_t b0 = rg.x;
    uint32_t g_next = 0;
    uint4 rc_next = make_uint4(0, 0, 0, 0);
    if (b0 + threadIdx.x < rg.y) {
        g_next = list[b0 + threadIdx.x];
        if (mshift) rc_next = __ldg(rect + g_next);
    }
    while (b0 < rg.y) {
        // every pixel terminated: stop — unless the per-tile list is being exported, which needs the whole list walked
        const bool all_done = __syncthreads_count(done) == kBatch;
        if (all_done && (!dbg_list || dbg_len)) break;
        // stage A: walk the list in chunks of 256 entries and collect, in order, the ids that belong to THIS tile (all of
        // them when the lists are per tile; about one in five when they are per macro tile) until 256 are waiting
        uint32_t nh = 0;
        while (b0 < rg.y && nh < (uint32_t)kBatch) {
            const uint32_t q = b0 + threadIdx.x;
            bool hit = false;
            const uint32_t g = g_next;
            const uint4 rc = rc_next;
            {   // the id and rectangle of the NEXT chunk's entry travel while this chunk is handled
                const uint32_t qn = q + kBatch;
                if (qn < rg.y) {
                    g_next = list[qn];
                    if (mshift) rc_next = __ldg(rect + g_next);
                }
            }
            if (q < rg.y)
                hit = !mshift || ((uint32_t)tx >= rc.x && (uint32_t)tx < rc.y && (uint32_t)ty >= rc.z && (uint32_t)ty < rc.w);
            const uint32_t balh = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_hcnt[warp] = __popc(balh);
            __syncthreads();
            uint32_t ph = __popc(balh & ((1u << lane) - 1u)), tot = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = s_hcnt[w];
                ph += (w < (int)warp) ? c : 0u;
                tot += c;
            }
            if (hit) {
                s_ids[nh + ph] = g;
                if (dbg_list) dbg_list[dbg_pos + ph] = g;   // debug export: the per-tile list exactly as consumed
            }
            nh += tot;
            dbg_pos += tot;
            b0 += kBatch;
            __syncthreads();
        }
        // stage B: the records of those ids; the ones that cannot reach alpha >= 1/255 anywhere in the tile are dropped
        uint32_t cnt = 0;
        for (uint32_t i0 = 0; i0 < nh; i0 += kBatch) {
            const uint32_t i = i0 + threadIdx.x;
            bool keep = false;
            float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
            float r2 = 0.0f;
            if (i < nh) {
                const uint32_t g = s_ids[i];
                r0 = __ldg(rec + 3ull * g);
                r1 = __ldg(rec + 3ull * g + 1);
                r2 = __ldg(reinterpret_cast<const float*>(rec + 3ull * g + 2));
                keep = entry_reaches_tile(r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, X0, X1, Y0, Y1);
            }
            const uint32_t bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0) s_wcnt[warp] = __popc(bal);
            __syncthreads();
            uint32_t pos = cnt + __popc(bal & ((1u << lane) - 1u));
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = s_wcnt[w];
                pos += (w < (int)warp) ? c : 0u;
                cnt += c;
            }
            if (keep) { s_r0[pos] = r0; s_r1[pos] = r1; s_b[pos] = r2; }
            __syncthreads();
        }
        // pad the staged list to a multiple of 8 with null entries (opacity 0 -> alpha 0 -> skipped), so the blend loop
        // runs in fixed groups of 8 with immediate shared-memory offsets
        if (threadIdx.x < 8 && cnt + threadIdx.x < ((cnt + 7u) & ~7u)) {
            s_r0[cnt + threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
            s_r1[cnt + threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
            s_b[cnt + threadIdx.x] = 0.0f;
        }
        __syncthreads();
        // blend: branch-free per pair; a warp leaves the batch as soon as all of its pixels have terminated
        for (uint32_t k0 = 0; k0 < cnt && !all_done; k0 += 8) {
            if (__all_sync(0xffffffffu, done)) break;
#pragma unroll
            for (uint32_t k = k0; k < k0 + 8; ++k) {
                const float4 a0 = s_r0[k];
                const float4 a1 = s_r1[k];
                const float dx = __fsub_rn(a0.x, fi), dy = __fsub_rn(a0.y, fj);
                const float power = __fmaf_rn(-0.5f, __fmaf_rn(__fmul_rn(a0.z, dx), dx, __fmul_rn(__fmul_rn(a1.x, dy), dy)),
                                              -__fmul_rn(__fmul_rn(a0.w, dx), dy));
                const float alpha = fminf(0.99f, __fmul_rn(a1.y, ex2_ftz(__fmul_rn(power, 1.44269504f))));
                const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                const bool valid = !done && !(power > 0.0f) && !(alpha < 1.0f / 255.0f);
                const bool stop = valid && (Tn < 1e-4f);
                const bool blend = valid && !stop;
                done = done || stop;
                const float wgt = blend ? __fmul_rn(alpha, T) : 0.0f;
                C0 = __fmaf_rn(a1.z, wgt, C0);
                C1 = __fmaf_rn(a1.w, wgt, C1);
                C2 = __fmaf_rn(s_b[k], wgt, C2);
                T = blend ? Tn : T;
            }
        }
    }
    // retained lists (hyrf_set_retain_lists): how much of this tile's list was written before every pixel had terminated
    if (dbg_len && threadIdx.x == 0) dbg_len[tile] = dbg_pos - dbg_ranges[tile].x;
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
    const uint32_t bgb = __ballot_sync(0xffffffffu, want_bg);
    if (bgb) {
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&counters->n_bg, (uint32_t)__popc(bgb));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (want_bg) bg_list[base + __popc(bgb & ((1u << lane) - 1u))] = (uint32_t)(py * W + px);
    }
}

}  // namespace

void hy_launch_raster(hyrf_scene* s, const FrameDev& f, const uint2* ranges, const uint32_t* list, bool macro,
                      float* out_rgb, uint32_t* launches, const uint32_t* tile_queue, uint32_t* dbg_list, uint32_t* dbg_len) {
    // Four kernels, the same bits (hyrf_set_raster_mode): 1 this file's (a pixel per thread, every warp blends every staged
    // entry), 2 per-warp lists over 8 x 4 blocks (raster_warp.cu), 3 per-warp lists over 8 x 8 blocks with two pixels per
    // lane on the two-wide fp32 instructions (raster_pair.cu), 4 the same two-pixel loop over every staged entry. Mode 0
    // chooses between 3 and 4 from the tiles touched per visible Gaussian in the previous frame: per-warp lists pay as long
    // as splats leave blocks of a tile untouched; when a splat covers ~100 tiles (the 4K points of config 5) nearly every
    // block is reached and the masks and lists are pure cost. Measured raster stage, mode 3 / 4 / 1: config 3 (10 tiles per
    // splat) 0.153 / 0.179 / 0.178 ms; 500k @ 1080p (35) 0.193 / 0.198 / 0.245; 4M @ 1080p (35) 0.229 / 0.236 / 0.281;
    // 500k @ 4K (120) 0.657 / 0.632 / 0.840; 4M @ 4K (117) 0.728 / 0.704 / 0.925.
    constexpr uint64_t kAllEntriesMinTilesPerSplat = 64;
    int mode = s->raster_mode;
    if (mode == 0) mode = (s->lastV != 0 && s->lastD > kAllEntriesMinTilesPerSplat * s->lastV) ? 4 : 3;
    s->last_raster_mode = mode;
    if (mode == 2) { hy_launch_raster_warp(s, f, ranges, list, macro, out_rgb, launches, tile_queue, dbg_list, dbg_len); return; }
    if (mode == 3 || mode == 4) {
        hy_launch_raster_pair(s, f, ranges, list, macro, out_rgb, launches, tile_queue, dbg_list, dbg_len, /*all=*/mode == 4);
        return;
    }
    const unsigned grid = (unsigned)(f.gx * f.gy);
    const bool want_fg = (s->debug_mask >> HYRF_DBG_FG) & 1u;
    const bool want_mask = (s->debug_mask >> HYRF_DBG_BG_MASK) & 1u;
    const float tau = (f.ablation & HYRF_ABL_NO_BG) ? INFINITY : f.tau_T;   // no background: empty S6 list
    raster_kernel<<<grid, kBatch, 0, s->stream>>>(ranges, list, s->rec, f.W, f.H, f.gx, tau, out_rgb, s->finalT,
                                                  s->bg_list, s->counters, want_mask ? s->bg_mask : nullptr,
                                                  want_fg ? s->fg : nullptr, tile_queue, s->rect,
                                                  macro ? f.mshift : 0, f.mgx, dbg_list, s->ranges, dbg_len, f.ty0, f.ty1);
    ++*launches;
}
