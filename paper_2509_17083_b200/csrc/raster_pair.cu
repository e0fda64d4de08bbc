// raster_pair.cu — S5, packed-fp32 variant of the per-warp-list rasterizer (raster_warp.cu): the same arithmetic, bit
// for bit (DESIGN.md §2 D10: every product and fused multiply-add of the oracle's order, IEEE round-to-nearest), with
// TWO pixels per lane evaluated by Blackwell's two-wide fp32 instructions (fma.rn.f32x2 / mul.rn.f32x2 / add.rn.f32x2
// -> FFMA2 / FMUL2 / FADD2: two independent IEEE operations per lane in ONE issue slot).
//
// Why: the blend loop is bound by instruction issue, not by the fp32 pipes (profiles/r2: 30 issued instructions per
// (pixel, Gaussian) pair of which 19 are fp32 arithmetic; the probe of csrc/probe.cu puts FFMA2 at 2.0 per clock and SM
// against 4.0 for FFMA: same flops, half the issue slots). With two pixels per lane the arithmetic of a pair of
// pairs is 17 two-wide instructions instead of 2 x 19, the staged record is read once for both, and only the
// compare / select tail stays per pixel: ~39 issue slots per entry and lane instead of ~61.
//
// Layout: one CTA of 128 threads per 16 x 16 tile; a warp owns an 8 x 8 pixel block = two stacked 8 x 4 blocks, a lane
// the pixels (x, y) and (x, y + 4) of it. The per-warp lists are built as in raster_warp.cu, from 4-bit masks over the
// 8 x 8 blocks. Staged records hold every
// field TWICE (u u | v v | A A | -B -B | C C | o o | r r | g g | b b) so that each 16-byte shared-memory load
// delivers two ready-made two-wide operands. -B is stored instead of B: -((B dx) dy) == ((-B) dx) dy exactly.
#include "raster_common.cuh"
#include "scene.h"

namespace {

constexpr int kThreads = 128;
constexpr int kWarps = kThreads / 32;
constexpr int kStage = 256;                        // staged records per round
constexpr uint32_t kRecBytes = 80;                 // 9 fields x 2 x 4 B = 72, padded to a multiple of 16
constexpr uint32_t kNullSlot = kStage;             // a null record (opacity 0 -> alpha 0 -> skipped)

typedef unsigned long long f2;                     // two binary32 values in one 64-bit register pair (.x low, .y high)

__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float lo(f2 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return a; }
__device__ __forceinline__ float hi(f2 v) { float a, b; asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); return b; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// ALL: every warp blends every staged record (no block masks, no per-warp lists): for splats that cover many tiles
// nearly every 8 x 8 block is reached anyway (raster.cu's case), and what remains is this kernel's two-pixels-per-lane loop.
template <bool ALL>
__global__ void __launch_bounds__(kThreads)
raster_pair_kernel(const uint2* __restrict__ ranges, const uint32_t* __restrict__ list, const float4* __restrict__ rec,
                   int W, int H, int gx, float tau_T, float* __restrict__ out_rgb, float* __restrict__ finalT,
                   uint32_t* __restrict__ bg_list, FrameCounters* __restrict__ counters, uint8_t* __restrict__ bg_mask,
                   float* __restrict__ dbg_fg, const uint32_t* __restrict__ tile_queue, const uint4* __restrict__ rect,
                   int mshift, int mgx, uint32_t* __restrict__ dbg_list, const uint2* __restrict__ dbg_ranges, uint32_t* __restrict__ dbg_len,
        int ty0, int ty1) {
    __shared__ __align__(16) uint8_t s_rec[(kStage + 1) * kRecBytes];
    __shared__ __align__(16) uint16_t s_widx[kWarps][kStage + 8];   // per warp: byte offsets of the records it blends
    __shared__ uint8_t s_mask[kStage];       // per staged record: bit w set when warp w's 8 x 8 block can reach it
    __shared__ uint32_t s_ids[kStage];       // ids waiting for stage B
    __shared__ uint32_t s_cnt[kWarps];
    const int tile = tile_queue ? (int)tile_queue[blockIdx.x] : (int)blockIdx.x;
    const int tx = tile % gx, ty = tile / gx;
    if (ty < ty0 || ty >= ty1) return;   // screen strips (hyrf_set_strip): another device's tile rows
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const int px = tx * HY_TILE + (int)(warp & 1u) * 8 + (int)(lane & 7u);
    const int py0 = ty * HY_TILE + (int)(warp >> 1) * 8 + (int)(lane >> 3), py1 = py0 + 4;
    const bool in0 = px < W && py0 < H, in1 = px < W && py1 < H;
    const f2 fi = pk((float)px, (float)px), fj = pk((float)py0, (float)py1);
    const float X0 = (float)(tx * HY_TILE), Y0 = (float)(ty * HY_TILE);
    const float X1 = fminf(X0 + (float)(HY_TILE - 1), (float)(W - 1)), Y1 = fminf(Y0 + (float)(HY_TILE - 1), (float)(H - 1));
    const uint2 rg = ranges[mshift ? (ty >> mshift) * mgx + (tx >> mshift) : tile];
    uint32_t dbg_pos = dbg_list ? dbg_ranges[tile].x : 0u;   // debug export of the per-tile list this CTA consumed
    f2 T = pk(1.0f, 1.0f), C0 = pk(0.0f, 0.0f), C1 = C0, C2 = C0;
    bool done0 = !in0, done1 = !in1;
    uint32_t b0 = rg.x;
    uint32_t g_next = 0;
    uint4 rc_next = make_uint4(0, 0, 0, 0);
    if (b0 + threadIdx.x < rg.y) {
        g_next = list[b0 + threadIdx.x];
        if (mshift) rc_next = __ldg(rect + g_next);
    }
    if (threadIdx.x < kRecBytes / 16) reinterpret_cast<uint4*>(s_rec + kNullSlot * kRecBytes)[threadIdx.x] = make_uint4(0u, 0u, 0u, 0u);
    const f2 kHalf = pk(-0.5f, -0.5f), kLog2e = pk(1.44269504f, 1.44269504f), kOne = pk(1.0f, 1.0f), kMinus1 = pk(-1.0f, -1.0f);
    while (b0 < rg.y) {
        // every pixel terminated: stop — unless the per-tile list is being exported, which needs the whole list walked
        const bool all_done = __syncthreads_count(done0 && done1) == kThreads;
        if (all_done && (!dbg_list || dbg_len)) break;
        // stage A: walk the list in chunks of 128 entries and collect, in order, the ids that belong to THIS tile until
        // at least 128 are waiting (at most 255)
        uint32_t nh = 0;
        while (b0 < rg.y && nh < (uint32_t)kThreads) {
            const uint32_t q = b0 + threadIdx.x;
            bool hit = false;
            const uint32_t g = g_next;
            const uint4 rc = rc_next;
            {   // the id and rectangle of the NEXT chunk's entry travel while this chunk is handled
                const uint32_t qn = q + kThreads;
                if (qn < rg.y) {
                    g_next = list[qn];
                    if (mshift) rc_next = __ldg(rect + g_next);
                }
            }
            if (q < rg.y)
                hit = !mshift || ((uint32_t)tx >= rc.x && (uint32_t)tx < rc.y && (uint32_t)ty >= rc.z && (uint32_t)ty < rc.w);
            const uint32_t balh = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_cnt[warp] = __popc(balh);
            __syncthreads();
            uint32_t ph = __popc(balh & ((1u << lane) - 1u)), tot = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = s_cnt[w];
                ph += (w < (int)warp) ? c : 0u;
                tot += c;
            }
            if (hit) {
                s_ids[nh + ph] = g;
                if (dbg_list) dbg_list[dbg_pos + ph] = g;   // debug export: the per-tile list exactly as consumed
            }
            nh += tot;
            dbg_pos += tot;
            b0 += kThreads;
            __syncthreads();
        }
        // stage B: the records of those ids; the ones that cannot reach alpha >= 1/255 anywhere in the tile are dropped
        uint32_t cnt = 0;
        for (uint32_t i0 = 0; i0 < nh; i0 += kThreads) {
            const uint32_t i = i0 + threadIdx.x;
            bool keep = false;
            float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
            float r2 = 0.0f;
            uint32_t wmask = 0;
            if (i < nh) {
                const uint32_t g = s_ids[i];
                r0 = __ldg(rec + 3ull * g);
                r1 = __ldg(rec + 3ull * g + 1);
                r2 = __ldg(reinterpret_cast<const float*>(rec + 3ull * g + 2));
                keep = entry_reaches_tile(r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, X0, X1, Y0, Y1);
                if (!ALL && keep) wmask = entry_block_mask4(r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, X0, Y0, W, H);   // which warps' 8 x 8 blocks?
            }
            const uint32_t bal = __ballot_sync(0xffffffffu, keep);
            if (lane == 0) s_cnt[warp] = __popc(bal);
            __syncthreads();
            uint32_t pos = cnt + __popc(bal & ((1u << lane) - 1u));
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = s_cnt[w];
                pos += (w < (int)warp) ? c : 0u;
                cnt += c;
            }
            if (keep) {   // (u u v v) (A A -B -B) (C C o o) (r r g g) (b b)
                float4* o = reinterpret_cast<float4*>(s_rec + pos * kRecBytes);
                o[0] = make_float4(r0.x, r0.x, r0.y, r0.y);
                o[1] = make_float4(r0.z, r0.z, -r0.w, -r0.w);
                o[2] = make_float4(r1.x, r1.x, r1.y, r1.y);
                o[3] = make_float4(r1.z, r1.z, r1.w, r1.w);
                *reinterpret_cast<float2*>(o + 4) = make_float2(r2, r2);
                if (!ALL) s_mask[pos] = (uint8_t)wmask;
            }
            __syncthreads();
        }
        // this warp's list: byte offsets of the staged records its 8 x 8 block can reach, in order, padded to a
        // multiple of 4 with the null record
        uint32_t n_w = ALL ? cnt : 0u;
        for (uint32_t i0 = 0; !ALL && i0 < cnt; i0 += 32) {
            const uint32_t i = i0 + lane;
            const bool h = i < cnt && ((s_mask[i] >> warp) & 1u);
            const uint32_t bal = __ballot_sync(0xffffffffu, h);
            if (h) s_widx[warp][n_w + __popc(bal & ((1u << lane) - 1u))] = (uint16_t)(i * kRecBytes);
            n_w += __popc(bal);
        }
        if (!ALL && lane < 4 && n_w + lane < ((n_w + 3u) & ~3u)) s_widx[warp][n_w + lane] = (uint16_t)(kNullSlot * kRecBytes);
        __syncwarp();
        // blend: branch-free per entry, two pixels per lane; a warp leaves as soon as all of its 64 pixels have terminated
        for (uint32_t k0 = 0; k0 < n_w && !all_done; k0 += 4) {
            if (__all_sync(0xffffffffu, done0 && done1)) break;
            uint2 offs = make_uint2(0u, 0u);
            if (!ALL) offs = *reinterpret_cast<const uint2*>(&s_widx[warp][k0]);
            const uint32_t ow[2] = {offs.x, offs.y};
#pragma unroll
            for (uint32_t k = 0; k < 4; ++k) {
                const uint8_t* r = ALL ? s_rec + (k0 + k < cnt ? k0 + k : kNullSlot) * kRecBytes
                                       : s_rec + ((k & 1u) ? (ow[k >> 1] >> 16) : (ow[k >> 1] & 0xFFFFu));
                const ulonglong2 a0 = *reinterpret_cast<const ulonglong2*>(r);        // (u u) (v v)
                const ulonglong2 a1 = *reinterpret_cast<const ulonglong2*>(r + 16);   // (A A) (-B -B)
                const ulonglong2 a2 = *reinterpret_cast<const ulonglong2*>(r + 32);   // (C C) (o o)
                const ulonglong2 a3 = *reinterpret_cast<const ulonglong2*>(r + 48);   // (r r) (g g)
                const f2 a4 = *reinterpret_cast<const f2*>(r + 64);                   // (b b)
                // D10, in the oracle's operation order, two pixels at a time
                const f2 dx = fma2(fi, kMinus1, a0.x), dy = fma2(fj, kMinus1, a0.y);          // u - i, v - j (exact product)
                const f2 q = fma2(mul2(a1.x, dx), dx, mul2(mul2(a2.x, dy), dy));              // fma(A dx, dx, (C dy) dy)
                const f2 power = fma2(kHalf, q, mul2(mul2(a1.y, dx), dy));                    // fma(-0.5, q, -((B dx) dy))
                const f2 arg = mul2(power, kLog2e);
                const f2 e = pk(ex2_ftz(lo(arg)), ex2_ftz(hi(arg)));
                const f2 oe = mul2(a2.y, e);
                const float al0 = fminf(0.99f, lo(oe)), al1 = fminf(0.99f, hi(oe));
                const f2 alpha = pk(al0, al1);
                const f2 Tn = mul2(T, fma2(alpha, kMinus1, kOne));                            // T (1 - alpha)
                const f2 aT = mul2(alpha, T);
                const bool v0 = !done0 && !(lo(power) > 0.0f) && !(al0 < 1.0f / 255.0f);
                const bool v1 = !done1 && !(hi(power) > 0.0f) && !(al1 < 1.0f / 255.0f);
                const bool s0 = v0 && (lo(Tn) < 1e-4f), s1 = v1 && (hi(Tn) < 1e-4f);
                const bool bl0 = v0 && !s0, bl1 = v1 && !s1;
                done0 = done0 || s0; done1 = done1 || s1;
                const f2 wgt = pk(bl0 ? lo(aT) : 0.0f, bl1 ? hi(aT) : 0.0f);
                C0 = fma2(a3.x, wgt, C0);
                C1 = fma2(a3.y, wgt, C1);
                C2 = fma2(a4, wgt, C2);
                T = pk(bl0 ? lo(Tn) : lo(T), bl1 ? hi(Tn) : hi(T));
            }
        }
    }
    // retained lists (hyrf_set_retain_lists): how much of this tile's list was written before every pixel had terminated
    if (dbg_len && threadIdx.x == 0) dbg_len[tile] = dbg_pos - dbg_ranges[tile].x;
    const float Tv[2] = {lo(T), hi(T)};
    const float Cv[2][3] = {{lo(C0), lo(C1), lo(C2)}, {hi(C0), hi(C1), hi(C2)}};
    const int pys[2] = {py0, py1};
    const bool ins[2] = {in0, in1};
    // S6 work list: pixels with T > tau_T, appended with one atomic per warp (order arbitrary)
    bool want[2];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        want[p] = ins[p] && Tv[p] > tau_T;
        if (ins[p]) {
            const size_t o = (size_t)pys[p] * W + px;
            out_rgb[3 * o] = Cv[p][0]; out_rgb[3 * o + 1] = Cv[p][1]; out_rgb[3 * o + 2] = Cv[p][2];
            finalT[o] = Tv[p];
            if (dbg_fg) { dbg_fg[3 * o] = Cv[p][0]; dbg_fg[3 * o + 1] = Cv[p][1]; dbg_fg[3 * o + 2] = Cv[p][2]; }
            if (bg_mask) bg_mask[o] = want[p] ? 1 : 0;
        }
    }
    const uint32_t bg0 = __ballot_sync(0xffffffffu, want[0]), bg1 = __ballot_sync(0xffffffffu, want[1]);
    if (bg0 | bg1) {
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(&counters->n_bg, (uint32_t)(__popc(bg0) + __popc(bg1)));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (want[0]) bg_list[base + __popc(bg0 & ((1u << lane) - 1u))] = (uint32_t)(py0 * W + px);
        if (want[1]) bg_list[base + __popc(bg0) + __popc(bg1 & ((1u << lane) - 1u))] = (uint32_t)(py1 * W + px);
    }
}

}  // namespace

void hy_launch_raster_pair(hyrf_scene* s, const FrameDev& f, const uint2* ranges, const uint32_t* list, bool macro,
                           float* out_rgb, uint32_t* launches, const uint32_t* tile_queue, uint32_t* dbg_list, uint32_t* dbg_len,
                           bool all) {
    const unsigned grid = (unsigned)(f.gx * f.gy);
    const bool want_fg = (s->debug_mask >> HYRF_DBG_FG) & 1u;
    const bool want_mask = (s->debug_mask >> HYRF_DBG_BG_MASK) & 1u;
    const float tau = (f.ablation & HYRF_ABL_NO_BG) ? INFINITY : f.tau_T;   // no background: empty S6 list
    auto kern = all ? raster_pair_kernel<true> : raster_pair_kernel<false>;
    kern<<<grid, kThreads, 0, s->stream>>>(ranges, list, s->rec, f.W, f.H, f.gx, tau, out_rgb, s->finalT,
                                                         s->bg_list, s->counters, want_mask ? s->bg_mask : nullptr,
                                                         want_fg ? s->fg : nullptr, tile_queue, s->rect,
                                                         macro ? f.mshift : 0, f.mgx, dbg_list, s->ranges, dbg_len, f.ty0, f.ty1);
    ++*launches;
}
