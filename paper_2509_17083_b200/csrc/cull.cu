// cull.cu — S1: visibility pre-culling against the camera frustum + order-preserving compaction.
// PAPER.md:112–122 (Eq. 8–9): eliminate points that will not project into the image frame BEFORE the neural
// fields are queried. Arithmetic: DESIGN.md §2 D1. HBM-bound streaming: 12 B read per stored Gaussian,
// 4 B written per visible one; warp ballots give the stable (id-ordered) compaction the depth tie-break needs.
#include "scene.h"

namespace {

constexpr int kCullThreads = 256;
constexpr int kCullItems = 1024;  // per block: 4 coalesced sweeps of 256

__global__ void __launch_bounds__(kCullThreads)
cull_mark_kernel(const float* __restrict__ pos, uint32_t N, FrameDev f, uint32_t* __restrict__ flag_words,
                 uint32_t* __restrict__ block_counts, uint8_t* __restrict__ dbg_mask) {
    __shared__ uint32_t warp_cnt[kCullThreads / 32];
    const uint32_t base = blockIdx.x * kCullItems;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t cnt = 0;
#pragma unroll
    for (int k = 0; k < kCullItems / kCullThreads; ++k) {
        const uint32_t i = base + k * kCullThreads + threadIdx.x;
        bool keep = false;
        if (i < N) {
            const float px = __ldg(pos + i), py = __ldg(pos + N + i), pz = __ldg(pos + 2ull * N + i);
            float X, Y, Z;
            hy_to_camera(f, px, py, pz, X, Y, Z);
            keep = (Z > f.z_near) && (fabsf(X) <= __fmul_rn(f.limx, Z)) && (fabsf(Y) <= __fmul_rn(f.limy, Z));
            if (dbg_mask) dbg_mask[i] = keep ? 1 : 0;
        }
        const uint32_t bal = __ballot_sync(0xffffffffu, keep);
        if (lane == 0) {
            const uint32_t word = (base >> 5) + k * (kCullThreads / 32) + warp;
            if (word * 32u < N) flag_words[word] = bal;
            cnt += __popc(bal);
        }
    }
    if (lane == 0) warp_cnt[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < kCullThreads / 32; ++w) s += warp_cnt[w];
        block_counts[blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(kCullThreads)
cull_compact_kernel(const uint32_t* __restrict__ flag_words, const uint32_t* __restrict__ block_offs,
                    const uint32_t* __restrict__ block_counts, uint32_t N, uint32_t* __restrict__ vis_idx,
                    FrameCounters* __restrict__ counters) {
    __shared__ uint32_t word_prefix[kCullItems / 32];
    const uint32_t base = blockIdx.x * kCullItems;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) {  // 32 words per block: exclusive scan of their popcounts by one warp
        const uint32_t word = (base >> 5) + lane;
        const uint32_t c = (word * 32u < N) ? __popc(flag_words[word]) : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= (uint32_t)d) incl += v;
        }
        word_prefix[lane] = incl - c;
    }
    __syncthreads();
    const uint32_t boff = block_offs[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kCullItems / kCullThreads; ++k) {
        const uint32_t wl = k * (kCullThreads / 32) + warp;
        const uint32_t word = (base >> 5) + wl;
        if (word * 32u >= N) continue;
        const uint32_t bits = flag_words[word];
        if ((bits >> lane) & 1u) {
            const uint32_t rank = boff + word_prefix[wl] + __popc(bits & ((1u << lane) - 1u));
            vis_idx[rank] = base + k * kCullThreads + threadIdx.x;
        }
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        counters->V = boff + block_counts[blockIdx.x];
        counters->D = 0ull;
        counters->n_bg = 0u;
        counters->bin_ticket = 0u;
        counters->bin_done = 0u;
    }
}

}  // namespace

void hy_launch_cull(hyrf_scene* s, const FrameDev& f, uint32_t* launches) {
    const uint32_t nb = (s->N + kCullItems - 1) / kCullItems;
    uint32_t* counts = s->block_counts;
    uint32_t* offs = s->block_counts + nb;
    const bool want_mask = (s->debug_mask >> HYRF_DBG_VIS_MASK) & 1u;
    cull_mark_kernel<<<nb, kCullThreads, 0, s->stream>>>(s->pos, s->N, f, s->flag_words, counts,
                                                         want_mask ? s->dbg_vis_mask : nullptr);
    ++*launches;
    hy_launch_scan(counts, offs, nb, s->scan_scratch, s->stream, launches);
    cull_compact_kernel<<<nb, kCullThreads, 0, s->stream>>>(s->flag_words, offs, counts, s->N, s->vis_idx,
                                                            s->counters);
    ++*launches;
}
