// bin.cu — S4b: tile binning. PAPER.md:47 ("ordered by depth ... projected onto 2D image planes"), :57 (the set of
// sorted Gaussians projected onto the pixel); order defined in DESIGN.md §2 D9: (tile, depth bits, id) ascending.
// Design: Gaussians are first ordered by (depth bits, id) — V items — and emit their tile entries in that order;
// one stable sort of the D entries by tile id (only ceil(log2 tiles) key bits) then yields the final lists.
// That moves 8 B per entry per pass over 2 passes instead of 12 B over 6 passes of a 64-bit (tile|depth) key.
#include "scene.h"

namespace {

__global__ void depth_prepare_kernel(const uint32_t* __restrict__ depth_key, const FrameCounters* __restrict__ c,
                                     uint32_t* __restrict__ key, uint32_t* __restrict__ val, uint32_t N) {
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N || j >= c->V) return;
    key[j] = depth_key[j];
    val[j] = j;
}

// tt_sorted[k] = tiles touched by the k-th Gaussian in depth order (0 beyond V); counters->D += block sums.
__global__ void __launch_bounds__(256)
tiles_gather_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ tiles,
                    FrameCounters* __restrict__ c, uint32_t* __restrict__ tt_sorted, uint32_t N) {
    __shared__ unsigned long long wsum[8];
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t t = 0;
    if (k < N) {
        if (k < c->V) t = tiles[order[k]];
        tt_sorted[k] = t;
    }
    unsigned long long s = t;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long b = 0;
        for (int w = 0; w < 8; ++w) b += wsum[w];
        if (b) atomicAdd(&c->D, b);
    }
}

// One warp per Gaussian (in depth order): lanes stride over the rectangle's tiles.
__global__ void __launch_bounds__(256)
emit_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ offs, const uint4* __restrict__ rect,
            const uint32_t* __restrict__ tiles, uint32_t V, uint32_t gx, uint32_t* __restrict__ ent_key,
            uint32_t* __restrict__ ent_val) {
    const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= V) return;
    const uint32_t g = order[warp];
    const uint32_t nt = tiles[g];
    if (nt == 0) return;
    const uint4 rc = rect[g];
    const uint32_t w = rc.y - rc.x;
    const uint32_t base = offs[warp];
    for (uint32_t i = lane; i < nt; i += 32) {
        const uint32_t ty = rc.z + i / w, tx = rc.x + i % w;
        ent_key[base + i] = ty * gx + tx;
        ent_val[base + i] = g;
    }
}

__global__ void ranges_kernel(const uint32_t* __restrict__ keys, uint32_t D, uint2* __restrict__ ranges) {
    const uint32_t q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= D) return;
    const uint32_t t = keys[q];
    if (q == 0 || keys[q - 1] != t) ranges[t].x = q;
    if (q + 1 == D || keys[q + 1] != t) ranges[t].y = q + 1;
}

}  // namespace

void hy_launch_depth_prepare(hyrf_scene* s, uint32_t* launches) {
    depth_prepare_kernel<<<(s->N + 255) / 256, 256, 0, s->stream>>>(s->depth_key, s->counters, s->sort_a_key,
                                                                    s->sort_a_val, s->N);
    ++*launches;
}

void hy_launch_tiles_gather(hyrf_scene* s, const uint32_t* order, uint32_t* launches) {
    tiles_gather_kernel<<<(s->N + 255) / 256, 256, 0, s->stream>>>(order, s->tiles, s->counters, s->tt_sorted, s->N);
    ++*launches;
}

void hy_launch_emit(hyrf_scene* s, const uint32_t* order, uint32_t V, uint32_t* launches) {
    if (V == 0) return;
    const uint32_t gx = (uint32_t)((s->lastW + HY_TILE - 1) / HY_TILE);
    const uint64_t threads = (uint64_t)V * 32ull;
    emit_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, s->stream>>>(order, s->offs, s->rect, s->tiles, V, gx,
                                                                          s->ent_key[0], s->ent_val[0]);
    ++*launches;
}

void hy_launch_ranges(hyrf_scene* s, const uint32_t* keys, uint64_t D, uint32_t n_tiles, uint32_t* launches) {
    cudaMemsetAsync(s->ranges, 0, sizeof(uint2) * n_tiles, s->stream);
    if (D == 0) return;
    ranges_kernel<<<(unsigned)((D + 255) / 256), 256, 0, s->stream>>>(keys, (uint32_t)D, s->ranges);
    ++*launches;
}
