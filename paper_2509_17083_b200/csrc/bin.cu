// bin.cu — S4b: tile binning. PAPER.md:47 ("ordered by depth ... projected onto 2D image planes"), :57 (the set of
// sorted Gaussians projected onto the pixel); order defined in DESIGN.md §2 D9: (tile, depth bits, id) ascending.
// Radix route, used only for tile grids beyond bin_ordered.cu's limit: Gaussians are first ordered by (depth bits, id)
// — V items — and emit their tile entries in that order; one stable sort of the D entries by tile id (only
// ceil(log2 tiles) key bits) then yields the final lists. That moves 8 B per entry per pass over 2 passes instead of
// 12 B over 6 passes of a 64-bit (tile|depth) key.
#include "scene.h"

namespace {

// tt_sorted[k] = tiles touched by the k-th Gaussian in depth order
__global__ void __launch_bounds__(256)
tiles_gather_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ tiles, uint32_t V,
                    uint32_t* __restrict__ tt_sorted) {
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < V) tt_sorted[k] = tiles[order[k]];
}

// A warp takes 32 consecutive Gaussians of the depth order. Each lane writes the first entries of its own Gaussian
// (neighbouring lanes own neighbouring output slots), then the warp sweeps the long rectangles together.
__global__ void __launch_bounds__(256)
emit_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ offs, const uint4* __restrict__ rect,
            const uint32_t* __restrict__ tiles, uint32_t V, uint32_t gx, uint32_t* __restrict__ ent_key,
            uint32_t* __restrict__ ent_val) {
    constexpr uint32_t kOwn = 4;
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    uint32_t g = 0, nt = 0, base = 0;
    uint4 rc = make_uint4(0, 1, 0, 0);
    if (k < V) {
        g = order[k];
        nt = tiles[g];
        rc = rect[g];
        base = offs[k];
    }
    uint32_t w = rc.y - rc.x;
    const uint32_t own = nt < kOwn ? nt : kOwn;
    for (uint32_t i = 0; i < own; ++i) {
        ent_key[base + i] = (rc.z + i / w) * gx + rc.x + i % w;
        ent_val[base + i] = g;
    }
    uint32_t big = __ballot_sync(0xffffffffu, nt > kOwn);
    while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const uint32_t g2 = __shfl_sync(0xffffffffu, g, src), nt2 = __shfl_sync(0xffffffffu, nt, src);
        const uint32_t b2 = __shfl_sync(0xffffffffu, base, src);
        const uint32_t x0 = __shfl_sync(0xffffffffu, rc.x, src), y0 = __shfl_sync(0xffffffffu, rc.z, src);
        const uint32_t w2 = __shfl_sync(0xffffffffu, w, src);
        for (uint32_t i = kOwn + lane; i < nt2; i += 32) {
            ent_key[b2 + i] = (y0 + i / w2) * gx + x0 + i % w2;
            ent_val[b2 + i] = g2;
        }
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

void hy_launch_tiles_gather(hyrf_scene* s, const uint32_t* order, uint32_t V, uint32_t* launches) {
    if (V == 0) return;
    tiles_gather_kernel<<<(V + 255) / 256, 256, 0, s->stream>>>(order, s->tiles, V, s->tt_sorted);
    ++*launches;
}

void hy_launch_emit(hyrf_scene* s, const uint32_t* order, uint32_t V, uint32_t* launches) {
    if (V == 0) return;
    const uint32_t gx = (uint32_t)((s->lastW + HY_TILE - 1) / HY_TILE);
    emit_kernel<<<(V + 255) / 256, 256, 0, s->stream>>>(order, s->offs, s->rect, s->tiles, V, gx,
                                                                          s->ent_key[0], s->ent_val[0]);
    ++*launches;
}

void hy_launch_ranges(hyrf_scene* s, const uint32_t* keys, uint64_t D, uint32_t n_tiles, uint32_t* launches) {
    cudaMemsetAsync(s->ranges, 0, sizeof(uint2) * n_tiles, s->stream);
    if (D == 0) return;
    ranges_kernel<<<(unsigned)((D + 255) / 256), 256, 0, s->stream>>>(keys, (uint32_t)D, s->ranges);
    ++*launches;
}
