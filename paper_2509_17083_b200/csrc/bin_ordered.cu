// bin_ordered.cu — S4b–c for frames of up to kMaxTiles tiles: the per-tile lists, ordered by (depth bits, id), written
// in ONE ordered counting pass instead of materialising (tile, id) pairs and radix-sorting them.
// PAPER.md:47 ("ordered by depth"), :57 (the sorted set a pixel blends); order defined in DESIGN.md §2 D9.
//
// Input: the visible Gaussians already in (depth bits, id) order (radix.cu, V items). Output: list[D] of visible ranks
// and ranges[tile] = [start, end). The depth order is cut into chunks of `chunk` consecutive Gaussians, one CTA each:
//   bin_count_kernel : cnt[chunk][tile]  = entries chunk c sends to tile t            (shared-memory histogram)
//   bin_prefix_kernel: cnt[chunk][tile] <- sum over earlier chunks; totals[tile]      (column prefix)
//   bin_emit_kernel  : start[tile] = exclusive scan of totals; every entry goes to
//                      start[t] + cnt[c][t] + (entries of earlier Gaussians of the chunk in tile t).
// Inside a chunk, warp w owns chunk/8 consecutive Gaussians; it walks their tile rectangles flattened 32 entries
// at a time, in order, so "earlier" is: earlier warps (per-warp counts, prefixed) + earlier iterations (running
// per-warp counter) + lower lanes of this iteration (match.any on the tile id). No atomics decide an output slot,
// so the lists are deterministic and bit-equal to the oracle's. Traffic: 3 reads of the 16-B rectangle per visible
// Gaussian + 4 B written per entry + the count matrix (rows x tiles x 4 B, L2-resident) three times, against
// 8 B written + 2 x 16 B sorted + 8 B histogram + 4 B range scan per entry on the radix route (bin.cu).
#include "scene.h"

namespace {

constexpr int kBinThreads = 256;
constexpr int kBinWarps = kBinThreads / 32;
constexpr uint32_t kMaxTiles = 10240;   // 20 B of shared memory per tile in bin_emit_kernel
constexpr uint32_t kMaxRows = 1024;

struct BinArgs {
    const uint32_t* order;   // [V] visible rank of the k-th Gaussian in depth order
    const uint4* rect;       // [V] (x0, x1, y0, y1) by visible rank
    const uint32_t* tiles;   // [V] tiles touched by visible rank
    const FrameCounters* counters;
    uint32_t chunk;          // Gaussians per CTA (multiple of 256)
    uint32_t T, gx;
    uint32_t* M;             // [rows][T]
    uint32_t* totals;        // [T]
    uint2* ranges;           // [T]
    uint32_t* list;          // [cap]
    uint32_t cap;
};

// Warp-collective: visits the tile entries of Gaussians k0..k1-1 of the depth order, 32 entries per call of f,
// ordered by (k, tile index inside the rectangle: y outer, x inner). f(tile, g, active).
template <class F>
__device__ __forceinline__ void walk_entries(const BinArgs& A, uint32_t k0, uint32_t k1, F&& f) {
    const uint32_t lane = threadIdx.x & 31u;
    for (uint32_t kb = k0; kb < k1; kb += 32) {
        const uint32_t k = kb + lane;
        uint32_t g = 0, nt = 0, x0 = 0, y0 = 0, w = 1;
        if (k < k1) {
            g = __ldg(A.order + k);
            nt = __ldg(A.tiles + g);
            if (nt) {
                const uint4 rc = __ldg(A.rect + g);
                x0 = rc.x; y0 = rc.z; w = rc.y - rc.x;
            }
        }
        uint32_t incl = nt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= (uint32_t)d) incl += u;
        }
        const uint32_t E = __shfl_sync(0xffffffffu, incl, 31);
        const uint32_t excl = incl - nt;
        for (uint32_t e0 = 0; e0 < E; e0 += 32) {
            const uint32_t e = e0 + lane;
            const bool act = e < E;
            uint32_t q = 0;   // number of Gaussians of the batch whose entries all precede e
#pragma unroll
            for (int s = 16; s >= 1; s >>= 1) {
                const uint32_t v = __shfl_sync(0xffffffffu, incl, (int)(q + s - 1));
                if (v <= e) q += s;
            }
            q = q > 31u ? 31u : q;
            const uint32_t i = e - __shfl_sync(0xffffffffu, excl, (int)q);
            const uint32_t xq = __shfl_sync(0xffffffffu, x0, (int)q), yq = __shfl_sync(0xffffffffu, y0, (int)q);
            const uint32_t wq = __shfl_sync(0xffffffffu, w, (int)q), gq = __shfl_sync(0xffffffffu, g, (int)q);
            const uint32_t ii = act ? i : 0u;
            const uint32_t row = (uint32_t)__fdividef((float)ii + 0.5f, (float)wq);   // exact: |error| << 0.5 / w
            const uint32_t tile = (yq + row) * A.gx + xq + (ii - row * wq);
            f(tile, gq, act);
        }
    }
}

__device__ __forceinline__ void chunk_bounds(const BinArgs& A, uint32_t& k0, uint32_t& k1, uint32_t& V) {
    V = A.counters->V;
    k0 = blockIdx.x * A.chunk;
    k1 = k0 + A.chunk < V ? k0 + A.chunk : V;
}

__global__ void __launch_bounds__(kBinThreads)
bin_count_kernel(const BinArgs A) {
    extern __shared__ uint32_t s_cnt[];
    uint32_t k0, k1, V;
    chunk_bounds(A, k0, k1, V);
    if (k0 >= V) return;
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) s_cnt[t] = 0;
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5, seg = A.chunk / kBinWarps;
    const uint32_t w0 = k0 + warp * seg, w1 = w0 + seg < k1 ? w0 + seg : k1;
    if (w0 < k1)
        walk_entries(A, w0, w1, [&](uint32_t tile, uint32_t, bool act) {
            if (act) atomicAdd(&s_cnt[tile], 1u);
        });
    __syncthreads();
    uint32_t* row = A.M + (size_t)blockIdx.x * A.T;
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) row[t] = s_cnt[t];
}

// cnt[c][t] <- sum_{c' < c} cnt[c'][t]; totals[t] = column sum. A CTA owns 32 tiles (lanes) x 32 row groups (warps).
__global__ void __launch_bounds__(1024)
bin_prefix_kernel(const BinArgs A) {
    __shared__ uint32_t s_part[32][33];
    const uint32_t V = A.counters->V;
    const uint32_t rows = (V + A.chunk - 1) / A.chunk;
    const uint32_t lane = threadIdx.x & 31u, grp = threadIdx.x >> 5;
    const uint32_t t = blockIdx.x * 32 + lane;
    const uint32_t per = (rows + 31) / 32;
    const uint32_t r0 = grp * per, r1 = r0 + per < rows ? r0 + per : rows;
    uint32_t sum = 0;
    if (t < A.T)
        for (uint32_t r = r0; r < r1; ++r) sum += A.M[(size_t)r * A.T + t];
    s_part[grp][lane] = sum;
    __syncthreads();
    uint32_t run = 0, total = 0;
#pragma unroll 8
    for (uint32_t g2 = 0; g2 < 32; ++g2) {
        const uint32_t v = s_part[g2][lane];
        if (g2 < grp) run += v;
        total += v;
    }
    if (t < A.T) {
        for (uint32_t r = r0; r < r1; ++r) {
            uint32_t* p = A.M + (size_t)r * A.T + t;
            const uint32_t v = *p;
            *p = run;
            run += v;
        }
        if (grp == 0) A.totals[t] = total;
    }
}

__global__ void __launch_bounds__(kBinThreads)
bin_emit_kernel(const BinArgs A) {
    extern __shared__ uint32_t s_mem[];
    __shared__ uint32_t s_warp[kBinWarps];
    uint32_t* s_base = s_mem;                                               // [T] first slot of this chunk per tile
    unsigned short* s_wcnt = reinterpret_cast<unsigned short*>(s_mem + A.T); // [warps][Tp] per-warp counts -> running
    const uint32_t Tp = (A.T + 1u) & ~1u;
    uint32_t k0, k1, V;
    chunk_bounds(A, k0, k1, V);
    if (k0 >= V && blockIdx.x != 0) return;   // CTA 0 always runs: it owns ranges[] (all empty when V = 0)
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    // start[t] = exclusive scan of totals over the tiles (every CTA recomputes it: T <= 10240 values from L2)
    const uint32_t per = (A.T + kBinThreads - 1) / kBinThreads;
    const uint32_t t0 = threadIdx.x * per, t1 = t0 + per < A.T ? t0 + per : A.T;
    uint32_t mine = 0;
    for (uint32_t t = t0; t < t1; ++t) mine += A.totals[t];
    uint32_t incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= (uint32_t)d) incl += u;
    }
    if (lane == 31) s_warp[warp] = incl;
    for (uint32_t i = threadIdx.x; i < kBinWarps * Tp / 2; i += kBinThreads) reinterpret_cast<uint32_t*>(s_wcnt)[i] = 0;
    __syncthreads();
    uint32_t start = incl - mine;
    for (uint32_t w2 = 0; w2 < warp; ++w2) start += s_warp[w2];
    const uint32_t* row = A.M + (size_t)blockIdx.x * A.T;
    for (uint32_t t = t0; t < t1; ++t) {
        const uint32_t n = A.totals[t];
        if (blockIdx.x == 0) A.ranges[t] = n ? make_uint2(start, start + n) : make_uint2(0u, 0u);   // empty: [0, 0)
        s_base[t] = start + row[t];
        start += n;
    }
    // per-warp counts
    const uint32_t seg = A.chunk / kBinWarps;
    const uint32_t w0 = k0 + warp * seg, w1 = w0 + seg < k1 ? w0 + seg : k1;
    uint32_t* wc32 = reinterpret_cast<uint32_t*>(s_wcnt + (size_t)warp * Tp);
    if (w0 < k1)
        walk_entries(A, w0, w1, [&](uint32_t tile, uint32_t, bool act) {
            if (act) atomicAdd(&wc32[tile >> 1], (tile & 1u) ? 0x10000u : 1u);   // seg <= 8191: no carry
        });
    __syncthreads();
    // per tile: counts -> exclusive prefix over the warps
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) {
        uint32_t run = 0;
#pragma unroll
        for (int w2 = 0; w2 < kBinWarps; ++w2) {
            const uint32_t c = s_wcnt[(size_t)w2 * Tp + t];
            s_wcnt[(size_t)w2 * Tp + t] = (unsigned short)run;
            run += c;
        }
    }
    __syncthreads();
    // ordered emission
    unsigned short* wc = s_wcnt + (size_t)warp * Tp;
    if (w0 < k1)
        walk_entries(A, w0, w1, [&](uint32_t tile, uint32_t g, bool act) {
            const uint32_t peers = __match_any_sync(0xffffffffu, act ? tile : (0x80000000u | lane));
            uint32_t c = 0;
            if (act) c = wc[tile];
            __syncwarp();
            if (act && lane == (uint32_t)(__ffs(peers) - 1)) wc[tile] = (unsigned short)(c + __popc(peers));
            __syncwarp();
            if (act) {
                const uint32_t slot = s_base[tile] + c + __popc(peers & ((1u << lane) - 1u));
                if (slot < A.cap) A.list[slot] = g;
            }
        });
}

uint32_t chunk_for(uint32_t N) {
    uint32_t c = (N + kMaxRows - 1) / kMaxRows;
    c = (c + 255u) / 256u * 256u;
    return c < 1024u ? 1024u : c;
}

}  // namespace

bool hy_bin_ordered_supported(uint32_t N, uint32_t n_tiles) {
    return n_tiles <= kMaxTiles && chunk_for(N) / kBinWarps <= 8191u;
}

// uint32 elements of workspace: count matrix + totals
size_t hy_bin_ordered_ws_elems(uint32_t N, uint32_t max_tiles) {
    if (!hy_bin_ordered_supported(N, 1)) return 0;
    const uint32_t T = max_tiles < kMaxTiles ? max_tiles : kMaxTiles;
    const size_t rows = (N + chunk_for(N) - 1) / chunk_for(N);
    return rows * T + T + 64;
}

hyrf_status hy_launch_bin_ordered(hyrf_scene* s, const uint32_t* order, uint32_t n_tiles, uint32_t gx,
                                  uint32_t* launches) {
    BinArgs A;
    A.order = order; A.rect = s->rect; A.tiles = s->tiles; A.counters = s->counters;
    A.chunk = chunk_for(s->N);
    A.T = n_tiles; A.gx = gx;
    const uint32_t rows = (s->N + A.chunk - 1) / A.chunk;
    A.M = s->bin_ws;
    A.totals = s->bin_ws + (size_t)rows * n_tiles;
    A.ranges = s->ranges;
    A.list = s->ent_val[0];
    A.cap = (uint32_t)(s->d_capacity > 0xFFFFFFFFull ? 0xFFFFFFFFull : s->d_capacity);
    const size_t smem_count = (size_t)n_tiles * 4;
    const size_t smem_emit = (size_t)n_tiles * 4 + (size_t)kBinWarps * ((n_tiles + 1u) & ~1u) * 2;
    static size_t attr_count = 0, attr_emit = 0;
    if (smem_count > attr_count) {
        HY_CUDA_OK(cudaFuncSetAttribute(bin_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kMaxTiles * 4)));
        attr_count = kMaxTiles * 4;
    }
    if (smem_emit > attr_emit) {
        HY_CUDA_OK(cudaFuncSetAttribute(bin_emit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kMaxTiles * 20)));
        attr_emit = kMaxTiles * 20;
    }
    bin_count_kernel<<<rows, kBinThreads, smem_count, s->stream>>>(A);
    bin_prefix_kernel<<<(n_tiles + 31) / 32, 1024, 0, s->stream>>>(A);
    bin_emit_kernel<<<rows, kBinThreads, smem_emit, s->stream>>>(A);
    *launches += 3;
    return HYRF_OK;
}
