// bin_ordered.cu — S4b–c for frames of up to kMaxTiles tiles: the per-tile lists, ordered by (depth bits, id), written
// in ONE ordered counting pass instead of materialising (tile, id) pairs and radix-sorting them.
// PAPER.md:47 ("ordered by depth"), :57 (the sorted set a pixel blends); order defined in DESIGN.md §2 D9.
//
// Input: the visible Gaussians already in (depth bits, id) order (radix.cu, V items). Output: list[D] of visible ranks
// and ranges[tile] = [start, end).
//   bin_offsets_kernel: offs[k] = tile entries of the Gaussians before k in depth order (single-pass scan, look-back)
//   bin_pairs_kernel  : the (tile, rank) pairs of every Gaussian, written at offs[k] — i.e. in depth order
//   The pair sequence 0..D-1 is cut into chunks of Ec pairs, one CTA each (near Gaussians cover hundreds of tiles and
//   far ones a few, so cutting by pairs — not by Gaussians — is what balances the CTAs):
//   bin_count_kernel  : cnt[chunk][tile]  = pairs of chunk c in tile t                 (shared-memory histogram)
//   bin_prefix_kernel : cnt[chunk][tile] <- sum over earlier chunks; totals[tile]      (column prefix)
//   bin_scatter_kernel: start[tile] = exclusive scan of totals; a pair goes to
//                       start[t] + cnt[c][t] + (earlier pairs of the chunk in tile t).
// This is one stable counting-sort pass over all tile ids at once (up to 10240 bins) where the radix route needs
// ceil(log2(tiles) / 8) passes. Inside a chunk warp w owns Ec/8 consecutive pairs and takes them 32 at a time, in
// order, so "earlier" is: earlier warps (per-warp counts, prefixed) + earlier iterations (running per-warp counter) +
// lower lanes of this iteration (match.any on the tile id). No atomic decides an output slot, so the lists are
// deterministic and bit-equal to the oracle's.
#include "scene.h"

namespace {

constexpr int kBinThreads = 256;
constexpr int kBinWarps = kBinThreads / 32;
constexpr uint32_t kMaxTiles = 10240;     // 20 B of shared memory per tile in bin_emit_kernel
constexpr uint32_t kMinChunk = 16384;     // entries per CTA
constexpr uint32_t kMaxChunk = 61440;     // per-chunk per-tile counts are kept in 16 bits
constexpr int kOffItems = 2048;           // Gaussians per CTA of the offsets scan

struct BinArgs {
    const uint32_t* order;   // [V] visible rank of the k-th Gaussian in depth order
    const uint4* rect;       // [V] (x0, x1, y0, y1) by visible rank
    const uint32_t* tiles;   // [V] tiles touched by visible rank
    FrameCounters* counters;
    uint32_t* offs;          // [V] exclusive prefix of tiles touched, in depth order
    unsigned long long* scan_state;   // look-back words of bin_offsets_kernel, tagged with the frame number
    uint32_t frame;
    uint32_t Ec;             // entries per CTA (multiple of 8)
    uint32_t rows_cap;       // rows of M
    uint32_t T, gx;
    uint32_t* M;             // [rows_cap][T]
    uint32_t* totals;        // [T]
    uint32_t* starts;        // [T] exclusive scan of totals
    uint2* ranges;           // [T]
    uint32_t* tile_queue;    // [T] tile ids, longest list first (the rasterizer's launch order)
    uint32_t* pair_tile;     // [cap] tile id of every pair, depth order
    uint32_t* pair_rank;     // [cap] visible rank of every pair
    uint32_t* list;          // [cap]
    uint32_t cap;
    uint32_t shift;          // 0: bins are tiles; HY_MACRO_SHIFT: bins are macro tiles (rectangles are coarsened)
    uint32_t use_dm;         // pair count comes from counters->Dm (the run the rasterizer consumes) or ->D
    uint32_t fine_T, fine_gx; // the tile grid (for the rasterizer's tile queue) when the bins are macro tiles
};

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= (uint32_t)d) v += u;
    }
    return v;
}

// ---- offs[k] = sum of tiles touched by the Gaussians before k (depth order): one pass, decoupled look-back ------
// Look-back word: [63:34] frame number, [33:32] 1 = block aggregate / 2 = inclusive prefix, [31:0] value. Tagging with
// the frame number means the words never have to be cleared between frames.
__device__ __forceinline__ unsigned long long off_word(uint32_t frame, uint32_t kind, uint32_t v) {
    return ((unsigned long long)frame << 34) | ((unsigned long long)kind << 32) | v;
}

__global__ void __launch_bounds__(kBinThreads)
bin_offsets_kernel(const BinArgs A) {
    __shared__ uint32_t s_tile, s_prefix;
    __shared__ uint32_t s_warp[kBinWarps];
    if (threadIdx.x == 0) s_tile = atomicAdd(&A.counters->bin_ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t V = A.counters->V;
    const uint32_t base = tile * kOffItems;
    if (base >= V) return;   // tickets are handed out in order: every earlier tile exists and is running or done
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    constexpr int kPer = kOffItems / kBinThreads;   // 8 rounds; a warp owns 256 consecutive Gaussians
    const uint32_t wbase = base + warp * (kPer * 32);
    uint32_t v[kPer], ex[kPer];
    uint32_t run = 0;
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
        const uint32_t k = wbase + i * 32 + lane;
        v[i] = k < V ? __ldg(A.tiles + __ldg(A.order + k)) : 0u;
    }
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
        const uint32_t incl = warp_incl_scan(v[i], lane);
        ex[i] = run + incl - v[i];
        run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) s_warp[warp] = run;
    __syncthreads();
    uint32_t woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kBinWarps; ++w) {
        if (w < (int)warp) woff += s_warp[w];
        total += s_warp[w];
    }
    volatile unsigned long long* st = A.scan_state;
    if (warp == 0) {
        if (lane == 0) st[tile] = off_word(A.frame, tile == 0 ? 2u : 1u, total);
        uint32_t prefix = 0;
        if (tile > 0) {
            int p = (int)tile - 1;
            while (true) {
                const int idx = p - (int)lane;
                unsigned long long w = off_word(A.frame, 2u, 0u);   // before the first tile: inclusive 0
                if (idx >= 0) {
                    do { w = st[idx]; } while ((uint32_t)(w >> 34) != A.frame);
                }
                const uint32_t kind = (uint32_t)(w >> 32) & 3u, val = (uint32_t)w;
                const uint32_t incl_mask = __ballot_sync(0xffffffffu, kind == 2u);
                const uint32_t upto = incl_mask ? (uint32_t)__ffs(incl_mask) - 1u : 31u;
                uint32_t part = lane <= upto ? val : 0u;
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) part += __shfl_xor_sync(0xffffffffu, part, d);
                prefix += part;
                if (incl_mask) break;
                p -= 32;
            }
            if (lane == 0) st[tile] = off_word(A.frame, 2u, prefix + total);
        }
        if (lane == 0) s_prefix = prefix;
    }
    __syncthreads();
    const uint32_t add = s_prefix + woff;
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
        const uint32_t k = wbase + i * 32 + lane;
        if (k < V) A.offs[k] = add + ex[i];
    }
}


// ---- (tile, rank) pairs in depth order ----------------------------------------------------------------------------
// A warp takes 32 consecutive Gaussians of the depth order. Each lane writes the first pairs of its own Gaussian
// (neighbouring lanes own neighbouring output slots), then the warp sweeps the long rectangles together.
__global__ void __launch_bounds__(kBinThreads)
bin_pairs_kernel(const BinArgs A) {
    constexpr uint32_t kOwn = 4;
    const uint32_t V = A.counters->V;
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31u;
    if (blockIdx.x * blockDim.x >= V) return;
    uint32_t g = 0, nt = 0, base = 0;
    uint4 rc = make_uint4(0, 1, 0, 0);
    if (k < V) {
        g = __ldg(A.order + k);
        nt = __ldg(A.tiles + g);
        rc = __ldg(A.rect + g);
        base = A.offs[k];
        if (A.shift) {   // tile rectangle -> macro-tile rectangle
            const uint32_t r = (1u << A.shift) - 1u;
            rc = make_uint4(rc.x >> A.shift, (rc.y + r) >> A.shift, rc.z >> A.shift, (rc.w + r) >> A.shift);
        }
        if (nt == 0) rc = make_uint4(0, 1, 0, 0);
    }
    const uint32_t w = rc.y - rc.x;
    const uint32_t own = nt < kOwn ? nt : kOwn;
    for (uint32_t i = 0; i < own; ++i) {
        const uint32_t row = i / w;
        if (base + i < A.cap) {
            A.pair_tile[base + i] = (rc.z + row) * A.gx + rc.x + (i - row * w);
            A.pair_rank[base + i] = g;
        }
    }
    uint32_t big = __ballot_sync(0xffffffffu, nt > kOwn);
    while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const uint32_t g2 = __shfl_sync(0xffffffffu, g, src), nt2 = __shfl_sync(0xffffffffu, nt, src);
        const uint32_t b2 = __shfl_sync(0xffffffffu, base, src);
        const uint32_t x0 = __shfl_sync(0xffffffffu, rc.x, src), y0 = __shfl_sync(0xffffffffu, rc.z, src);
        const uint32_t w2 = __shfl_sync(0xffffffffu, w, src);
        const float rw = 1.0f / (float)w2;
        for (uint32_t i = kOwn + lane; i < nt2; i += 32) {
            const uint32_t row = (uint32_t)(((float)i + 0.5f) * rw);   // exact: |error| << 0.5 / w
            if (b2 + i < A.cap) {
                A.pair_tile[b2 + i] = (y0 + row) * A.gx + x0 + (i - row * w2);
                A.pair_rank[b2 + i] = g2;
            }
        }
    }
}

__device__ __forceinline__ uint32_t pair_count(const BinArgs& A) {
    const unsigned long long D = A.use_dm ? A.counters->Dm : A.counters->D;
    return (uint32_t)(D < A.cap ? D : A.cap);
}

__global__ void __launch_bounds__(kBinThreads)
bin_count_kernel(const BinArgs A) {
    extern __shared__ uint32_t s_cnt[];
    const uint32_t D = pair_count(A);
    const uint32_t e0 = blockIdx.x * A.Ec;
    if (e0 >= D) return;
    const uint32_t e1 = e0 + A.Ec < D ? e0 + A.Ec : D;
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) s_cnt[t] = 0;
    __syncthreads();
    for (uint32_t eb = e0; eb < e1; eb += kBinThreads * 8) {
        uint32_t tl[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t e = eb + u * kBinThreads + threadIdx.x;
            tl[u] = e < e1 ? __ldg(A.pair_tile + e) : 0xFFFFFFFFu;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (tl[u] != 0xFFFFFFFFu) atomicAdd(&s_cnt[tl[u]], 1u);
    }
    __syncthreads();
    uint32_t* row = A.M + (size_t)blockIdx.x * A.T;
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) row[t] = s_cnt[t];
}

// cnt[c][t] <- sum_{c' < c} cnt[c'][t]; totals[t] = column sum. A CTA owns 32 tiles (lanes) x 32 row groups (warps).
__global__ void __launch_bounds__(1024)
bin_prefix_kernel(const BinArgs A) {
    __shared__ uint32_t s_part[32][33];
    const uint32_t D = pair_count(A);
    const uint32_t rows = (D + A.Ec - 1) / A.Ec;
    const uint32_t lane = threadIdx.x & 31u, grp = threadIdx.x >> 5;
    const uint32_t t = blockIdx.x * 32 + lane;
    const uint32_t per = (rows + 31) / 32;
    const uint32_t r0 = grp * per < rows ? grp * per : rows, r1 = r0 + per < rows ? r0 + per : rows;
    // rows <= ~1024 -> at most 32 rows per group: kept in registers, all loads in flight at once
    constexpr int kRows = 8;
    uint32_t sum = 0;
    if (t < A.T)
        for (uint32_t rb = r0; rb < r1; rb += kRows) {
            uint32_t v[kRows];
#pragma unroll
            for (int i = 0; i < kRows; ++i) v[i] = rb + i < r1 ? A.M[(size_t)(rb + i) * A.T + t] : 0u;
#pragma unroll
            for (int i = 0; i < kRows; ++i) sum += v[i];
        }
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
        for (uint32_t rb = r0; rb < r1; rb += kRows) {
            uint32_t v[kRows];
#pragma unroll
            for (int i = 0; i < kRows; ++i) v[i] = rb + i < r1 ? A.M[(size_t)(rb + i) * A.T + t] : 0u;
#pragma unroll
            for (int i = 0; i < kRows; ++i) {
                if (rb + i < r1) A.M[(size_t)(rb + i) * A.T + t] = run;
                run += v[i];
            }
        }
        if (grp == 0) A.totals[t] = total;
    }
    // the last CTA to finish turns totals[] into start[] (exclusive scan over the tiles) and writes ranges[]
    __shared__ bool s_last;
    __shared__ uint32_t s_wsum[32];
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&A.counters->bin_done, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const uint32_t per_t = (A.T + 1023u) / 1024u;
    const uint32_t t0 = threadIdx.x * per_t < A.T ? threadIdx.x * per_t : A.T, t1 = t0 + per_t < A.T ? t0 + per_t : A.T;
    uint32_t mine = 0;
    for (uint32_t t2 = t0; t2 < t1; ++t2) mine += __ldcg(A.totals + t2);
    const uint32_t incl = warp_incl_scan(mine, lane);
    if (lane == 31) s_wsum[grp] = incl;
    __syncthreads();
    uint32_t start = incl - mine;
    for (uint32_t w2 = 0; w2 < grp; ++w2) start += s_wsum[w2];
    for (uint32_t t2 = t0; t2 < t1; ++t2) {
        const uint32_t n = __ldcg(A.totals + t2);
        A.ranges[t2] = n ? make_uint2(start, start + n) : make_uint2(0u, 0u);   // empty: [0, 0)
        A.starts[t2] = start;
        start += n;
    }
}

// STAGED (long lists over few bins: the 4K frames of config 5, 43 M pairs over 2 040 macro tiles): the chunk's entries
// are first put in bin order in shared memory and every bin's run is then written out as one piece. Written directly,
// a bin's run of a chunk arrives as eight pieces of ~3 entries at eight different times, one from each warp; with
// 740 resident CTAs x 2 040 bins x 8 warps there are far more partially written sectors than the L2 can hold, and
// the scatter moved 1.04 GB to DRAM for a 173 MB list (and read 1.27 GB): 1.22 of the 3.7 ms of that frame.
constexpr uint32_t kStagedMaxBins = 2560, kStagedChunk = 16384;
constexpr size_t kStagedMinCap = 8u << 20;

template <bool STAGED>
__global__ void __launch_bounds__(kBinThreads)
bin_scatter_kernel(const BinArgs A) {
    extern __shared__ uint32_t s_mem[];
    uint32_t* s_base = s_mem;                                               // [T] first slot of this chunk per tile
    unsigned short* s_wcnt = reinterpret_cast<unsigned short*>(s_mem + A.T); // [warps][Tp] per-warp counts -> running
    const uint32_t Tp = (A.T + 1u) & ~1u;
    uint32_t* l_start = s_mem + A.T + kBinWarps * Tp / 2;                    // STAGED: [T + 1] first slot of a bin in s_list
    uint32_t* s_list = l_start + A.T + 1;                                    // STAGED: [Ec] the chunk's entries in bin order
    const uint32_t D = pair_count(A);
    const uint32_t c0 = blockIdx.x * A.Ec;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (blockIdx.x == gridDim.x - 1) {
        // one extra CTA orders the tiles for the rasterizer: 33 buckets by floor(log2(list length)), longest first;
        // the order inside a bucket is arbitrary and only affects scheduling
        __shared__ uint32_t s_bucket[33];
        if (threadIdx.x < 33) s_bucket[threadIdx.x] = 0;
        __syncthreads();
        const uint32_t nq = A.shift ? A.fine_T : A.T;          // the queue holds TILES; their length is their bin's
        auto len_of = [&](uint32_t t) {
            if (!A.shift) return __ldg(A.totals + t);
            const uint32_t tx = t % A.fine_gx, ty = t / A.fine_gx;
            return __ldg(A.totals + (ty >> A.shift) * A.gx + (tx >> A.shift));
        };
        for (uint32_t t = threadIdx.x; t < nq; t += kBinThreads) atomicAdd(&s_bucket[32 - __clz(len_of(t))], 1u);
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t run = 0;
            for (int b = 32; b >= 0; --b) { const uint32_t c = s_bucket[b]; s_bucket[b] = run; run += c; }
        }
        __syncthreads();
        for (uint32_t t = threadIdx.x; t < nq; t += kBinThreads)
            A.tile_queue[atomicAdd(&s_bucket[32 - __clz(len_of(t))], 1u)] = t;
        return;
    }
    if (c0 >= D) return;
    const uint32_t* row = A.M + (size_t)blockIdx.x * A.T;
    for (uint32_t t = threadIdx.x; t < A.T; t += kBinThreads) s_base[t] = __ldg(A.starts + t) + __ldg(row + t);
    for (uint32_t i = threadIdx.x; i < kBinWarps * Tp / 2; i += kBinThreads) reinterpret_cast<uint32_t*>(s_wcnt)[i] = 0;
    __syncthreads();
    // warp w owns pairs [w0, w1) of the chunk
    const uint32_t Ew = A.Ec / kBinWarps;
    const uint32_t c1 = c0 + A.Ec < D ? c0 + A.Ec : D;
    const uint32_t w0 = c0 + warp * Ew < c1 ? c0 + warp * Ew : c1, w1 = w0 + Ew < c1 ? w0 + Ew : c1;
    // per-warp counts (two 16-bit counters per word; <= Ew <= 7680 pairs per warp: no carry)
    uint32_t* wc32 = reinterpret_cast<uint32_t*>(s_wcnt + (size_t)warp * Tp);
    constexpr int kU = 16;   // pairs per lane fetched together: the loads of 512 pairs are in flight at once
    for (uint32_t eb = w0; eb < w1; eb += 32 * kU) {
        uint32_t tl[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const uint32_t e = eb + u * 32 + lane;
            tl[u] = e < w1 ? __ldg(A.pair_tile + e) : 0xFFFFFFFFu;
        }
#pragma unroll
        for (int u = 0; u < kU; ++u)
            if (tl[u] != 0xFFFFFFFFu) atomicAdd(&wc32[tl[u] >> 1], (tl[u] & 1u) ? 0x10000u : 1u);
    }
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
        if (STAGED) l_start[t] = run;   // the chunk's count of this bin, scanned below
    }
    __syncthreads();
    if (STAGED) {
        // exclusive scan of the bins' counts: a thread owns a contiguous stretch of bins
        __shared__ uint32_t s_part[kBinThreads];
        const uint32_t per = (A.T + kBinThreads - 1) / kBinThreads;
        const uint32_t t0 = threadIdx.x * per, t1 = t0 + per < A.T ? t0 + per : A.T;
        uint32_t sum = 0;
        for (uint32_t t = t0; t < t1; ++t) sum += l_start[t];
        s_part[threadIdx.x] = sum;
        __syncthreads();
        if (warp == 0) {   // 256 partial sums: 8 per lane
            uint32_t v[kBinThreads / 32], tot = 0;
#pragma unroll
            for (int i = 0; i < kBinThreads / 32; ++i) { v[i] = s_part[lane * (kBinThreads / 32) + i]; tot += v[i]; }
            uint32_t incl = tot;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= (uint32_t)d) incl += u;
            }
            uint32_t run = incl - tot;
#pragma unroll
            for (int i = 0; i < kBinThreads / 32; ++i) { s_part[lane * (kBinThreads / 32) + i] = run; run += v[i]; }
        }
        __syncthreads();
        uint32_t run = s_part[threadIdx.x];
        for (uint32_t t = t0; t < t1; ++t) { const uint32_t c = l_start[t]; l_start[t] = run; run += c; }
        if (threadIdx.x == kBinThreads - 1) l_start[A.T] = c1 - c0;
        __syncthreads();
    }
    // ordered scatter, 32 pairs per step
    unsigned short* wc = s_wcnt + (size_t)warp * Tp;
    const uint32_t tbits = 32u - (uint32_t)__clz(A.T > 1u ? A.T - 1u : 1u);   // bits of the largest bin id
    for (uint32_t eb = w0; eb < w1; eb += 32 * kU) {
        uint32_t tl[kU], gl[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const uint32_t e = eb + u * 32 + lane;
            const bool in = e < w1;
            tl[u] = in ? __ldg(A.pair_tile + e) : 0xFFFFFFFFu;
            gl[u] = in ? __ldg(A.pair_rank + e) : 0u;
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            if (eb + u * 32 >= w1) break;                    // warp-uniform
            const uint32_t tile = tl[u];
            const bool act = tile != 0xFFFFFFFFu;
            // lanes with the same bin, one ballot per bit of the bin id (consecutive pairs mostly differ in their bin, the
            // case in which match.any is slowest: radix.cu)
            uint32_t peers = __ballot_sync(0xffffffffu, act);
            for (uint32_t b = 0; b < tbits; ++b) {
                const bool bit = (tile >> b) & 1u;
                const uint32_t bal = __ballot_sync(0xffffffffu, bit);
                peers &= bit ? bal : ~bal;
            }
            uint32_t c = 0;
            if (act) c = wc[tile];
            __syncwarp();
            if (act && lane == (uint32_t)(__ffs(peers) - 1)) wc[tile] = (unsigned short)(c + __popc(peers));
            __syncwarp();
            if (act) {
                const uint32_t k = c + __popc(peers & ((1u << lane) - 1u));   // place in the chunk's run of this bin
                if (STAGED) s_list[l_start[tile] + k] = gl[u];
                else A.list[s_base[tile] + k] = gl[u];   // slot < D <= cap
            }
        }
    }
    if (STAGED) {
        // every bin's run of this chunk in one piece: a warp per bin, lanes along the run
        __syncthreads();
        for (uint32_t t = warp; t < A.T; t += kBinWarps) {
            const uint32_t a = l_start[t], n = l_start[t + 1] - a, dst = s_base[t];
            for (uint32_t k = lane; k < n; k += 32) A.list[dst + k] = s_list[a + k];
        }
    }
}

// pairs per CTA: at most ~1024 chunks; with few bins (macro tiles) the per-CTA set-up is cheap and small chunks give
// the scatter more CTAs to fill the machine with, with thousands of bins it must be amortised over more pairs
// (with a few hundred bins the pieces are long enough as they are, and the small chunks only add rows: config 4 and
// 4M @ 1080p, 330 and 510 macro tiles, were 5 - 10 % slower staged)
bool scatter_staged(size_t cap, uint32_t T) { return T > 1024 && T <= kStagedMaxBins && cap >= kStagedMinCap; }

uint32_t chunk_entries(size_t cap, uint32_t T) {
    if (scatter_staged(cap, T)) return kStagedChunk;   // the chunk is staged in shared memory (bin_scatter_kernel<true>)
    size_t c = (cap + 1023) / 1024;
    c = (c + 2047) / 2048 * 2048;
    const size_t lo = T <= 1024 ? 2048 : kMinChunk;
    if (c < lo) c = lo;
    if (c > kMaxChunk) c = kMaxChunk;
    return (uint32_t)c;
}

}  // namespace

bool hy_bin_ordered_supported(uint32_t /*N*/, uint32_t n_tiles) { return n_tiles <= kMaxTiles; }

// uint32 elements of workspace for a list capacity of `cap` entries: count matrix + totals + look-back words
size_t hy_bin_ordered_ws_elems(uint32_t N, size_t cap, uint32_t max_tiles) {
    const uint32_t T = max_tiles < kMaxTiles ? max_tiles : kMaxTiles;
    // the count matrix of the largest run: rows x bins grows with the bin count inside each chunk-size regime, so the
    // two candidates are the most bins of the small-chunk regime and the most bins overall
    auto cells = [&](uint32_t t) { return ((cap + chunk_entries(cap, t) - 1) / chunk_entries(cap, t) + 1) * (size_t)t; };
    const size_t small = cells(T < 1024 ? T : 1024), m = cells(T) > small ? cells(T) : small;
    return 2 * ((size_t)N / kOffItems + 2) + m + 2 * T + 64;
}

// macro = false: bins are tiles -> s->ranges only (the ranges of the per-tile lists the rasterizer writes for the debug
//                export / the backward pass); no list is scattered.
// macro = true : bins are macro tiles (HY_MACRO x HY_MACRO tiles) -> s->mranges, list in ent_key[1], s->tile_queue:
//                what the rasterizer walks; n_tiles / gx are still those of the TILE grid.
hyrf_status hy_launch_bin_ordered(hyrf_scene* s, const uint32_t* order, uint32_t n_tiles, uint32_t gx,
                                  uint32_t* launches, bool macro, uint32_t shift) {
    BinArgs A;
    A.shift = macro ? shift : 0;
    A.use_dm = macro;
    A.fine_T = n_tiles; A.fine_gx = gx;
    if (macro) {
        const uint32_t gy = n_tiles / gx;
        const uint32_t mgx = (gx + (1u << shift) - 1) >> shift, mgy = (gy + (1u << shift) - 1) >> shift;
        gx = mgx;
        n_tiles = mgx * mgy;
    }
    A.order = order; A.rect = s->rect; A.tiles = macro ? s->mtiles : s->tiles; A.counters = s->counters;
    A.offs = s->offs;
    A.cap = (uint32_t)(s->d_capacity > 0xFFFFFFF0ull ? 0xFFFFFFF0ull : s->d_capacity);
    A.Ec = chunk_entries(s->d_capacity, n_tiles);
    A.rows_cap = (uint32_t)((s->d_capacity + A.Ec - 1) / A.Ec + 1);
    A.T = n_tiles; A.gx = gx;
    const uint32_t T_max = (uint32_t)(((s->desc.max_width + HY_TILE - 1) / HY_TILE) * ((s->desc.max_height + HY_TILE - 1) / HY_TILE));
    const uint32_t T_ws = T_max < kMaxTiles ? T_max : kMaxTiles;
    // workspace: look-back words first (their place must not depend on the run: they are only valid by frame tag),
    // then the count matrix of this run, its totals and starts
    A.scan_state = reinterpret_cast<unsigned long long*>(s->bin_ws);
    A.M = s->bin_ws + 2 * ((size_t)s->N / kOffItems + 2);
    A.totals = A.M + (size_t)A.rows_cap * n_tiles;
    A.starts = A.totals + n_tiles;
    (void)T_ws;
    A.frame = ++s->bin_frame & 0x3FFFFFFFu;
    if (A.frame == 0) A.frame = ++s->bin_frame & 0x3FFFFFFFu;   // 0 is the tag of freshly cleared words
    A.ranges = macro ? s->mranges : s->ranges;
    A.tile_queue = s->tile_queue;
    A.pair_tile = s->ent_key[0];
    A.pair_rank = s->ent_val[0];
    A.list = macro ? s->ent_key[1] : s->ent_val[1];
    const size_t smem_count = (size_t)n_tiles * 4;
    const size_t smem_scatter = (size_t)n_tiles * 4 + (size_t)kBinWarps * ((n_tiles + 1u) & ~1u) * 2;
    bool& attr_set = s->bin_attr_set;
    if (!attr_set) {
        HY_CUDA_OK(cudaFuncSetAttribute(bin_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kMaxTiles * 4)));
        HY_CUDA_OK(cudaFuncSetAttribute(bin_scatter_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kMaxTiles * 20)));
        HY_CUDA_OK(cudaFuncSetAttribute(bin_scatter_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kStagedMaxBins * 20 + 8 + kStagedChunk * 4)));
        attr_set = true;
    }
    const uint32_t off_blocks = (s->N + kOffItems - 1) / kOffItems;
    bin_offsets_kernel<<<off_blocks, kBinThreads, 0, s->stream>>>(A);
    bin_pairs_kernel<<<(s->N + kBinThreads - 1) / kBinThreads, kBinThreads, 0, s->stream>>>(A);
    bin_count_kernel<<<A.rows_cap, kBinThreads, smem_count, s->stream>>>(A);
    bin_prefix_kernel<<<(n_tiles + 31) / 32, 1024, 0, s->stream>>>(A);
    // the tile-level run only supplies the per-tile ranges (the lists themselves are written by the rasterizer as it
    // consumes them, api.cu): its scatter would produce a list nobody reads
    if (macro) {
        if (scatter_staged(s->d_capacity, n_tiles)) {
            const size_t smem_staged = smem_scatter + ((size_t)n_tiles + 1 + A.Ec) * 4;
            bin_scatter_kernel<true><<<A.rows_cap + 1, kBinThreads, smem_staged, s->stream>>>(A);   // + 1: the tile-queue CTA
        } else {
            bin_scatter_kernel<false><<<A.rows_cap + 1, kBinThreads, smem_scatter, s->stream>>>(A);
        }
    }
    *launches += macro ? 5 : 4;
    return HYRF_OK;
}
