// radix.cu — stable LSD radix sort of (uint32 key, uint32 value) pairs, 8 bits per pass, only the key bits in use.
// S4c of the pass (PAPER.md:47 "ordered by depth", :57): the order (tile, depth bits, id) of DESIGN.md §2 D9 is
// produced by two stable sorts — Gaussians by depth bits (ties keep id order because the compaction is stable),
// then tile entries by tile id. Stability comes from warp match + per-warp digit counters, not atomics on output.
#include "scene.h"

namespace {

constexpr int kRadixThreads = 256;
constexpr int kRadixPer = 16;
constexpr int kRadixItems = kRadixThreads * kRadixPer;  // 4096 keys per block
constexpr int kWarps = kRadixThreads / 32;
constexpr int kWarpItems = kRadixItems / kWarps;        // 512 consecutive keys per warp

__global__ void __launch_bounds__(kRadixThreads)
radix_hist_kernel(const uint32_t* __restrict__ keys, size_t n_cap, const uint32_t* __restrict__ n_dev, int shift,
                  uint32_t mask, uint32_t* __restrict__ hist, uint32_t nb) {
    __shared__ uint32_t h[256];
    const size_t n = n_dev ? (size_t)*n_dev : n_cap;
    h[threadIdx.x] = 0;
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * kRadixItems;
    if (base < n) {
#pragma unroll
        for (int k = 0; k < kRadixPer; ++k) {
            const size_t i = base + (size_t)k * kRadixThreads + threadIdx.x;
            if (i < n) atomicAdd(&h[(keys[i] >> shift) & mask], 1u);
        }
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nb + blockIdx.x] = h[threadIdx.x];
}

__global__ void __launch_bounds__(kRadixThreads)
radix_scatter_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                     uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, size_t n_cap,
                     const uint32_t* __restrict__ n_dev, int shift, uint32_t mask,
                     const uint32_t* __restrict__ hist_scanned, uint32_t nb) {
    __shared__ uint32_t cnt[kWarps][256];
    const size_t n = n_dev ? (size_t)*n_dev : n_cap;
    const size_t base = (size_t)blockIdx.x * kRadixItems;
    if (base >= n) return;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int d = threadIdx.x; d < kWarps * 256; d += kRadixThreads) (&cnt[0][0])[d] = 0;
    __syncthreads();

    uint32_t key[kRadixPer], val[kRadixPer], packed[kRadixPer];
    const size_t wbase = base + (size_t)warp * kWarpItems;
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const size_t i = wbase + (size_t)k * 32 + lane;
        const bool valid = i < n;
        key[k] = valid ? keys_in[i] : 0u;
        val[k] = valid ? vals_in[i] : 0u;
        const uint32_t d = (key[k] >> shift) & mask;
        const uint32_t peers = __match_any_sync(0xffffffffu, valid ? d : (0x80000000u | lane));
        uint32_t c = 0;
        if (valid) c = cnt[warp][d];
        __syncwarp();
        if (valid && lane == (uint32_t)(__ffs(peers) - 1)) cnt[warp][d] = c + __popc(peers);
        __syncwarp();
        packed[k] = valid ? ((d << 16) | (c + __popc(peers & ((1u << lane) - 1u)))) : 0xffffffffu;
    }
    __syncthreads();
    {   // digit d: global offset of this block, then exclusive scan over the warps
        const uint32_t d = threadIdx.x;
        uint32_t run = hist_scanned[(size_t)d * nb + blockIdx.x];
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t t = cnt[w][d];
            cnt[w][d] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        if (packed[k] != 0xffffffffu) {
            const uint32_t pos = cnt[warp][packed[k] >> 16] + (packed[k] & 0xffffu);
            keys_out[pos] = key[k];
            vals_out[pos] = val[k];
        }
    }
}

}  // namespace

size_t hy_radix_hist_elems(size_t n_cap) {
    const size_t nb = (n_cap + kRadixItems - 1) / kRadixItems;
    return 2 * 256 * (nb ? nb : 1);
}

void hy_launch_radix(uint32_t* key_a, uint32_t* val_a, uint32_t* key_b, uint32_t* val_b, size_t n_cap,
                     const uint32_t* n_dev, int key_bits, uint32_t* hist, uint32_t* scan_scratch, cudaStream_t st,
                     uint32_t** out_key, uint32_t** out_val, uint32_t* launches) {
    uint32_t *ki = key_a, *vi = val_a, *ko = key_b, *vo = val_b;
    const size_t nb = (n_cap + kRadixItems - 1) / kRadixItems;
    if (n_cap > 0) {
        uint32_t* hist_scanned = hist + 256 * nb;
        for (int shift = 0; shift < key_bits; shift += 8) {
            const int bits = key_bits - shift < 8 ? key_bits - shift : 8;
            const uint32_t mask = (1u << bits) - 1u;
            radix_hist_kernel<<<(unsigned)nb, kRadixThreads, 0, st>>>(ki, n_cap, n_dev, shift, mask, hist,
                                                                      (uint32_t)nb);
            ++*launches;
            hy_launch_scan(hist, hist_scanned, 256 * nb, scan_scratch, st, launches);
            radix_scatter_kernel<<<(unsigned)nb, kRadixThreads, 0, st>>>(ki, vi, ko, vo, n_cap, n_dev, shift, mask,
                                                                         hist_scanned, (uint32_t)nb);
            ++*launches;
            uint32_t* t = ki; ki = ko; ko = t;
            t = vi; vi = vo; vo = t;
        }
    }
    *out_key = ki;
    *out_val = vi;
}
