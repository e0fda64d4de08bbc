// radix.cu — stable LSD radix sort of (uint32 key, uint32 value) pairs, 8 bits per pass, only the key bits in use.
// S4c of the pass (PAPER.md:47 "ordered by depth", :57): the order (tile, depth bits, id) of DESIGN.md §2 D9 is
// produced by two stable sorts — Gaussians by depth bits (ties keep id order because the compaction is stable),
// then tile entries by tile id.
// One kernel per digit ("onesweep"): a block takes a ticket, ranks its 4096 keys (warp ballots + per-warp digit
// counters: stable, no atomics on the output), publishes its digit counts, resolves its global offsets by
// decoupled look-back over earlier tickets, re-orders the tile in shared memory and writes digit runs coalesced.
// The digit histograms of all passes come from one upfront kernel. HBM traffic per pass = read 8 B + write 8 B per
// pair, the minimum for an out-of-place pass.
#include "scene.h"

namespace {

constexpr int kRadixThreads = 256;
constexpr int kRadixPer = 16;
constexpr int kRadixItems = kRadixThreads * kRadixPer;  // 4096 pairs per block
constexpr int kWarps = kRadixThreads / 32;
constexpr int kWarpItems = kRadixItems / kWarps;        // 512 consecutive pairs per warp
constexpr int kMaxPasses = 4;
constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kValMask = (1u << 30) - 1u;
constexpr size_t kStateBudgetElems = (8u << 20) / 4;    // keep one state slice per pass while they fit in 8 MB

// workspace (uint32 elements): [0, 1024) global digit histograms [pass][256]; [1024, 1028) tickets; [1040, ...) states
constexpr size_t kWsHist = 0, kWsTicket = kMaxPasses * 256, kWsState = kWsTicket + 16;

// exclusive scan of one value per thread over the 256 threads of the block
__device__ __forceinline__ uint32_t block_scan256(uint32_t v, uint32_t* warp_sums /*[8]*/) {
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= (uint32_t)d) incl += u;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    uint32_t off = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) off += (w < (int)warp) ? warp_sums[w] : 0u;
    __syncthreads();
    return off + incl - v;
}

// digit histograms of every pass in one read of the keys
__global__ void __launch_bounds__(kRadixThreads)
radix_global_hist_kernel(const uint32_t* __restrict__ keys, size_t n_cap, const uint32_t* __restrict__ n_dev,
                         int passes, int key_bits, uint32_t* __restrict__ ghist) {
    __shared__ uint32_t h[kMaxPasses][256];
    const size_t n = n_dev ? (size_t)*n_dev : n_cap;
    for (int p = 0; p < passes; ++p) h[p][threadIdx.x] = 0;
    __syncthreads();
    for (size_t base = (size_t)blockIdx.x * kRadixItems; base < n; base += (size_t)gridDim.x * kRadixItems) {
#pragma unroll 4
        for (int k = 0; k < kRadixPer; ++k) {
            const size_t i = base + (size_t)k * kRadixThreads + threadIdx.x;
            if (i < n) {
                const uint32_t key = keys[i];
                for (int p = 0; p < passes; ++p) {
                    const int bits = key_bits - 8 * p < 8 ? key_bits - 8 * p : 8;
                    atomicAdd(&h[p][(key >> (8 * p)) & ((1u << bits) - 1u)], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int p = 0; p < passes; ++p) {
        const uint32_t c = h[p][threadIdx.x];
        if (c) atomicAdd(&ghist[p * 256 + threadIdx.x], c);
    }
}

__global__ void __launch_bounds__(kRadixThreads)
radix_onesweep_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                      uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, size_t n_cap,
                      const uint32_t* __restrict__ n_dev, int shift, uint32_t mask, const uint32_t* __restrict__ ghist,
                      uint32_t* __restrict__ ticket, volatile uint32_t* __restrict__ state) {
    __shared__ uint32_t cnt[kWarps][256];
    __shared__ uint32_t s_key[kRadixItems];
    __shared__ uint32_t s_val[kRadixItems];
    __shared__ uint32_t s_delta[256];
    __shared__ uint32_t s_warp[kWarps];
    __shared__ uint32_t s_tile;
    const size_t n = n_dev ? (size_t)*n_dev : n_cap;
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    for (int d = threadIdx.x; d < kWarps * 256; d += kRadixThreads) (&cnt[0][0])[d] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const size_t base = (size_t)tile * kRadixItems;
    if (base >= n) return;   // tickets are handed out in order: every earlier tile exists and is running or done
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    uint32_t key[kRadixPer], val[kRadixPer], packed[kRadixPer];
    const size_t wbase = base + (size_t)warp * kWarpItems;
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const size_t i = wbase + (size_t)k * 32 + lane;
        const bool valid = i < n;
        key[k] = valid ? keys_in[i] : 0u;
        val[k] = valid ? (vals_in ? vals_in[i] : (uint32_t)i) : 0u;   // no values yet: the value is the index
    }
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const bool valid = wbase + (size_t)k * 32 + lane < n;
        const uint32_t d = (key[k] >> shift) & mask;
        // lanes holding the same digit, from one ballot per digit bit: 9 VOTE + 16 logic instructions. match.any costs
        // several times that when most lanes of a warp hold distinct digits, which is the rule for the low bytes of
        // depth keys; beside the field kernel, on the few SMs it leaves, a pass went from 101 to 74 us (config 3)
        uint32_t peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
        for (int b = 0; b < 8; ++b) {
            const bool bit = (d >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            peers &= bit ? bal : ~bal;
        }
        uint32_t c = 0;
        if (valid) c = cnt[warp][d];
        __syncwarp();
        if (valid && lane == (uint32_t)(__ffs(peers) - 1)) cnt[warp][d] = c + __popc(peers);
        __syncwarp();
        packed[k] = valid ? ((d << 16) | (c + __popc(peers & ((1u << lane) - 1u)))) : 0xffffffffu;
    }
    __syncthreads();
    // thread d owns digit d: exclusive scan over the warps, block total, publish, look back
    const uint32_t d = threadIdx.x;
    uint32_t total = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
        const uint32_t t = cnt[w][d];
        cnt[w][d] = total;
        total += t;
    }
    state[(size_t)tile * 256 + d] = total | (tile == 0 ? kFlagIncl : kFlagAgg);
    const uint32_t gexcl = block_scan256(ghist[d], s_warp);      // first output slot of digit d over the whole array
    const uint32_t dstart = block_scan256(total, s_warp);        // first slot of digit d inside this tile
    uint32_t prefix = 0;
    if (tile > 0) {
        // look back 16 predecessors per round trip: the loads of a round are independent, so the latency of the
        // walk is paid once per 16 tiles instead of once per tile
        constexpr int kLook = 16;
        long long p = (long long)tile - 1;
        bool found = false;
        while (!found) {
            uint32_t v[kLook];
#pragma unroll
            for (int i = 0; i < kLook; ++i) v[i] = (p - i >= 0) ? state[(size_t)(p - i) * 256 + d] : (2u << 30);
#pragma unroll
            for (int i = 0; i < kLook; ++i) {
                if (found) continue;
                while ((v[i] >> 30) == 0u) v[i] = state[(size_t)(p - i) * 256 + d];
                prefix += v[i] & kValMask;
                found = (v[i] >> 30) == 2u;
            }
            p -= kLook;
        }
        state[(size_t)tile * 256 + d] = ((prefix + total) & kValMask) | kFlagIncl;
    }
    s_delta[d] = gexcl + prefix - dstart;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) cnt[w][d] += dstart;
    __syncthreads();
    // re-order the tile in shared memory, then write digit runs
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        if (packed[k] != 0xffffffffu) {
            const uint32_t lp = cnt[warp][packed[k] >> 16] + (packed[k] & 0xffffu);
            s_key[lp] = key[k];
            s_val[lp] = val[k];
        }
    }
    __syncthreads();
    const uint32_t count = (uint32_t)((n - base) < (size_t)kRadixItems ? (n - base) : (size_t)kRadixItems);
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const uint32_t i = k * kRadixThreads + threadIdx.x;
        if (i < count) {
            const uint32_t kk = s_key[i];
            const uint32_t pos = i + s_delta[(kk >> shift) & mask];
            keys_out[pos] = kk;
            vals_out[pos] = s_val[i];
        }
    }
}

size_t state_slices(size_t nb) { return (nb * 256 * kMaxPasses <= kStateBudgetElems) ? kMaxPasses : 1; }

}  // namespace

size_t hy_radix_hist_elems(size_t n_cap) {
    const size_t nb = (n_cap + kRadixItems - 1) / kRadixItems + 1;
    const size_t one = nb * 256;
    return kWsState + (one > kStateBudgetElems ? one : kStateBudgetElems) + 64;
}

// Largest pair count one sort call supports (30-bit digit prefixes in the look-back words).
size_t hy_radix_max_items() { return (size_t)kValMask; }

void hy_launch_radix(uint32_t* key_a, uint32_t* val_a, uint32_t* key_b, uint32_t* val_b, size_t n_cap,
                     const uint32_t* n_dev, int key_bits, uint32_t* ws, uint32_t* /*scan_scratch*/, cudaStream_t st,
                     uint32_t** out_key, uint32_t** out_val, uint32_t* launches, bool iota_vals) {
    uint32_t *ki = key_a, *vi = val_a, *ko = key_b, *vo = val_b;
    if (n_cap > 0 && key_bits > 0) {
        const size_t nb = (n_cap + kRadixItems - 1) / kRadixItems;
        const int passes = (key_bits + 7) / 8;
        const size_t slices = state_slices(nb + 1);
        const size_t slice = (nb + 1) * 256;
        cudaMemsetAsync(ws, 0, (kWsState + (slices > 1 ? (size_t)passes * slice : 0)) * sizeof(uint32_t), st);
        int dev = 0, sms = 0;   // grid-stride histogram: one wave of resident CTAs
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) sms = 1;
        const unsigned hgrid = (unsigned)(nb < (size_t)sms * 8 ? nb : (size_t)sms * 8);
        radix_global_hist_kernel<<<hgrid, kRadixThreads, 0, st>>>(ki, n_cap, n_dev, passes, key_bits, ws + kWsHist);
        ++*launches;
        for (int p = 0; p < passes; ++p) {
            const int bits = key_bits - 8 * p < 8 ? key_bits - 8 * p : 8;
            uint32_t* state = ws + kWsState + (slices > 1 ? (size_t)p * slice : 0);
            if (slices == 1) cudaMemsetAsync(state, 0, slice * sizeof(uint32_t), st);
            radix_onesweep_kernel<<<(unsigned)nb, kRadixThreads, 0, st>>>(ki, (p == 0 && iota_vals) ? nullptr : vi, ko, vo, n_cap, n_dev, 8 * p,
                                                                         (1u << bits) - 1u, ws + kWsHist + p * 256,
                                                                         ws + kWsTicket + p, state);
            ++*launches;
            uint32_t* t = ki; ki = ko; ko = t;
            t = vi; vi = vo; vo = t;
        }
    }
    *out_key = ki;
    *out_val = vi;
}
