// radix.cu — stable LSD radix sort of (uint32 key, uint32 value) pairs, 9 bits per pass, only the key bits in use.
// S4c of the pass (PAPER.md:47 "ordered by depth", :57): the order (tile, depth bits, id) of DESIGN.md §2 D9 is
// produced by two stable sorts — Gaussians by depth bits (ties keep id order because the compaction is stable),
// then tile entries by tile id.
// One kernel per digit ("onesweep"): a block takes a ticket, ranks its 4096 keys (warp ballots + per-warp digit
// counters: stable, no atomics on the output), publishes its digit counts, resolves its global offsets by
// decoupled look-back over earlier tickets, re-orders the tile in shared memory and writes digit runs coalesced.
// The digit histograms of all passes come from one upfront kernel. HBM traffic per pass = read 8 B + write 8 B per
// pair, the minimum for an out-of-place pass.
//
// Two things keep the number of real passes at three for the depth sort of a frame, which runs beside the field
// kernel on the few SMs that kernel leaves (every pass costs the frame SM-microseconds):
//   * the digits are those of (key - key_sub) with key_sub <= every key (the depth sort passes the bits of z_near: the
//     keys are the bits of depths Z > z_near, positive floats, whose order as integers is their order as floats);
//     a depth range of 2^16 : 1 then fits 27 bits = three 9-bit digits whatever the absolute depths are;
//   * a pass whose digit is the same for every key (seen in its histogram: one bin holds all n) permutes nothing; its
//     blocks copy their tile and leave (no ranking, no look-back). Four passes are always launched for 32-bit keys,
//     the fourth normally being such a copy.
#include "scene.h"

namespace {

constexpr int kRadixThreads = 256;
constexpr int kRadixPer = 16;
constexpr int kRadixItems = kRadixThreads * kRadixPer;  // 4096 pairs per block
constexpr int kWarps = kRadixThreads / 32;
constexpr int kWarpItems = kRadixItems / kWarps;        // 512 consecutive pairs per warp
constexpr int kDigitBits = 9;
constexpr int kBins = 1 << kDigitBits;                  // 512: thread t owns the adjacent bins 2t, 2t + 1
constexpr int kMaxPasses = 4;                           // 36 bits >= 32
constexpr uint32_t kValMask = (1u << 30) - 1u;            // largest pair count of one sort (32-bit indices with room to spare)

// workspace (uint32 elements): [0, 2048) global digit histograms [pass][512]; [2048, 2052) tickets; then one status word
// per tile and pass (these three are cleared per sort), the tiles' digit counts (two 16-bit counts per word) and their
// inclusive prefixes (rows of 512 words) — both reused by every pass: a row is only read once its tile's status word
// of the current pass says so
constexpr size_t kWsHist = 0, kWsTicket = kMaxPasses * kBins, kWsFlags = kWsTicket + 16;
size_t tiles_padded(size_t n_cap) { return ((n_cap + kRadixItems - 1) / kRadixItems + 1 + 31) / 32 * 32; }

// exclusive scan over the 512 bins, two adjacent bins (v0, v1) per thread: returns the exclusive prefix of v0
__device__ __forceinline__ uint32_t block_scan_pairs(uint32_t v0, uint32_t v1, uint32_t* warp_sums /*[8]*/) {
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t v = v0 + v1;
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
radix_global_hist_kernel(const uint32_t* __restrict__ keys, uint32_t n_cap, const uint32_t* __restrict__ n_dev,
                         int passes, uint32_t key_sub, uint32_t* __restrict__ ghist) {
    __shared__ uint32_t h[kMaxPasses][kBins];
    const uint32_t n = n_dev ? *n_dev : n_cap;
    for (int i = threadIdx.x; i < passes * kBins; i += kRadixThreads) (&h[0][0])[i] = 0;
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31;
    for (uint32_t base = blockIdx.x * kRadixItems; base < n; base += gridDim.x * kRadixItems) {
#pragma unroll 4
        for (int k = 0; k < kRadixPer; ++k) {
            const uint32_t i = base + k * kRadixThreads + threadIdx.x;
            const bool in = i < n;
            const uint32_t key = in ? keys[i] - key_sub : 0u;
            for (int p = 0; p < passes; ++p) {
                const uint32_t d = (key >> (kDigitBits * p)) & (kBins - 1);
                // the high digits are often the same for a whole warp (depths share their exponent; the top digit is
                // usually 0 for every key): one add for the warp instead of 32 serialised ones on the same address
                bool uniform = false;
                uint32_t bal = 0;
                if (p >= 2) {   // (p is uniform; every lane takes part in the three warp operations)
                    bal = __ballot_sync(0xffffffffu, in);
                    const uint32_t d_first = __shfl_sync(0xffffffffu, d, __ffs(bal | 0x80000000u) - 1);
                    uniform = __all_sync(0xffffffffu, !in || d == d_first);
                }
                if (uniform) {
                    if (bal && lane == (uint32_t)(__ffs(bal) - 1)) atomicAdd(&h[p][d], (uint32_t)__popc(bal));
                } else if (in) {
                    atomicAdd(&h[p][d], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * kBins; i += kRadixThreads) {
        const uint32_t c = (&h[0][0])[i];
        if (c) atomicAdd(&ghist[i], c);
    }
}

__device__ __forceinline__ uint32_t ld_flag(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_flag(uint32_t* p, uint32_t v) { asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }

// ranks of the 16 rows of a warp's 512 keys within the warp, per digit (stable): packed[k] = digit << 16 | rank.
// FULL: every key of the tile exists (no validity predicates in the ballots).
template <bool FULL>
__device__ __forceinline__ void rank_rows(const uint32_t (&key)[kRadixPer], uint32_t (&packed)[kRadixPer], uint32_t key_sub,
                                          int shift, uint32_t wbase, uint32_t n, uint32_t lane, unsigned short* cw) {
    const uint32_t below = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const bool valid = FULL || wbase + (uint32_t)k * 32u + lane < n;
        const uint32_t d = ((key[k] - key_sub) >> shift) & (kBins - 1);
        // lanes holding the same digit, from one ballot per digit bit: match.any costs several times that when most
        // lanes of a warp hold distinct digits, which is the rule for the low bits of depth keys
        uint32_t peers = FULL ? 0xffffffffu : __ballot_sync(0xffffffffu, valid);
#pragma unroll
        for (int b = 0; b < kDigitBits; ++b) {
            const bool bit = (d >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            peers &= bit ? bal : ~bal;
        }
        uint32_t c = 0;
        if (valid) c = cw[d];
        __syncwarp();
        if (valid && (peers & below) == 0u) cw[d] = (unsigned short)(c + __popc(peers));   // the lowest peer writes
        __syncwarp();
        packed[k] = valid ? ((d << 16) | (c + __popc(peers & below))) : 0xffffffffu;
    }
}

#ifndef HY_RADIX_MINB
#define HY_RADIX_MINB 3
#endif
__global__ void __launch_bounds__(kRadixThreads, HY_RADIX_MINB)
radix_onesweep_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                      uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, uint32_t n_cap,
                      const uint32_t* __restrict__ n_dev, int shift, uint32_t key_sub, const uint32_t* __restrict__ ghist,
                      uint32_t* __restrict__ ticket, uint32_t* __restrict__ flags, uint32_t* __restrict__ agg, uint2* __restrict__ incl) {
    __shared__ unsigned short cnt[kWarps][kBins];   // per warp and digit: count, then first slot in the re-ordered tile
    __shared__ uint32_t s_key[kRadixItems];
    __shared__ uint32_t s_val[kRadixItems];
    __shared__ uint32_t s_delta[kBins];
    __shared__ uint32_t s_warp[kWarps];
    __shared__ uint32_t s_tile, s_back;
    const uint32_t n = n_dev ? *n_dev : n_cap;
    const uint32_t t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const uint2 gh = *reinterpret_cast<const uint2*>(ghist + 2 * t);   // the whole array's counts of this thread's two digits
    // one digit for every key: this pass permutes nothing. Copy the tile (tickets and look-back are not needed)
    if (__syncthreads_or((gh.x == n) | (gh.y == n))) {
        const uint32_t base = blockIdx.x * kRadixItems;
#pragma unroll 4
        for (int k = 0; k < kRadixPer; ++k) {
            const uint32_t i = base + k * kRadixThreads + t;
            if (i < n) {
                keys_out[i] = keys_in[i];
                vals_out[i] = vals_in ? vals_in[i] : i;
            }
        }
        return;
    }
    if (t == 0) s_tile = atomicAdd(ticket, 1u);
    for (int d = t; d < kWarps * kBins / 2; d += kRadixThreads) reinterpret_cast<uint32_t*>(&cnt[0][0])[d] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base = tile * kRadixItems;
    if (base >= n) return;   // tickets are handed out in order: every earlier tile exists and is running or done
    const bool full = base + kRadixItems <= n;

    uint32_t key[kRadixPer], val[kRadixPer], packed[kRadixPer];
    const uint32_t wbase = base + warp * kWarpItems;
    if (full) {
#pragma unroll
        for (int k = 0; k < kRadixPer; ++k) {
            const uint32_t i = wbase + k * 32 + lane;
            key[k] = keys_in[i];
            val[k] = vals_in ? vals_in[i] : i;   // no values yet: the value is the index
        }
        rank_rows<true>(key, packed, key_sub, shift, wbase, n, lane, cnt[warp]);
    } else {
#pragma unroll
        for (int k = 0; k < kRadixPer; ++k) {
            const uint32_t i = wbase + k * 32 + lane;
            const bool valid = i < n;
            key[k] = valid ? keys_in[i] : 0u;
            val[k] = valid ? (vals_in ? vals_in[i] : i) : 0u;
        }
        rank_rows<false>(key, packed, key_sub, shift, wbase, n, lane, cnt[warp]);
    }
    __syncthreads();
    // thread t owns digits 2t, 2t + 1: exclusive scan over the warps, block totals, publish, look back
    uint32_t total[2] = {0u, 0u};
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
        const uint32_t c2 = *reinterpret_cast<const uint32_t*>(&cnt[w][2 * t]);
        *reinterpret_cast<uint32_t*>(&cnt[w][2 * t]) = total[0] | (total[1] << 16);
        total[0] += c2 & 0xFFFFu;
        total[1] += c2 >> 16;
    }
    // Decoupled look-back with ONE status word per tile (0 nothing, 1 digit counts of the tile published, 2 inclusive
    // prefixes published) and plain arrays of counts: a warp finds the nearest predecessor whose inclusive prefixes
    // are out, then every thread adds that row and the count rows in between for its two digits. (Per-digit status
    // words made every thread walk and test its own chain: a quarter of the kernel's instructions.)
    agg[(size_t)tile * (kBins / 2) + t] = total[0] | (total[1] << 16);   // (counts of one tile: <= 4096)
    if (tile == 0) incl[t] = make_uint2(total[0], total[1]);
    __threadfence();
    const uint32_t gexcl = block_scan_pairs(gh.x, gh.y, s_warp);          // first output slot of digit 2t over the whole array
    if (t == 0) st_flag(flags + tile, tile == 0 ? 2u : 1u);                // (after the barriers of the scan: every thread's rows are out)
    const uint32_t dstart = block_scan_pairs(total[0], total[1], s_warp); // first slot of digit 2t inside this tile
    uint32_t prefix[2] = {0u, 0u};
    if (tile > 0) {
        uint32_t top = tile - 1;   // the look-back window is tiles top, top - 1, ..., top - 31
        for (;;) {
            if (warp == 0) {
                uint32_t back;
                for (;;) {
                    const uint32_t fl = lane <= top ? ld_flag(flags + (top - lane)) : 2u;
                    const uint32_t two = __ballot_sync(0xffffffffu, fl == 2u), zero = __ballot_sync(0xffffffffu, fl == 0u);
                    const uint32_t first2 = two ? (uint32_t)__ffs(two) - 1u : 32u;            // nearest tile with inclusive prefixes
                    if ((zero & (first2 < 32u ? (1u << first2) - 1u : 0xffffffffu)) == 0u) { back = first2; break; }   // all in front of it counted
                }
                if (lane == 0) s_back = back;
            }
            __syncthreads();
            const uint32_t back = s_back;
            __threadfence();
            const uint32_t n_agg = back < 32u ? back : 32u;
            for (uint32_t i = 0; i < n_agg; ++i) {
                const uint32_t v = __ldcg(agg + (size_t)(top - i) * (kBins / 2) + t);
                prefix[0] += v & 0xFFFFu; prefix[1] += v >> 16;
            }
            if (back < 32u) {
                if (back <= top) {   // (beyond tile 0 the sentinel stands for an all-zero inclusive row)
                    const uint2 v = __ldcg(incl + (size_t)(top - back) * (kBins / 2) + t);
                    prefix[0] += v.x; prefix[1] += v.y;
                }
                break;
            }
            top -= 32u;   // 32 counted tiles and no inclusive one among them: go on further back (top >= 32 here)
            __syncthreads();
        }
        incl[(size_t)tile * (kBins / 2) + t] = make_uint2(prefix[0] + total[0], prefix[1] + total[1]);
        __threadfence();
        __syncthreads();
        if (t == 0) st_flag(flags + tile, 2u);
    }
    s_delta[2 * t] = gexcl + prefix[0] - dstart;
    s_delta[2 * t + 1] = gexcl + gh.x + prefix[1] - (dstart + total[0]);
    {
        const uint32_t add = dstart | ((dstart + total[0]) << 16);   // (no carry between the halves: slots < 4096)
#pragma unroll
        for (int w = 0; w < kWarps; ++w) *reinterpret_cast<uint32_t*>(&cnt[w][2 * t]) += add;
    }
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
    const uint32_t count = n - base < (uint32_t)kRadixItems ? n - base : (uint32_t)kRadixItems;
#pragma unroll
    for (int k = 0; k < kRadixPer; ++k) {
        const uint32_t i = k * kRadixThreads + t;
        if (i < count) {
            const uint32_t kk = s_key[i];
            const uint32_t pos = i + s_delta[((kk - key_sub) >> shift) & (kBins - 1)];
            keys_out[pos] = kk;
            vals_out[pos] = s_val[i];
        }
    }
}

}  // namespace

size_t hy_radix_hist_elems(size_t n_cap) {
    const size_t nbp = tiles_padded(n_cap);
    return kWsFlags + kMaxPasses * nbp + nbp * (kBins / 2) + nbp * kBins + 64;
}

// Largest pair count one sort call supports.
size_t hy_radix_max_items() { return (size_t)kValMask; }

// key_sub: a value no key is below; the digits are those of key - key_sub (see the head of this file). 0 = plain keys.
void hy_launch_radix(uint32_t* key_a, uint32_t* val_a, uint32_t* key_b, uint32_t* val_b, size_t n_cap,
                     const uint32_t* n_dev, int key_bits, uint32_t* ws, uint32_t* /*scan_scratch*/, cudaStream_t st,
                     uint32_t** out_key, uint32_t** out_val, uint32_t* launches, bool iota_vals, uint32_t key_sub) {
    uint32_t *ki = key_a, *vi = val_a, *ko = key_b, *vo = val_b;
    if (n_cap > 0 && key_bits > 0) {
        const size_t nb = (n_cap + kRadixItems - 1) / kRadixItems;
        const int passes = (key_bits + kDigitBits - 1) / kDigitBits;
        const size_t nbp = tiles_padded(n_cap);
        uint32_t* const agg = ws + kWsFlags + kMaxPasses * nbp;
        uint2* const incl = reinterpret_cast<uint2*>(agg + nbp * (kBins / 2));
        cudaMemsetAsync(ws, 0, (kWsFlags + (size_t)passes * nbp) * sizeof(uint32_t), st);
        int dev = 0, sms = 0;   // grid-stride histogram: one wave of resident CTAs
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) sms = 1;
        const unsigned hgrid = (unsigned)(nb < (size_t)sms * 8 ? nb : (size_t)sms * 8);
        radix_global_hist_kernel<<<hgrid, kRadixThreads, 0, st>>>(ki, (uint32_t)n_cap, n_dev, passes, key_sub, ws + kWsHist);
        ++*launches;
        for (int p = 0; p < passes; ++p) {
            radix_onesweep_kernel<<<(unsigned)nb, kRadixThreads, 0, st>>>(ki, (p == 0 && iota_vals) ? nullptr : vi, ko, vo, (uint32_t)n_cap, n_dev,
                                                                         kDigitBits * p, key_sub, ws + kWsHist + p * kBins,
                                                                         ws + kWsTicket + p, ws + kWsFlags + (size_t)p * nbp, agg, incl);
            ++*launches;
            uint32_t* t = ki; ki = ko; ko = t;
            t = vi; vi = vo; vo = t;
        }
    }
    *out_key = ki;
    *out_val = vi;
}
