// scan.cu — device-wide exclusive prefix sum of uint32 (reduce, scan the partials recursively, apply).
// Used by the compaction (S1), the tile-entry offsets (S4b) and the radix sort's digit offsets (S4c).
#include "scene.h"

namespace {

constexpr int kScanThreads = 256;
constexpr int kScanPer = 8;
constexpr int kScanItems = kScanThreads * kScanPer;  // 2048 per block

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
    __shared__ uint32_t warp_sums[kScanThreads / 32];
    __shared__ uint32_t block_total;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= (uint32_t)d) incl += u;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < kScanThreads / 32 ? warp_sums[lane] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int d = 1; d < kScanThreads / 32; d <<= 1) {
            uint32_t u = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= (uint32_t)d) wi += u;
        }
        if (lane < kScanThreads / 32) warp_sums[lane] = wi - w;
        if (lane == kScanThreads / 32 - 1) block_total = wi;
    }
    __syncthreads();
    *total = block_total;
    return warp_sums[warp] + incl - v;
}

__global__ void __launch_bounds__(kScanThreads)
scan_reduce_kernel(const uint32_t* __restrict__ in, size_t n, uint32_t* __restrict__ partial) {
    const size_t base = (size_t)blockIdx.x * kScanItems + (size_t)threadIdx.x * kScanPer;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanPer; ++k)
        if (base + k < n) s += in[base + k];
    uint32_t total;
    block_exclusive_scan(s, &total);
    if (threadIdx.x == 0) partial[blockIdx.x] = total;
}

// out[i] = base[block] + exclusive scan within the block. base may be null (single block).
__global__ void __launch_bounds__(kScanThreads)
scan_apply_kernel(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, size_t n,
                  const uint32_t* __restrict__ base_of_block) {
    const size_t base = (size_t)blockIdx.x * kScanItems + (size_t)threadIdx.x * kScanPer;
    uint32_t v[kScanPer];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < kScanPer; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0u;
        s += v[k];
    }
    uint32_t total;
    uint32_t excl = block_exclusive_scan(s, &total);
    excl += base_of_block ? base_of_block[blockIdx.x] : 0u;
#pragma unroll
    for (int k = 0; k < kScanPer; ++k) {
        if (base + k < n) out[base + k] = excl;
        excl += v[k];
    }
}

}  // namespace

size_t hy_scan_scratch_elems(size_t n) {
    size_t total = 0;
    while (n > (size_t)kScanItems) {
        n = (n + kScanItems - 1) / kScanItems;
        total += 2 * n;  // partial sums + their scanned copy
    }
    return total + 8;
}

void hy_launch_scan(const uint32_t* in, uint32_t* out, size_t n, uint32_t* scratch, cudaStream_t st,
                    uint32_t* launches) {
    if (n == 0) return;
    const size_t nb = (n + kScanItems - 1) / kScanItems;
    if (nb == 1) {
        scan_apply_kernel<<<1, kScanThreads, 0, st>>>(in, out, n, nullptr);
        ++*launches;
        return;
    }
    uint32_t* partial = scratch;
    uint32_t* partial_scanned = scratch + nb;
    scan_reduce_kernel<<<(unsigned)nb, kScanThreads, 0, st>>>(in, n, partial);
    ++*launches;
    hy_launch_scan(partial, partial_scanned, nb, scratch + 2 * nb, st, launches);
    scan_apply_kernel<<<(unsigned)nb, kScanThreads, 0, st>>>(in, out, n, partial_scanned);
    ++*launches;
}

// The frame's counters to the (pinned, device-visible) host block: 16 words by one warp (see api.cu render_impl).
namespace {
__global__ void counters_to_host_kernel(const uint32_t* __restrict__ dev, volatile uint32_t* __restrict__ host) {
    if (threadIdx.x < sizeof(FrameCounters) / 4) host[threadIdx.x] = dev[threadIdx.x];
    __threadfence_system();
}
}  // namespace

void hy_launch_counters_to_host(const FrameCounters* dev, FrameCounters* pinned_host, cudaStream_t st) {
    static_assert(sizeof(FrameCounters) % 4 == 0 && sizeof(FrameCounters) <= 128, "one warp copies the counters");
    counters_to_host_kernel<<<1, 32, 0, st>>>(reinterpret_cast<const uint32_t*>(dev), reinterpret_cast<volatile uint32_t*>(pinned_host));
}
