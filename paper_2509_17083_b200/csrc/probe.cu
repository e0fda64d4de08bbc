// probe.cu — the two microprobes SURVEY.md §8(d) asks for before any roofline is quoted: MEASURED_PEAKS.json holds
// the HBM copy rate and the dense bf16 rate, but neither of the ceilings the two dominant stages of the pass run
// against: (1) the rate at which an SM can look up scattered sectors of an L2-resident table (what bounds the grid
// gathers of S2, Eq. 3: 256 look-ups per visible Gaussian into tables that fit the 126 MB L2), and (2) the
// sustained instruction issue rate of plain fp32 ALU code with one MUFU per ~20 instructions (what bounds the
// alpha-blend loop of S5, Eq. 1). `bench.py --probe` runs them through hyrf_probe_gather / hyrf_probe_issue
// and writes the JSON line kept under profiles/. Nothing here is on the render path.
#include <cuda_runtime.h>
#include <stdint.h>

#include "scene.h"

namespace {

constexpr int kProbeThreads = 256;

__device__ __forceinline__ uint32_t mix(uint32_t x) {   // a cheap integer hash (two rounds of multiply-xorshift)
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// Every lane performs `iters` x 8 independent look-ups of one entry (EB = 4 or 8 bytes) of a table of n_entries
// (a power of two). `share` lanes in a row read the SAME 32-byte sector (share = 1: 32 distinct sectors per
// instruction; 2: 16 — the two-lane gather of field_mma.cu; 4: 8), `line` = 1 spreads consecutive groups over the
// four sectors of one 128-byte line instead of over the whole table (distinct sectors, shared tags).
template <int EB>
__global__ void __launch_bounds__(kProbeThreads)
gather_probe_kernel(const uint8_t* __restrict__ table, uint32_t n_entries, uint32_t iters, uint32_t share, uint32_t line,
                    uint32_t* __restrict__ sink) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t grp = lane / share;                    // lanes of one group hit one sector
    const uint32_t wid = gid >> 5;
    const uint32_t per_sector = 32u / EB;
    uint32_t acc = 0;
    for (uint32_t it = 0; it < iters; ++it) {
        uint32_t v[8];
#pragma unroll
        for (uint32_t k = 0; k < 8; ++k) {
            const uint32_t seq = (it * 8u + k) * 0x9E3779B9u;
            uint32_t sector;
            if (line) {   // groups 4g .. 4g+3 of a warp share a 128-byte line, one sector each
                const uint32_t ln = mix(seq ^ (wid * 0x85ebca6bu) ^ ((grp >> 2) * 0xc2b2ae35u));
                sector = (ln << 2) | (grp & 3u);
            } else {
                sector = mix(seq ^ (wid * 0x85ebca6bu) ^ (grp * 0xc2b2ae35u));
            }
            const uint32_t e = (sector * per_sector + (lane % share) % per_sector) & (n_entries - 1u);
            if (EB == 4) v[k] = __ldg(reinterpret_cast<const uint32_t*>(table) + e);
            else { const uint2 t = __ldg(reinterpret_cast<const uint2*>(table) + e); v[k] = t.x ^ t.y; }
        }
#pragma unroll
        for (uint32_t k = 0; k < 8; ++k) acc += v[k];
    }
    if (acc == 0x12345678u) sink[gid] = acc;              // keeps the loads alive, practically never taken
}

// Issue probe: every thread runs 8 independent chains; one iteration = `kBody` fp32 instructions in the mix asked for.
//   kind 0: FFMA only (3-register form)            kind 1: FFMA + integer ALU alternating (two pipes)
//   kind 2: the blend-loop mix: 16 fp32 ops + 1 MUFU.EX2 + 3 compare/select per "pair"
template <int KIND>
__global__ void __launch_bounds__(kProbeThreads)
issue_probe_kernel(uint32_t iters, float seed, float* __restrict__ sink) {
    float a[8];
    uint32_t q[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = seed + (float)(threadIdx.x + i); q[i] = threadIdx.x * 7u + i; }
    const float m = 0.999f, c = 1e-3f;
    for (uint32_t it = 0; it < iters; ++it) {
        if (KIND == 0) {
#pragma unroll
            for (int r = 0; r < 4; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = __fmaf_rn(a[i], m, c);                 // 32 FFMA
        } else if (KIND == 1) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) { a[i] = __fmaf_rn(a[i], m, c); q[i] = (q[i] ^ (q[i] >> 3)) + 0x9E37u; }   // 16 FFMA + 32 ALU
        } else if (KIND == 3) {   // packed fp32: FFMA2 = two independent fma.rn per lane in one issue slot (sm_100)
            unsigned long long mm, cc;
            asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
            asm("mov.b64 %0, {%1, %1};" : "=l"(cc) : "f"(c));
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 8; i += 2) {
                    unsigned long long v;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(a[i]), "f"(a[i + 1]));
                    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v) : "l"(mm), "l"(cc));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[i]), "=f"(a[i + 1]) : "l"(v));
                }                                                                          // 32 FFMA2 = 64 fma
        } else {
#pragma unroll
            for (int i = 0; i < 2; ++i) {   // two "pairs" per iteration
                const float dx = a[i] - 1.5f, dy = a[i + 2] - 2.5f;                                    // 2
                const float power = __fmaf_rn(-0.5f, __fmaf_rn(a[4] * dx, dx, (a[5] * dy) * dy), -((a[6] * dx) * dy));   // 7
                float e;
                asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(power * 1.44269504f));        // 1 + MUFU
                const float alpha = fminf(0.99f, a[7] * e);                                            // 2
                const float Tn = a[i + 2] * (1.0f - alpha);                                            // 2
                const bool valid = !(power > 0.0f) && !(alpha < 1.0f / 255.0f);                        // 2
                const bool blend = valid && !(Tn < 1e-4f);                                             // 1
                const float w = blend ? alpha * a[i + 2] : 0.0f;                                       // 2
                a[4] = __fmaf_rn(c, w, a[4]); a[5] = __fmaf_rn(m, w, a[5]); a[6] = __fmaf_rn(c, w, a[6]);   // 3
                a[i + 2] = blend ? Tn : a[i + 2];                                                      // 1
                a[i] = a[i] * m + c;                                                                   // 2
            }
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i] + (float)q[i];
    if (s == 1.2345e-30f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void fill_kernel(uint32_t* p, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = mix((uint32_t)i) | 1u;
}

}  // namespace

extern "C" hyrf_status hyrf_probe_gather(int32_t device, uint64_t table_bytes, uint32_t entry_bytes, uint32_t ctas_per_sm,
                                         uint32_t share, uint32_t line, uint32_t iters, double* lookups_per_s,
                                         double* sectors_per_s, float* ms_out) {
    if (!lookups_per_s || !sectors_per_s || !ms_out) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_probe_gather: NULL output");
    if ((entry_bytes != 4 && entry_bytes != 8) || table_bytes < 4096 || (table_bytes & (table_bytes - 1)) || ctas_per_sm < 1 ||
        ctas_per_sm > 8 || (share != 1 && share != 2 && share != 4) || line > 1 || iters < 1)
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_probe_gather: table_bytes must be a power of two >= 4096, entry_bytes 4 or 8, ctas_per_sm 1..8, share 1/2/4, line 0/1");
    cudaError_t e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return hy_cuda_fail(e, "cudaDeviceGetAttribute");
    uint8_t* table = nullptr;
    uint32_t* sink = nullptr;
    const uint32_t grid = (uint32_t)sms * ctas_per_sm;
    if ((e = cudaMalloc(&table, table_bytes)) != cudaSuccess) return hy_cuda_fail(e, "cudaMalloc(probe table)");
    if ((e = cudaMalloc(&sink, (size_t)grid * kProbeThreads * 4)) != cudaSuccess) { cudaFree(table); return hy_cuda_fail(e, "cudaMalloc(probe sink)"); }
    fill_kernel<<<1024, 256>>>(reinterpret_cast<uint32_t*>(table), table_bytes / 4);
    const uint32_t n_entries = (uint32_t)(table_bytes / entry_bytes);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {   // the first repetitions also bring the table into L2
        cudaEventRecord(e0);
        if (entry_bytes == 4) gather_probe_kernel<4><<<grid, kProbeThreads>>>(table, n_entries, iters, share, line, sink);
        else gather_probe_kernel<8><<<grid, kProbeThreads>>>(table, n_entries, iters, share, line, sink);
        cudaEventRecord(e1);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 2 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(table); cudaFree(sink);
    if (e != cudaSuccess) return hy_cuda_fail(e, "gather_probe_kernel");
    const double lookups = (double)grid * kProbeThreads * 8.0 * iters;
    *lookups_per_s = lookups / (best * 1e-3);
    *sectors_per_s = *lookups_per_s / share;   // distinct 32-byte sectors touched per second
    *ms_out = best;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_probe_issue(int32_t device, uint32_t kind, uint32_t ctas_per_sm, uint32_t iters,
                                        double* warp_instr_per_s, float* ms_out) {
    if (!warp_instr_per_s || !ms_out) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_probe_issue: NULL output");
    if (kind > 3 || ctas_per_sm < 1 || ctas_per_sm > 8 || iters < 1) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_probe_issue: kind 0..3, ctas_per_sm 1..8");
    cudaError_t e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return hy_cuda_fail(e, "cudaDeviceGetAttribute");
    const uint32_t grid = (uint32_t)sms * ctas_per_sm;
    iters = (iters + 15u) & ~15u;
    float* sink = nullptr;
    if ((e = cudaMalloc(&sink, (size_t)grid * kProbeThreads * 4)) != cudaSuccess) return hy_cuda_fail(e, "cudaMalloc(probe sink)");
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        if (kind == 3) issue_probe_kernel<3><<<grid, kProbeThreads>>>(iters, 0.5f, sink);
        else if (kind == 0) issue_probe_kernel<0><<<grid, kProbeThreads>>>(iters, 0.5f, sink);
        else if (kind == 1) issue_probe_kernel<1><<<grid, kProbeThreads>>>(iters, 0.5f, sink);
        else issue_probe_kernel<2><<<grid, kProbeThreads>>>(iters, 0.5f, sink);
        cudaEventRecord(e1);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 1 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return hy_cuda_fail(e, "issue_probe_kernel");
    // SASS instructions per thread and iteration of the main loop, counted in `cuobjdump -sass` of this file (nvcc 12.9,
    // -O3 -fmad=false): kind 0 is unrolled x 4 into 128 FFMA + 4 of loop control; kind 1 x 2 into 32 FFMA + 96 integer
    // ALU + 4; kind 2 x 2 into 107 (20 FFMA, 40 FMUL, 16 FADD, 4 FMNMX, 12 FSETP, 8 FSEL, 4 MUFU.EX2, 3 of loop control):
    // one MUFU per 26.75 issued instructions. iters is rounded up to a multiple of 4 by the caller below.
    const double body = kind == 0 ? 33.0 : (kind == 1 ? 66.0 : (kind == 3 ? 32.25 : 53.5));   // kind 3: x 16 into 512 FFMA2 + 4
    *warp_instr_per_s = (double)grid * (kProbeThreads / 32) * body * iters / (best * 1e-3);
    *ms_out = best;
    return HYRF_OK;
}
