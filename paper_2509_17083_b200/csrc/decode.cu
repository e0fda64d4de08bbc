// decode.cu — decode of the compressed explicit Gaussians at upload (PAPER.md:227-229 items 1-2; DESIGN.md §2 D1'):
// positions stored as IEEE binary16, the five explicit properties (s_e, alpha_e, c_e) as residual-VQ codes.
//
// Once per hyrf_upload_explicit_rvq, not per frame: the render pass keeps reading the fp32 SoA and the Morton
// records built from it (hy_prepare_morton), so a frame costs the same with or without the compressed model.
// HBM-bound: per Gaussian 6 B of positions + 2 S B of codes in, 32 B out; the codebooks (S K 20 B) sit in shared
// memory when they fit 48 KB (the usual 6 x 64 codebooks are 7.5 KB), else they are read through L1/L2.
//
// Arithmetic (frozen in DESIGN.md §2 D1'): p = float(binary16), exact; x = C_0[k_0] + C_1[k_1] + ... in binary32,
// stage order, starting from the stage-0 row itself. A code >= K writes nothing and reports its Gaussian.
#include <cuda_fp16.h>

#include "scene.h"

namespace {

constexpr int kDecodeThreads = 256;
constexpr size_t kBookSmemMax = 48 * 1024;

// VEC Gaussians per thread: 4 (8-byte loads of positions and codes, 16-byte stores) when n % 4 == 0 and every row
// is 8-byte aligned, else 1.
template <int VEC>
__global__ void __launch_bounds__(kDecodeThreads)
explicit_decode_kernel(const uint16_t* __restrict__ pos_h, const uint16_t* __restrict__ codes,
                       const float* __restrict__ codebooks, uint32_t n, uint32_t S, uint32_t K, bool book_in_smem,
                       float* __restrict__ pos, float* __restrict__ scale, float* __restrict__ opac,
                       float* __restrict__ rgb, uint32_t* __restrict__ first_bad) {
    extern __shared__ float s_book[];
    const float* book = codebooks;
    if (book_in_smem) {
        const uint32_t words = S * K * 5;
        for (uint32_t w = threadIdx.x; w < words; w += kDecodeThreads) s_book[w] = __ldg(codebooks + w);
        __syncthreads();
        book = s_book;
    }
    const uint32_t groups = n / VEC;
    for (uint32_t g = blockIdx.x * kDecodeThreads + threadIdx.x; g < groups; g += gridDim.x * kDecodeThreads) {
        const size_t i0 = (size_t)g * VEC;
        float x[VEC][5];
        bool bad[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) bad[v] = false;
        for (uint32_t s = 0; s < S; ++s) {
            uint16_t k[VEC];
            if constexpr (VEC == 4) {
                const uint2 c = __ldg(reinterpret_cast<const uint2*>(codes + (size_t)s * n + i0));
                k[0] = (uint16_t)(c.x & 0xFFFFu); k[1] = (uint16_t)(c.x >> 16);
                k[2] = (uint16_t)(c.y & 0xFFFFu); k[3] = (uint16_t)(c.y >> 16);
            } else {
                k[0] = __ldg(codes + (size_t)s * n + i0);
            }
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const bool ok = k[v] < K;
                bad[v] |= !ok;
                const float* row = book + ((size_t)s * K + (ok ? k[v] : 0u)) * 5;
#pragma unroll
                for (int d = 0; d < 5; ++d) x[v][d] = (s == 0) ? row[d] : __fadd_rn(x[v][d], row[d]);
            }
        }
        bool any_bad = false;
#pragma unroll
        for (int v = 0; v < VEC; ++v)
            if (bad[v]) { atomicMin(first_bad, (uint32_t)(i0 + v)); any_bad = true; }
        if (any_bad) continue;
        if constexpr (VEC == 4) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const uint2 h = __ldg(reinterpret_cast<const uint2*>(pos_h + (size_t)a * n + i0));
                float4 p;
                p.x = __half2float(__ushort_as_half((unsigned short)(h.x & 0xFFFFu)));
                p.y = __half2float(__ushort_as_half((unsigned short)(h.x >> 16)));
                p.z = __half2float(__ushort_as_half((unsigned short)(h.y & 0xFFFFu)));
                p.w = __half2float(__ushort_as_half((unsigned short)(h.y >> 16)));
                *reinterpret_cast<float4*>(pos + (size_t)a * n + i0) = p;
            }
            *reinterpret_cast<float4*>(scale + i0) = make_float4(x[0][0], x[1][0], x[2][0], x[3][0]);
            *reinterpret_cast<float4*>(opac + i0) = make_float4(x[0][1], x[1][1], x[2][1], x[3][1]);
#pragma unroll
            for (int c = 0; c < 3; ++c)
                *reinterpret_cast<float4*>(rgb + (size_t)c * n + i0) =
                    make_float4(x[0][2 + c], x[1][2 + c], x[2][2 + c], x[3][2 + c]);
        } else {
#pragma unroll
            for (int a = 0; a < 3; ++a)
                pos[(size_t)a * n + i0] = __half2float(__ushort_as_half(__ldg(pos_h + (size_t)a * n + i0)));
            scale[i0] = x[0][0];
            opac[i0] = x[0][1];
#pragma unroll
            for (int c = 0; c < 3; ++c) rgb[(size_t)c * n + i0] = x[0][2 + c];
        }
    }
}

}  // namespace

// Enqueues the decode on the scene's stream. first_bad (device u32) must hold 0xFFFFFFFF; afterwards it holds the
// smallest Gaussian index with a code >= K, if any. Grid: the SM count x the resident CTAs per SM.
hyrf_status hy_launch_explicit_decode(hyrf_scene* s, const uint16_t* pos_h, const uint16_t* codes,
                                      const float* codebooks, uint32_t S, uint32_t K, uint32_t* first_bad) {
    const uint32_t n = s->N;
    const size_t book_bytes = (size_t)S * K * 5 * sizeof(float);
    const bool in_smem = book_bytes <= kBookSmemMax;
    const size_t smem = in_smem ? book_bytes : 0;
    const bool vec4 = (n % 4 == 0) && ((reinterpret_cast<uintptr_t>(pos_h) | reinterpret_cast<uintptr_t>(codes)) % 8 == 0);
    const int sms = s->sm_count;
    const uint32_t groups = vec4 ? n / 4 : n;
    const uint32_t want = (groups + kDecodeThreads - 1) / kDecodeThreads;
    int per_sm = 1;   // one wave of resident CTAs, grid-stride beyond
    if (vec4) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, explicit_decode_kernel<4>, kDecodeThreads, smem);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, explicit_decode_kernel<1>, kDecodeThreads, smem);
    const uint32_t cap = (uint32_t)sms * (uint32_t)(per_sm > 0 ? per_sm : 1);
    const uint32_t grid = want < cap ? (want ? want : 1u) : cap;
    if (vec4)
        explicit_decode_kernel<4><<<grid, kDecodeThreads, smem, s->stream>>>(pos_h, codes, codebooks, n, S, K, in_smem,
                                                                             s->pos, s->scale, s->opac, s->rgb, first_bad);
    else
        explicit_decode_kernel<1><<<grid, kDecodeThreads, smem, s->stream>>>(pos_h, codes, codebooks, n, S, K, in_smem,
                                                                             s->pos, s->scale, s->opac, s->rgb, first_bad);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return hy_cuda_fail(e, "explicit_decode_kernel");
    return HYRF_OK;
}
