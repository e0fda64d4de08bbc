// background.cu — S6: neural background composited behind the splats, PAPER.md:124–134 (Eq. 10–11) and A.2
// (:360–378, Eq. 15–18). For every pixel whose residual transmittance passes tau_T: ray through the pixel,
// intersection with the background sphere (positive root), contraction, bg grid encode, PE of the ray direction,
// bg decoder, sigmoid, out = C_fg + T * c_s. Arithmetic DESIGN.md §2 D11.
#include "mlp.cuh"
#include "scene.h"

namespace {

constexpr int kBgThreads = 128;

struct BgArgs {
    GridDev grid;
    MlpDev mlp;
    FrameDev f;
    uint32_t pe_octaves;
    const float* finalT;
    float* out_rgb;
    const uint32_t* bg_list;          // pixels with T > tau_T, compacted by the rasterizer
    const FrameCounters* counters;
};

template <int CL, int CHID, int CNH, int DT>   // DT: HY_DT_F32 / HY_DT_F16 / HY_DT_U8 (8-bit tables, fp16 decoders)
__global__ void __launch_bounds__(kBgThreads)
background_kernel(const BgArgs A) {
    extern __shared__ __align__(16) float smem_w[];
    constexpr bool FP16 = DT != HY_DT_F32;
    const int L = CL > 0 ? CL : (int)A.grid.levels;
    const int in_dim = (int)A.mlp.in_dim, hid = (int)A.mlp.hidden, nh = (int)A.mlp.n_hidden;
    const int nw = in_dim * hid + (nh - 1) * hid * hid + hid * 3;
    if (FP16) {
        const __half* w = reinterpret_cast<const __half*>(A.mlp.w);
        for (int i = threadIdx.x; i < nw; i += kBgThreads) smem_w[i] = __half2float(w[i]);
    } else {
        const float* w = reinterpret_cast<const float*>(A.mlp.w);
        for (int i = threadIdx.x; i < nw; i += kBgThreads) smem_w[i] = w[i];
    }
    __syncthreads();
    const FrameDev& f = A.f;
    constexpr int MAXD = CL > 0 ? (2 * CL + 24 > CHID ? 2 * CL + 24 : CHID) : HYRF_MAX_WIDTH;
    const uint32_t n_bg = A.counters->n_bg;
    for (uint32_t q = blockIdx.x * kBgThreads + threadIdx.x; q < n_bg; q += gridDim.x * kBgThreads) {
        const int p = (int)A.bg_list[q];
        const float T = A.finalT[p];
        const int pi = p % f.W, pj = p / f.W;
        const float dcx = __fdiv_rn(__fsub_rn((float)pi, f.cx), f.fx), dcy = __fdiv_rn(__fsub_rn((float)pj, f.cy), f.fy);
        float dw[3], d[3], ps[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) dw[k] = __fmaf_rn(f.R[6 + k], 1.0f, __fmaf_rn(f.R[3 + k], dcy, __fmul_rn(f.R[k], dcx)));
        const float n = __fsqrt_rn(__fmaf_rn(dw[2], dw[2], __fmaf_rn(dw[1], dw[1], __fmul_rn(dw[0], dw[0]))));
#pragma unroll
        for (int k = 0; k < 3; ++k) d[k] = __fdiv_rn(dw[k], n);
        const float Bq = __fmul_rn(2.0f, __fmaf_rn(f.o[2], d[2], __fmaf_rn(f.o[1], d[1], __fmul_rn(f.o[0], d[0]))));
        const float Cq = __fsub_rn(__fmaf_rn(f.o[2], f.o[2], __fmaf_rn(f.o[1], f.o[1], __fmul_rn(f.o[0], f.o[0]))),
                                   __fmul_rn(f.bg_radius, f.bg_radius));
        const float disc = __fmaf_rn(Bq, Bq, __fmul_rn(-4.0f, Cq));
        const float t = __fmul_rn(0.5f, __fadd_rn(-Bq, __fsqrt_rn(disc)));
#pragma unroll
        for (int k = 0; k < 3; ++k) ps[k] = __fmaf_rn(t, d[k], f.o[k]);
        float x[3];
        hy_contract(f, ps[0], ps[1], ps[2], x);
        float bufa[MAXD], bufb[MAXD], raw[3];
#pragma unroll
        for (int l = 0; l < L; ++l) {
            float f0, f1;
            hy_grid_level<DT>(A.grid, l, x, f0, f1);
            bufa[2 * l] = FP16 ? hy_round_half(f0) : f0;
            bufa[2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
        }
        if constexpr (CL > 0 && CNH == 1) {
            // layer by layer as loops over groups of four neurons: unrolled over its 64 neurons the decoder is ~4 500
            // instructions, and 20 warps per SM at different places in them wait for instruction fetches (mlp.cuh)
            hy_dir_pe<FP16>(d, 4, bufa + 2 * CL);
            mlp_dense_ct<FP16, 2 * CL + 24, true, CHID>(smem_w, bufa, bufb);
            mlp_dense_ct<FP16, CHID, false, 3>(smem_w + CHID * (2 * CL + 24), bufb, raw);
        } else if constexpr (CL > 0) {
            hy_dir_pe<FP16>(d, 4, bufa + 2 * CL);
            mlp_eval<2 * CL + 24, CHID, CNH, 3, FP16>(smem_w, 0, 0, 0, bufa, bufb, raw);
        } else {
            hy_dir_pe<FP16>(d, (int)A.pe_octaves, bufa + 2 * L);
            for (int k = 2 * L + 6 * (int)A.pe_octaves; k < in_dim; ++k) bufa[k] = 0.0f;
            mlp_eval<0, 0, 0, 3, FP16>(smem_w, in_dim, hid, nh, bufa, bufb, raw);
        }
#pragma unroll
        for (int k = 0; k < 3; ++k)
            A.out_rgb[3ull * p + k] = __fmaf_rn(T, hy_sigmoid(raw[k]), A.out_rgb[3ull * p + k]);
    }
}

template <int CL, int CHID, int CNH, int DT>
hyrf_status launch_one(const BgArgs& A, size_t smem, int grid, cudaStream_t st) {
    auto k = background_kernel<CL, CHID, CNH, DT>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(background)");
    k<<<grid, kBgThreads, smem, st>>>(A);
    return HYRF_OK;
}

}  // namespace

hyrf_status hy_launch_background(hyrf_scene* s, const FrameDev& f, float* out_rgb, uint32_t* launches) {
    BgArgs A;
    A.grid = s->bg_grid; A.mlp = s->bg_mlp; A.f = f;
    A.pe_octaves = s->desc.dir_pe_octaves;
    A.finalT = s->finalT; A.out_rgb = out_rgb;
    A.bg_list = s->bg_list; A.counters = s->counters;
    const hyrf_mlp_desc& m = s->desc.bg_mlp;
    const size_t smem = ((size_t)m.in_dim * m.hidden + (size_t)(m.n_hidden - 1) * m.hidden * m.hidden + (size_t)m.hidden * 3) * sizeof(float);
    const int P = f.W * f.H;
    const int need = (P + kBgThreads - 1) / kBgThreads;
    const int grid = need < s->sm_count * 8 ? need : s->sm_count * 8;
    const uint32_t L = s->desc.bg_grid.levels;
    const bool std_in = m.in_dim == 2 * L + 24 && s->desc.dir_pe_octaves == 4 && m.n_hidden == 1;
    hyrf_status st;
    const int dt = s->u8 ? HY_DT_U8 : (s->fp16 ? HY_DT_F16 : HY_DT_F32);
#define HY_DISPATCH(CL, CH, CN)                                                                   \
    (dt == HY_DT_U8 ? launch_one<CL, CH, CN, HY_DT_U8>(A, smem, grid, s->stream)                     \
                    : dt == HY_DT_F16 ? launch_one<CL, CH, CN, HY_DT_F16>(A, smem, grid, s->stream)  \
                                      : launch_one<CL, CH, CN, HY_DT_F32>(A, smem, grid, s->stream))
    if (std_in && L == 8 && m.hidden == 64)
        st = HY_DISPATCH(8, 64, 1);
    else if (std_in && L == 4 && m.hidden == 32 && dt != HY_DT_U8)
        st = s->fp16 ? launch_one<4, 32, 1, HY_DT_F16>(A, smem, grid, s->stream) : launch_one<4, 32, 1, HY_DT_F32>(A, smem, grid, s->stream);
    else
        st = HY_DISPATCH(0, 0, 0);
#undef HY_DISPATCH
    if (st == HYRF_OK) ++*launches;
    return st;
}
