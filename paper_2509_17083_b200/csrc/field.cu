// field.cu — S2 + S3 + S4a fused, CUDA-core fp32 path: per visible Gaussian
//   contraction (Eq. 2) -> geometry + appearance grid encodes (Eq. 3) -> direction PE (Eq. 5) ->
//   decoders Phi_geo, Phi_c (Eq. 4, 6) -> aggregation with the explicit parameters (Eq. 7) -> EWA projection,
//   radius and tile rectangle (3DGS rasterizer).
// Nothing between the gathers and the projected record touches HBM. The MLPs run as explicit fp32 fma chains in
// the order of DESIGN.md §2 D5, so every geometry decision (radius, rectangle) is bit-reproducible; this is the
// path for fp32 parameters (configs 1–2) and the "exact" mode of fp16 ones. The tensor-core path is field_mma.cu.
#include "field_common.cuh"
#include "mlp.cuh"
#include "scene.h"

namespace {

constexpr int kFieldThreads = 128;

// CL: levels of both grids (0 = run-time), CHID / CNH: hidden width / count (0 = run-time).
template <int CL, int CHID, int CNH, int DT>   // DT: HY_DT_F32 / HY_DT_F16 / HY_DT_U8 (8-bit tables, fp16 decoders)
__global__ void __launch_bounds__(kFieldThreads)
field_fma_kernel(const FieldArgs A) {
    extern __shared__ __align__(16) float smem_w[];
    constexpr bool FP16 = DT != HY_DT_F32;
    const int Lg = CL > 0 ? CL : (int)A.geo.levels;
    const int La = CL > 0 ? CL : (int)A.app.levels;
    const int geo_in = (int)A.geo_mlp.in_dim, app_in = (int)A.app_mlp.in_dim;
    const int hid_g = (int)A.geo_mlp.hidden, hid_a = (int)A.app_mlp.hidden;
    const int nh_g = (int)A.geo_mlp.n_hidden, nh_a = (int)A.app_mlp.n_hidden;
    const int nw_geo = geo_in * hid_g + (nh_g - 1) * hid_g * hid_g + hid_g * 8;
    const int nw_app = app_in * hid_a + (nh_a - 1) * hid_a * hid_a + hid_a * 3;
    float* wg = smem_w;
    float* wa = smem_w + nw_geo;
    if (FP16) {
        const __half* g = reinterpret_cast<const __half*>(A.geo_mlp.w);
        const __half* a = reinterpret_cast<const __half*>(A.app_mlp.w);
        for (int i = threadIdx.x; i < nw_geo; i += kFieldThreads) wg[i] = __half2float(g[i]);
        for (int i = threadIdx.x; i < nw_app; i += kFieldThreads) wa[i] = __half2float(a[i]);
    } else {
        const float* g = reinterpret_cast<const float*>(A.geo_mlp.w);
        const float* a = reinterpret_cast<const float*>(A.app_mlp.w);
        for (int i = threadIdx.x; i < nw_geo; i += kFieldThreads) wg[i] = g[i];
        for (int i = threadIdx.x; i < nw_app; i += kFieldThreads) wa[i] = a[i];
    }
    __syncthreads();
    const uint32_t V = A.counters->V;
    constexpr int MAXD = CL > 0 ? (2 * CL + 24 > CHID ? 2 * CL + 24 : CHID) : HYRF_MAX_WIDTH;
    for (uint32_t wi = blockIdx.x * kFieldThreads + threadIdx.x; wi < V; wi += gridDim.x * kFieldThreads) {
        const Explicit ex = fetch_visible(A, wi);
        const float px = ex.px, py = ex.py, pz = ex.pz;
        float x[3];
        hy_contract(A.f, px, py, pz, x);
        float bufa[MAXD], bufb[MAXD], raw[11];
        if (A.f.ablation & HYRF_ABL_NO_NEURAL) {   // explicit-only ablation: the decoders contribute nothing
#pragma unroll
            for (int k = 0; k < 11; ++k) raw[k] = 0.0f;
            aggregate_project<false>(A, ex, raw);
            continue;
        }
        // geometry field (Eq. 3, 4)
#pragma unroll
        for (int l = 0; l < Lg; ++l) {
            float f0, f1;
            hy_grid_level<DT>(A.geo, l, x, f0, f1);
            bufa[2 * l] = FP16 ? hy_round_half(f0) : f0;
            bufa[2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
        }
        if constexpr (CL > 0 && CNH == 2) {   // two hidden layers: layer by layer as loops (mlp.cuh mlp_dense_ct)
            mlp_dense_ct<FP16, 2 * CL, true, CHID>(wg, bufa, bufb);
            mlp_dense_ct<FP16, CHID, true, CHID>(wg + CHID * 2 * CL, bufb, bufa);
            mlp_dense_ct<FP16, CHID, false, 8>(wg + CHID * 2 * CL + CHID * CHID, bufa, raw);
        } else if (CL > 0) {
            mlp_eval<2 * CL, CHID, CNH, 8, FP16>(wg, 0, 0, 0, bufa, bufb, raw);
        } else {
            for (int k = 2 * Lg; k < geo_in; ++k) bufa[k] = 0.0f;
            mlp_eval<0, 0, 0, 8, FP16>(wg, geo_in, hid_g, nh_g, bufa, bufb, raw);
        }
        // appearance field (Eq. 3, 5, 6)
#pragma unroll
        for (int l = 0; l < La; ++l) {
            float f0, f1;
            hy_grid_level<DT>(A.app, l, x, f0, f1);
            bufa[2 * l] = FP16 ? hy_round_half(f0) : f0;
            bufa[2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
        }
        {
            const float dx = __fsub_rn(px, A.f.o[0]), dy = __fsub_rn(py, A.f.o[1]), dz = __fsub_rn(pz, A.f.o[2]);
            const float n = __fsqrt_rn(__fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))));
            float d[3] = {__fdiv_rn(dx, n), __fdiv_rn(dy, n), __fdiv_rn(dz, n)};
            if (CL > 0) hy_dir_pe<FP16>(d, 4, bufa + 2 * CL);
            else hy_dir_pe<FP16>(d, (int)A.pe_octaves, bufa + 2 * La);
        }
        if constexpr (CL > 0 && CNH == 2) {
            mlp_dense_ct<FP16, 2 * CL + 24, true, CHID>(wa, bufa, bufb);
            mlp_dense_ct<FP16, CHID, true, CHID>(wa + CHID * (2 * CL + 24), bufb, bufa);
            mlp_dense_ct<FP16, CHID, false, 3>(wa + CHID * (2 * CL + 24) + CHID * CHID, bufa, raw + 8);
        } else if (CL > 0) {
            mlp_eval<2 * CL + 24, CHID, CNH, 3, FP16>(wa, 0, 0, 0, bufa, bufb, raw + 8);
        } else {
            for (int k = 2 * La + 6 * (int)A.pe_octaves; k < app_in; ++k) bufa[k] = 0.0f;
            mlp_eval<0, 0, 0, 3, FP16>(wa, app_in, hid_a, nh_a, bufa, bufb, raw + 8);
        }
        aggregate_project<false>(A, ex, raw);
    }
}

template <int CL, int CHID, int CNH, int DT>
hyrf_status launch_one(const FieldArgs& A, size_t smem, int grid, cudaStream_t st) {
    auto k = field_fma_kernel<CL, CHID, CNH, DT>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(field)");
    k<<<grid, kFieldThreads, smem, st>>>(A);
    return HYRF_OK;
}

}  // namespace

void hy_fill_field_args(hyrf_scene* s, const FrameDev& f, FieldArgs* out) {
    FieldArgs& A = *out;
    A.geo = s->geo_grid; A.app = s->app_grid;
    A.geo_mlp = s->geo_mlp; A.app_mlp = s->app_mlp;
    A.f = f;
    A.gm = s->gm; A.gm_id = s->gm_id; A.vis_m = s->vis_m; A.id_words = s->id_words; A.word_rank = s->word_rank;
    A.N = s->N; A.pe_octaves = s->desc.dir_pe_octaves;
    A.counters = s->counters;
    A.rec = s->rec; A.rect = s->rect; A.tiles = s->tiles; A.mtiles = s->mtiles;
    A.dbg_raw = ((s->debug_mask >> HYRF_DBG_STAGE2_RAW) & 1u) ? s->dbg_raw : nullptr;
    A.dbg_attrs = ((s->debug_mask >> HYRF_DBG_STAGE3_ATTRS) & 1u) ? s->dbg_attrs : nullptr;
}

hyrf_status hy_launch_field_fma(hyrf_scene* s, const FrameDev& f, uint32_t* launches) {
    FieldArgs A;
    hy_fill_field_args(s, f, &A);
    const hyrf_mlp_desc &g = s->desc.geo_mlp, &a = s->desc.app_mlp;
    const size_t nw_geo = (size_t)g.in_dim * g.hidden + (size_t)(g.n_hidden - 1) * g.hidden * g.hidden + (size_t)g.hidden * 8;
    const size_t nw_app = (size_t)a.in_dim * a.hidden + (size_t)(a.n_hidden - 1) * a.hidden * a.hidden + (size_t)a.hidden * 3;
    const size_t smem = (nw_geo + nw_app) * sizeof(float);
    const int need = (int)((s->N + kFieldThreads - 1) / kFieldThreads);
    const int grid = need < s->sm_count * 3 ? need : s->sm_count * 3;
    const uint32_t L = s->desc.geo_grid.levels;
    const bool same = s->desc.app_grid.levels == L && g.hidden == a.hidden && g.n_hidden == a.n_hidden &&
                      g.in_dim == 2 * L && a.in_dim == 2 * L + 24 && s->desc.dir_pe_octaves == 4;
    hyrf_status st;
    const int dt = s->u8 ? HY_DT_U8 : (s->fp16 ? HY_DT_F16 : HY_DT_F32);
#define HY_DISPATCH(CL, CH, CN)                                                                   \
    (dt == HY_DT_U8 ? launch_one<CL, CH, CN, HY_DT_U8>(A, smem, grid, s->stream)                     \
                    : dt == HY_DT_F16 ? launch_one<CL, CH, CN, HY_DT_F16>(A, smem, grid, s->stream)  \
                                      : launch_one<CL, CH, CN, HY_DT_F32>(A, smem, grid, s->stream))
    if (same && L == 16 && g.hidden == 64 && g.n_hidden == 2) {
        st = HY_DISPATCH(16, 64, 2);
    } else if (same && L == 8 && g.hidden == 32 && g.n_hidden == 1 && dt != HY_DT_U8) {
        st = s->fp16 ? launch_one<8, 32, 1, HY_DT_F16>(A, smem, grid, s->stream)
                     : launch_one<8, 32, 1, HY_DT_F32>(A, smem, grid, s->stream);
    } else {
        st = HY_DISPATCH(0, 0, 0);
    }
#undef HY_DISPATCH
    if (st == HYRF_OK) ++*launches;
    return st;
}
