// field.cu — S2 + S3 + S4a fused, CUDA-core fp32 path: per visible Gaussian
//   contraction (Eq. 2) -> geometry + appearance grid encodes (Eq. 3) -> direction PE (Eq. 5) ->
//   decoders Phi_geo, Phi_c (Eq. 4, 6) -> aggregation with the explicit parameters (Eq. 7) -> EWA projection,
//   radius and tile rectangle (3DGS rasterizer).
// Nothing between the gathers and the projected record touches HBM. The MLPs run as explicit fp32 fma chains in
// the order of DESIGN.md §2 D5, so every geometry decision (radius, rectangle) is bit-reproducible; this is the
// path for fp32 parameters (configs 1–2) and the "exact" mode of fp16 ones. The tensor-core path is field_mma.cu.
#include "mlp.cuh"
#include "scene.h"

namespace {

constexpr int kFieldThreads = 128;

struct FieldArgs {
    GridDev geo, app;
    MlpDev geo_mlp, app_mlp;
    FrameDev f;
    const float* pos;
    const float* rgb;
    const float* scale;
    const float* opac;
    uint32_t N;
    uint32_t pe_octaves;
    const uint32_t* vis_idx;
    const FrameCounters* counters;
    float4* rec;
    uint32_t* depth_key;
    uint4* rect;
    uint32_t* tiles;
    float* dbg_raw;
    float* dbg_attrs;
};

// D7 + D8 for one Gaussian. raw = (alpha_n, s_n[3], r_n[4], c_n[3]).
__device__ __forceinline__ void aggregate_project(const FieldArgs& A, uint32_t j, uint32_t gid, float px, float py,
                                                  float pz, const float* raw) {
    const FrameDev& f = A.f;
    const float s_e = __ldg(A.scale + gid), a_e = __ldg(A.opac + gid);
    const float c_e0 = __ldg(A.rgb + gid), c_e1 = __ldg(A.rgb + A.N + gid), c_e2 = __ldg(A.rgb + 2ull * A.N + gid);
    // Eq. 7
    const float s0 = hy_sigmoid(__fadd_rn(raw[1], s_e));
    const float s1 = hy_sigmoid(__fadd_rn(raw[2], s_e));
    const float s2 = hy_sigmoid(__fadd_rn(raw[3], s_e));
    const float m = __fsqrt_rn(__fmaf_rn(raw[7], raw[7], __fmaf_rn(raw[6], raw[6], __fmaf_rn(raw[5], raw[5], __fmul_rn(raw[4], raw[4])))));
    const float den = fmaxf(m, 1e-12f);
    const float w = __fdiv_rn(raw[4], den), x = __fdiv_rn(raw[5], den), y = __fdiv_rn(raw[6], den), z = __fdiv_rn(raw[7], den);
    const float alpha = hy_sigmoid(__fadd_rn(raw[0], a_e));
    const float c0 = hy_sigmoid(__fadd_rn(raw[8], c_e0));
    const float c1 = hy_sigmoid(__fadd_rn(raw[9], c_e1));
    const float c2 = hy_sigmoid(__fadd_rn(raw[10], c_e2));
    if (A.dbg_raw) {
        for (int k = 0; k < 11; ++k) A.dbg_raw[11ull * j + k] = raw[k];
    }
    if (A.dbg_attrs) {
        float* o = A.dbg_attrs + 11ull * j;
        o[0] = s0; o[1] = s1; o[2] = s2; o[3] = w; o[4] = x; o[5] = y; o[6] = z; o[7] = alpha; o[8] = c0; o[9] = c1; o[10] = c2;
    }
    // D8
    float M[9];
    M[0] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(y, y, __fmul_rn(z, z))));
    M[1] = __fmul_rn(2.0f, __fmaf_rn(x, y, -__fmul_rn(w, z)));
    M[2] = __fmul_rn(2.0f, __fmaf_rn(x, z, __fmul_rn(w, y)));
    M[3] = __fmul_rn(2.0f, __fmaf_rn(x, y, __fmul_rn(w, z)));
    M[4] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(x, x, __fmul_rn(z, z))));
    M[5] = __fmul_rn(2.0f, __fmaf_rn(y, z, -__fmul_rn(w, x)));
    M[6] = __fmul_rn(2.0f, __fmaf_rn(x, z, -__fmul_rn(w, y)));
    M[7] = __fmul_rn(2.0f, __fmaf_rn(y, z, __fmul_rn(w, x)));
    M[8] = __fsub_rn(1.0f, __fmul_rn(2.0f, __fmaf_rn(x, x, __fmul_rn(y, y))));
    float L[9];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        L[3 * i + 0] = __fmul_rn(M[3 * i + 0], s0);
        L[3 * i + 1] = __fmul_rn(M[3 * i + 1], s1);
        L[3 * i + 2] = __fmul_rn(M[3 * i + 2], s2);
    }
    float S[9];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 3; ++k)
            S[3 * i + k] = __fmaf_rn(L[3 * i + 2], L[3 * k + 2], __fmaf_rn(L[3 * i + 1], L[3 * k + 1], __fmul_rn(L[3 * i], L[3 * k])));
    float X, Y, Z;
    hy_to_camera(f, px, py, pz, X, Y, Z);
    const float iz = __fdiv_rn(1.0f, Z), xn = __fmul_rn(X, iz), yn = __fmul_rn(Y, iz);
    const float J00 = __fmul_rn(f.fx, iz), J02 = __fmul_rn(-__fmul_rn(f.fx, xn), iz);
    const float J11 = __fmul_rn(f.fy, iz), J12 = __fmul_rn(-__fmul_rn(f.fy, yn), iz);
    float T0[3], T1[3], U0[3], U1[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        T0[k] = __fmaf_rn(J02, f.R[6 + k], __fmul_rn(J00, f.R[k]));
        T1[k] = __fmaf_rn(J12, f.R[6 + k], __fmul_rn(J11, f.R[3 + k]));
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        U0[k] = __fmaf_rn(T0[2], S[6 + k], __fmaf_rn(T0[1], S[3 + k], __fmul_rn(T0[0], S[k])));
        U1[k] = __fmaf_rn(T1[2], S[6 + k], __fmaf_rn(T1[1], S[3 + k], __fmul_rn(T1[0], S[k])));
    }
    const float a = __fadd_rn(__fmaf_rn(U0[2], T0[2], __fmaf_rn(U0[1], T0[1], __fmul_rn(U0[0], T0[0]))), 0.3f);
    const float b = __fmaf_rn(U0[2], T1[2], __fmaf_rn(U0[1], T1[1], __fmul_rn(U0[0], T1[0])));
    const float c = __fadd_rn(__fmaf_rn(U1[2], T1[2], __fmaf_rn(U1[1], T1[1], __fmul_rn(U1[0], T1[0]))), 0.3f);
    const float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
    const float u = __fmaf_rn(f.fx, xn, f.cx), v = __fmaf_rn(f.fy, yn, f.cy);
    float cA = 0.0f, cB = 0.0f, cC = 0.0f, radius = 0.0f;
    uint4 rc = make_uint4(0, 0, 0, 0);
    uint32_t nt = 0;
    if (det != 0.0f && isfinite(det)) {
        const float di = __fdiv_rn(1.0f, det);
        cA = __fmul_rn(c, di);
        cB = __fmul_rn(-b, di);
        cC = __fmul_rn(a, di);
        const float mid = __fmul_rn(0.5f, __fadd_rn(a, c));
        const float lam = __fadd_rn(mid, __fsqrt_rn(fmaxf(0.1f, __fmaf_rn(mid, mid, -det))));
        radius = ceilf(__fmul_rn(3.0f, __fsqrt_rn(lam)));
        const float gx = (float)f.gx, gy = (float)f.gy;
        const float fx0 = fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(u, radius), 0.0625f)), 0.0f), gx);
        const float fx1 = fminf(fmaxf(floorf(__fmul_rn(__fadd_rn(__fadd_rn(u, radius), 15.0f), 0.0625f)), 0.0f), gx);
        const float fy0 = fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(v, radius), 0.0625f)), 0.0f), gy);
        const float fy1 = fminf(fmaxf(floorf(__fmul_rn(__fadd_rn(__fadd_rn(v, radius), 15.0f), 0.0625f)), 0.0f), gy);
        if (fx0 == fx0 && fx1 == fx1 && fy0 == fy0 && fy1 == fy1) {
            rc = make_uint4((uint32_t)fx0, (uint32_t)fx1, (uint32_t)fy0, (uint32_t)fy1);
            if (rc.y > rc.x && rc.w > rc.z) nt = (rc.y - rc.x) * (rc.w - rc.z);
            else rc = make_uint4(rc.x, rc.y, rc.z, rc.w);
        }
    }
    A.rec[3ull * j + 0] = make_float4(u, v, cA, cB);
    A.rec[3ull * j + 1] = make_float4(cC, alpha, c0, c1);
    A.rec[3ull * j + 2] = make_float4(c2, Z, radius, __uint_as_float(nt));
    A.depth_key[j] = __float_as_uint(Z);
    A.rect[j] = rc;
    A.tiles[j] = nt;
}

// CL: levels of both grids (0 = run-time), CHID / CNH: hidden width / count (0 = run-time).
template <int CL, int CHID, int CNH, bool FP16>
__global__ void __launch_bounds__(kFieldThreads)
field_fma_kernel(const FieldArgs A) {
    extern __shared__ float smem_w[];
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
    for (uint32_t j = blockIdx.x * kFieldThreads + threadIdx.x; j < V; j += gridDim.x * kFieldThreads) {
        const uint32_t gid = A.vis_idx[j];
        const float px = __ldg(A.pos + gid), py = __ldg(A.pos + A.N + gid), pz = __ldg(A.pos + 2ull * A.N + gid);
        float x[3];
        hy_contract(A.f, px, py, pz, x);
        float bufa[MAXD], bufb[MAXD], raw[11];
        // geometry field (Eq. 3, 4)
#pragma unroll
        for (int l = 0; l < Lg; ++l) {
            float f0, f1;
            hy_grid_level<FP16>(A.geo, l, x, f0, f1);
            bufa[2 * l] = FP16 ? hy_round_half(f0) : f0;
            bufa[2 * l + 1] = FP16 ? hy_round_half(f1) : f1;
        }
        if (CL > 0) {
            mlp_eval<2 * CL, CHID, CNH, 8, FP16>(wg, 0, 0, 0, bufa, bufb, raw);
        } else {
            for (int k = 2 * Lg; k < geo_in; ++k) bufa[k] = 0.0f;
            mlp_eval<0, 0, 0, 8, FP16>(wg, geo_in, hid_g, nh_g, bufa, bufb, raw);
        }
        // appearance field (Eq. 3, 5, 6)
#pragma unroll
        for (int l = 0; l < La; ++l) {
            float f0, f1;
            hy_grid_level<FP16>(A.app, l, x, f0, f1);
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
        if (CL > 0) {
            mlp_eval<2 * CL + 24, CHID, CNH, 3, FP16>(wa, 0, 0, 0, bufa, bufb, raw + 8);
        } else {
            for (int k = 2 * La + 6 * (int)A.pe_octaves; k < app_in; ++k) bufa[k] = 0.0f;
            mlp_eval<0, 0, 0, 3, FP16>(wa, app_in, hid_a, nh_a, bufa, bufb, raw + 8);
        }
        aggregate_project(A, j, gid, px, py, pz, raw);
    }
}

template <int CL, int CHID, int CNH, bool FP16>
hyrf_status launch_one(const FieldArgs& A, size_t smem, int grid, cudaStream_t st) {
    auto k = field_fma_kernel<CL, CHID, CNH, FP16>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(field)");
    k<<<grid, kFieldThreads, smem, st>>>(A);
    return HYRF_OK;
}

}  // namespace

hyrf_status hy_launch_field_fma(hyrf_scene* s, const FrameDev& f, uint32_t* launches) {
    FieldArgs A;
    A.geo = s->geo_grid; A.app = s->app_grid;
    A.geo_mlp = s->geo_mlp; A.app_mlp = s->app_mlp;
    A.f = f;
    A.pos = s->pos; A.rgb = s->rgb; A.scale = s->scale; A.opac = s->opac;
    A.N = s->N; A.pe_octaves = s->desc.dir_pe_octaves;
    A.vis_idx = s->vis_idx; A.counters = s->counters;
    A.rec = s->rec; A.depth_key = s->depth_key; A.rect = s->rect; A.tiles = s->tiles;
    A.dbg_raw = ((s->debug_mask >> HYRF_DBG_STAGE2_RAW) & 1u) ? s->dbg_raw : nullptr;
    A.dbg_attrs = ((s->debug_mask >> HYRF_DBG_STAGE3_ATTRS) & 1u) ? s->dbg_attrs : nullptr;
    const hyrf_mlp_desc &g = s->desc.geo_mlp, &a = s->desc.app_mlp;
    const size_t nw_geo = (size_t)g.in_dim * g.hidden + (size_t)(g.n_hidden - 1) * g.hidden * g.hidden + (size_t)g.hidden * 8;
    const size_t nw_app = (size_t)a.in_dim * a.hidden + (size_t)(a.n_hidden - 1) * a.hidden * a.hidden + (size_t)a.hidden * 3;
    const size_t smem = (nw_geo + nw_app) * sizeof(float);
    const int need = (int)((s->N + kFieldThreads - 1) / kFieldThreads);
    const int grid = need < 148 * 3 ? need : 148 * 3;
    const uint32_t L = s->desc.geo_grid.levels;
    const bool same = s->desc.app_grid.levels == L && g.hidden == a.hidden && g.n_hidden == a.n_hidden &&
                      g.in_dim == 2 * L && a.in_dim == 2 * L + 24 && s->desc.dir_pe_octaves == 4;
    hyrf_status st;
    if (same && L == 16 && g.hidden == 64 && g.n_hidden == 2) {
        st = s->fp16 ? launch_one<16, 64, 2, true>(A, smem, grid, s->stream)
                     : launch_one<16, 64, 2, false>(A, smem, grid, s->stream);
    } else if (same && L == 8 && g.hidden == 32 && g.n_hidden == 1) {
        st = s->fp16 ? launch_one<8, 32, 1, true>(A, smem, grid, s->stream)
                     : launch_one<8, 32, 1, false>(A, smem, grid, s->stream);
    } else {
        st = s->fp16 ? launch_one<0, 0, 0, true>(A, smem, grid, s->stream)
                     : launch_one<0, 0, 0, false>(A, smem, grid, s->stream);
    }
    if (st == HYRF_OK) ++*launches;
    return st;
}
