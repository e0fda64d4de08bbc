// api.cu — the C-ABI of include/hyrf.h: scene creation, parameter upload, the render pass orchestration,
// debug fetches. Host logic only; every step of the path runs in the kernels of the other .cu files.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "scene.h"

static thread_local char g_err[512] = "";

hyrf_status hy_fail(hyrf_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

hyrf_status hy_cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_err, sizeof(g_err), "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), what);
    cudaGetLastError();
    return (e == cudaErrorMemoryAllocation) ? HYRF_ERR_OOM : HYRF_ERR_CUDA;
}

extern "C" const char* hyrf_last_error(void) { return g_err; }

hyrf_status hy_launch_field_fma(hyrf_scene* s, const FrameDev& f, uint32_t* launches);
hyrf_status hy_launch_field_mma(hyrf_scene* s, const FrameDev& f, uint32_t* launches);
hyrf_status hy_launch_field_ws(hyrf_scene* s, const FrameDev& f, uint32_t* launches);
void hy_launch_counters_to_host(const FrameCounters* dev, FrameCounters* pinned_host, cudaStream_t st);
bool hy_field_mma_supported(const hyrf_scene_desc& d);
hyrf_status hy_field_mma_prepare(hyrf_scene* s);
size_t hy_field_mma_packed_bytes();

namespace {

hyrf_status dev_alloc(hyrf_scene* s, void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    if (s->desc.alloc) {
        *p = s->desc.alloc(bytes, s->desc.user);
        if (!*p) return hy_fail(HYRF_ERR_OOM, "user allocator returned NULL for %zu bytes", bytes);
        return HYRF_OK;
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) { *p = nullptr; return hy_cuda_fail(e, "cudaMalloc"); }
    return HYRF_OK;
}

void dev_free(hyrf_scene* s, void* p) {
    if (!p) return;
    if (s->desc.release) s->desc.release(p, s->desc.user);
    else if (!s->desc.alloc) cudaFree(p);
}

template <typename T>
hyrf_status dev_alloc_t(hyrf_scene* s, T** p, size_t count) {
    return dev_alloc(s, reinterpret_cast<void**>(p), count * sizeof(T));
}

hyrf_status check_grid(const hyrf_grid_desc& g, const char* name) {
    if (g.levels == 0 || g.levels > HYRF_MAX_LEVELS)
        return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: levels %u outside [1, %u]", name, g.levels, HYRF_MAX_LEVELS);
    if (g.feats != 2) return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: feats must be 2 (got %u)", name, g.feats);
    if (g.log2_table == 0 || g.log2_table > 24)
        return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: log2_table %u outside [1, 24]", name, g.log2_table);
    if (!g.level_res) return hy_fail(HYRF_ERR_INVALID_ARG, "%s: level_res is NULL", name);
    for (uint32_t l = 0; l < g.levels; ++l)
        if (g.level_res[l] == 0 || g.level_res[l] > 65535u)
            return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: level_res[%u] = %u outside [1, 65535]", name, l, g.level_res[l]);
    return HYRF_OK;
}

hyrf_status check_mlp(const hyrf_mlp_desc& m, uint32_t min_in, uint32_t out, const char* name) {
    if (m.out_dim != out) return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: out_dim must be %u (got %u)", name, out, m.out_dim);
    if (m.n_hidden == 0 || m.n_hidden > 4) return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: n_hidden %u outside [1, 4]", name, m.n_hidden);
    if (m.hidden == 0 || m.hidden > HYRF_MAX_WIDTH) return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: hidden %u outside [1, %u]", name, m.hidden, HYRF_MAX_WIDTH);
    if (m.in_dim < min_in || m.in_dim > HYRF_MAX_WIDTH)
        return hy_fail(HYRF_ERR_UNSUPPORTED, "%s: in_dim %u outside [%u, %u]", name, m.in_dim, min_in, HYRF_MAX_WIDTH);
    return HYRF_OK;
}

size_t mlp_weights(const hyrf_mlp_desc& m) {
    return (size_t)m.in_dim * m.hidden + (size_t)(m.n_hidden - 1) * m.hidden * m.hidden + (size_t)m.hidden * m.out_dim;
}

// DESIGN.md §2 D3 layout: dense iff (N+1)^3 <= T; dense size rounded up to a multiple of 8.
size_t build_grid(const hyrf_grid_desc& d, GridDev* g) {
    const uint64_t T = 1ull << d.log2_table;
    g->levels = d.levels;
    g->table_mask = (uint32_t)(T - 1);
    g->dense_mask = 0;
    uint64_t off = 0;
    for (uint32_t l = 0; l < d.levels; ++l) {
        const uint64_t n1 = (uint64_t)d.level_res[l] + 1;
        const uint64_t dense = n1 * n1 * n1;
        g->res[l] = d.level_res[l];
        g->offset[l] = (uint32_t)off;
        if (dense <= T) {
            g->dense_mask |= 1u << l;
            off += (dense + 7) / 8 * 8;
        } else {
            off += T;
        }
    }
    return (size_t)off;
}

void free_entries(hyrf_scene* s) {
    for (int i = 0; i < 2; ++i) {
        dev_free(s, s->ent_key[i]); s->ent_key[i] = nullptr;
        dev_free(s, s->ent_val[i]); s->ent_val[i] = nullptr;
    }
    dev_free(s, s->hist); s->hist = nullptr;
    dev_free(s, s->bin_ws); s->bin_ws = nullptr;
    s->d_capacity = 0;
}

// Scratch that depends on the number of tile entries D (keys/values ping-pong + radix histograms).
hyrf_status ensure_entries(hyrf_scene* s, size_t need) {
    if (need <= s->d_capacity) return HYRF_OK;
    if (need >= 0xFFFFFFFFull) return hy_fail(HYRF_ERR_OOM, "tile-entry count %zu does not fit 32-bit offsets", need);
    cudaStreamSynchronize(s->stream);
    free_entries(s);
    size_t cap = need + need / 4 + 4096;
    if (cap > 0xFFFFFFF0ull) cap = 0xFFFFFFF0ull;
    hyrf_status st;
    for (int i = 0; i < 2; ++i) {
        if ((st = dev_alloc_t(s, &s->ent_key[i], cap)) != HYRF_OK) { free_entries(s); return st; }
        if ((st = dev_alloc_t(s, &s->ent_val[i], cap)) != HYRF_OK) { free_entries(s); return st; }
    }
    const size_t cap_sort = cap > s->N ? cap : s->N;
    s->hist_elems = hy_radix_hist_elems(cap_sort);
    if ((st = dev_alloc_t(s, &s->hist, s->hist_elems)) != HYRF_OK) { free_entries(s); return st; }
    {   // ordered-binning workspace scales with the list capacity (bin_ordered.cu); look-back words start cleared
        const size_t tiles_max = (size_t)((s->desc.max_width + HY_TILE - 1) / HY_TILE) * ((s->desc.max_height + HY_TILE - 1) / HY_TILE);
        const size_t elems = hy_bin_ordered_ws_elems(s->N, cap, (uint32_t)tiles_max);
        if ((st = dev_alloc_t(s, &s->bin_ws, elems)) != HYRF_OK) { free_entries(s); return st; }
        if (cudaMemsetAsync(s->bin_ws, 0, elems * sizeof(uint32_t), s->stream) != cudaSuccess) { free_entries(s); return hy_cuda_fail(cudaGetLastError(), "cudaMemsetAsync(bin_ws)"); }
    }
    const size_t need_scan = hy_scan_scratch_elems(s->hist_elems) + hy_scan_scratch_elems(s->N) + 64;
    if (need_scan > s->scan_scratch_elems) {
        dev_free(s, s->scan_scratch);
        s->scan_scratch = nullptr;
        s->scan_scratch_elems = 0;
        if ((st = dev_alloc_t(s, &s->scan_scratch, need_scan)) != HYRF_OK) { free_entries(s); return st; }
        s->scan_scratch_elems = need_scan;
    }
    s->d_capacity = cap;
    return HYRF_OK;
}

// the scene's S1 / depth-sort members become aliases of set k
void hy_select_pre_set(hyrf_scene* s, int k) {
    hyrf_scene::PreSet& P = s->pre[k];
    s->pre_cur = k;
    s->flag_words = P.flag_words; s->id_words = P.id_words; s->word_rank = P.word_rank; s->vis_m = P.vis_m;
    s->block_counts = P.block_counts; s->vis_idx = P.vis_idx;
    s->sort_a_key = P.sort_a_key; s->sort_a_val = P.sort_a_val; s->sort_b_key = P.sort_b_key; s->sort_b_val = P.sort_b_val;
    s->counters = P.counters; s->counters_host = P.counters_host;
}

void destroy(hyrf_scene* s) {
    if (!s) return;
    cudaStreamSynchronize(s->stream);
    void* ptrs[] = {s->pos, s->rgb, s->scale, s->opac, (void*)s->geo_grid.table, (void*)s->app_grid.table,
                    (void*)s->bg_grid.table, (void*)s->geo_mlp.w, (void*)s->app_mlp.w, (void*)s->bg_mlp.w, s->mma_w, s->both_table,
                    s->gm, s->gm_id, s->rec, s->rect, s->tiles, s->mtiles, s->mranges, s->tt_sorted, s->offs,
                    s->scan_scratch, s->ranges, s->list_len, s->tile_queue, s->fg, s->finalT, s->image, s->image2, s->bg_mask, s->bg_list,
                    s->dbg_raw, s->dbg_attrs, s->bwd_gT, s->bwd_grec, s->bwd_ssim};
    for (void* p : ptrs) dev_free(s, p);
    if (s->sort_stream) cudaStreamSynchronize(s->sort_stream);
    for (auto& P : s->pre) {   // (the scene's members of the same names are aliases of one of the two sets)
        void* pp[] = {P.flag_words, P.id_words, P.word_rank, P.vis_m, P.block_counts, P.vis_idx, P.sort_a_key, P.sort_a_val,
                      P.sort_b_key, P.sort_b_val, P.hist, P.scan, P.counters};
        for (void* p : pp) dev_free(s, p);
        if (P.counters_host) cudaFreeHost(P.counters_host);
        if (P.ev_free) cudaEventDestroy(P.ev_free);
    }
    free_entries(s);
    if (s->ev_start) cudaEventDestroy(s->ev_start);
    if (s->ev_frame_done) cudaEventDestroy(s->ev_frame_done);
    if (s->ev_counters) cudaEventDestroy(s->ev_counters);
    if (s->sort_stream) { cudaStreamSynchronize(s->sort_stream); cudaStreamDestroy(s->sort_stream); }
    if (s->ev_culled) cudaEventDestroy(s->ev_culled);
    if (s->ev_sorted) cudaEventDestroy(s->ev_sorted);
    if (s->copy_stream) {
        cudaStreamSynchronize(s->copy_stream);
        for (int k = 0; k < 2; ++k) { cudaEventDestroy(s->ev_rendered[k]); cudaEventDestroy(s->ev_copied[k]); }
        cudaStreamDestroy(s->copy_stream);
    }
    if (s->ev_valid)
        for (auto& e : s->ev) cudaEventDestroy(e);
    delete s;
}

}  // namespace

extern "C" hyrf_status hyrf_create_scene(const hyrf_scene_desc* desc, hyrf_scene** out) {
    if (!desc || !out) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_create_scene: NULL argument");
    *out = nullptr;
    if (desc->n_gaussians == 0) return hy_fail(HYRF_ERR_INVALID_ARG, "n_gaussians must be > 0");
    if (desc->max_width == 0 || desc->max_height == 0 || desc->max_width > 16384 || desc->max_height > 16384)
        return hy_fail(HYRF_ERR_INVALID_ARG, "max_width / max_height outside [1, 16384]");
    for (int a = 0; a < 3; ++a)
        if (!(desc->aabb_max[a] > desc->aabb_min[a]) || !isfinite(desc->aabb_min[a]) || !isfinite(desc->aabb_max[a]))
            return hy_fail(HYRF_ERR_INVALID_ARG, "aabb axis %d is empty or non-finite", a);
    if (desc->param_dtype != HYRF_F32 && desc->param_dtype != HYRF_F16 && desc->param_dtype != HYRF_U8)
        return hy_fail(HYRF_ERR_INVALID_ARG, "unknown param_dtype %d", (int)desc->param_dtype);
    // z_near > 0: the depth key is the bit pattern of Z and the projection divides by Z (DESIGN.md §2 D1, D8, D9);
    // tau_T is a transmittance
    if (!(desc->bg_radius > 0.0f) || !isfinite(desc->bg_radius) || !isfinite(desc->cull_tol) || desc->cull_tol < 0.0f ||
        !isfinite(desc->z_near) || !(desc->z_near > 0.0f) || !(desc->tau_T >= 0.0f) || !(desc->tau_T <= 1.0f))
        return hy_fail(HYRF_ERR_INVALID_ARG, "bg_radius (> 0) / cull_tol (>= 0) / z_near (> 0) / tau_T (in [0, 1]) out of range");
    if ((size_t)desc->n_gaussians > hy_radix_max_items())
        return hy_fail(HYRF_ERR_UNSUPPORTED, "n_gaussians %u exceeds the %zu items the depth sort supports", desc->n_gaussians, hy_radix_max_items());
    if ((desc->alloc == nullptr) != (desc->release == nullptr))
        return hy_fail(HYRF_ERR_INVALID_ARG, "alloc and release must be given together");
    if (desc->dir_pe_octaves == 0 || desc->dir_pe_octaves > 6)
        return hy_fail(HYRF_ERR_UNSUPPORTED, "dir_pe_octaves %u outside [1, 6]", desc->dir_pe_octaves);
    hyrf_status st;
    if ((st = check_grid(desc->geo_grid, "geo_grid")) != HYRF_OK) return st;
    if ((st = check_grid(desc->app_grid, "app_grid")) != HYRF_OK) return st;
    if ((st = check_grid(desc->bg_grid, "bg_grid")) != HYRF_OK) return st;
    const uint32_t pe = 6 * desc->dir_pe_octaves;
    if ((st = check_mlp(desc->geo_mlp, 2 * desc->geo_grid.levels, 8, "geo_mlp")) != HYRF_OK) return st;
    if ((st = check_mlp(desc->app_mlp, 2 * desc->app_grid.levels + pe, 3, "app_mlp")) != HYRF_OK) return st;
    if ((st = check_mlp(desc->bg_mlp, 2 * desc->bg_grid.levels + pe, 3, "bg_mlp")) != HYRF_OK) return st;
    if (desc->mlp_path != HYRF_MLP_AUTO && desc->mlp_path != HYRF_MLP_FMA && desc->mlp_path != HYRF_MLP_MMA &&
        desc->mlp_path != HYRF_MLP_HMMA && desc->mlp_path != HYRF_MLP_WS)
        return hy_fail(HYRF_ERR_INVALID_ARG, "unknown mlp_path %d", (int)desc->mlp_path);
    if ((desc->mlp_path == HYRF_MLP_MMA || desc->mlp_path == HYRF_MLP_HMMA || desc->mlp_path == HYRF_MLP_WS) && !hy_field_mma_supported(*desc))
        return hy_fail(HYRF_ERR_UNSUPPORTED, "mlp_path MMA / HMMA / WS needs fp16 parameters, 16-level grids, 32->64->64->8 and 56->64->64->3 decoders");

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return hy_fail(HYRF_ERR_CUDA, "no CUDA device available (%s)", e == cudaSuccess ? "count 0" : cudaGetErrorString(e));
    }
    if (desc->device < 0 || desc->device >= ndev) return hy_fail(HYRF_ERR_INVALID_ARG, "device %d outside [0, %d)", desc->device, ndev);
    if ((e = cudaSetDevice(desc->device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    int sm_count = 0;
    if ((e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, desc->device)) != cudaSuccess || sm_count < 1)
        return hy_cuda_fail(e, "cudaDeviceGetAttribute(MultiProcessorCount)");

    hyrf_scene* s = new (std::nothrow) hyrf_scene();
    if (!s) return hy_fail(HYRF_ERR_OOM, "host allocation failed");
    s->desc = *desc;
    s->sm_count = sm_count;   // persistent grids and the CTA slots left to the depth sort are sized from it
    s->res_geo.assign(desc->geo_grid.level_res, desc->geo_grid.level_res + desc->geo_grid.levels);
    s->res_app.assign(desc->app_grid.level_res, desc->app_grid.level_res + desc->app_grid.levels);
    s->res_bg.assign(desc->bg_grid.level_res, desc->bg_grid.level_res + desc->bg_grid.levels);
    s->desc.geo_grid.level_res = s->res_geo.data();
    s->desc.app_grid.level_res = s->res_app.data();
    s->desc.bg_grid.level_res = s->res_bg.data();
    s->N = desc->n_gaussians;
    s->fp16 = desc->param_dtype != HYRF_F32;
    s->u8 = desc->param_dtype == HYRF_U8;
    s->use_mma = desc->mlp_path != HYRF_MLP_FMA && hy_field_mma_supported(*desc);
    s->warp_mma = s->use_mma && desc->mlp_path == HYRF_MLP_HMMA;   // (needs the interleaved table; else the tcgen05 kernel runs)
    s->geo_entries = build_grid(s->desc.geo_grid, &s->geo_grid);
    s->app_entries = build_grid(s->desc.app_grid, &s->app_grid);
    s->bg_entries = build_grid(s->desc.bg_grid, &s->bg_grid);
    s->geo_mlp = MlpDev{nullptr, desc->geo_mlp.in_dim, desc->geo_mlp.hidden, desc->geo_mlp.n_hidden, 8};
    s->app_mlp = MlpDev{nullptr, desc->app_mlp.in_dim, desc->app_mlp.hidden, desc->app_mlp.n_hidden, 3};
    s->bg_mlp = MlpDev{nullptr, desc->bg_mlp.in_dim, desc->bg_mlp.hidden, desc->bg_mlp.n_hidden, 3};

    const size_t N = s->N;
    const size_t esz = s->fp16 ? 2 : 4;          // decoder weights
    const size_t tsz = s->u8 ? 1 : esz;          // table features
    const size_t P = (size_t)desc->max_width * desc->max_height;
    const size_t tiles = (size_t)((desc->max_width + HY_TILE - 1) / HY_TILE) * ((desc->max_height + HY_TILE - 1) / HY_TILE);
    const size_t cull_blocks = (N + 1023) / 1024;
    void *tg = nullptr, *ta = nullptr, *tb = nullptr, *wg = nullptr, *wa = nullptr, *wb = nullptr;
#define HY_TRY(x) if ((st = (x)) != HYRF_OK) { destroy(s); return st; }
    HY_TRY(dev_alloc_t(s, &s->pos, 3 * N));
    HY_TRY(dev_alloc_t(s, &s->rgb, 3 * N));
    HY_TRY(dev_alloc_t(s, &s->scale, N));
    HY_TRY(dev_alloc_t(s, &s->opac, N));
    HY_TRY(dev_alloc(s, &tg, s->geo_entries * 2 * tsz)); s->geo_grid.table = tg;
    HY_TRY(dev_alloc(s, &ta, s->app_entries * 2 * tsz)); s->app_grid.table = ta;
    HY_TRY(dev_alloc(s, &tb, s->bg_entries * 2 * tsz)); s->bg_grid.table = tb;
    HY_TRY(dev_alloc(s, &wg, mlp_weights(s->desc.geo_mlp) * esz)); s->geo_mlp.w = wg;
    HY_TRY(dev_alloc(s, &wa, mlp_weights(s->desc.app_mlp) * esz)); s->app_mlp.w = wa;
    HY_TRY(dev_alloc(s, &wb, mlp_weights(s->desc.bg_mlp) * esz)); s->bg_mlp.w = wb;
    if (s->use_mma) HY_TRY(dev_alloc(s, &s->mma_w, hy_field_mma_packed_bytes()));
    {   // same grid geometry for both fields (every paper configuration): one interleaved table for the tensor path
        const hyrf_grid_desc &g = s->desc.geo_grid, &a = s->desc.app_grid;
        bool same = g.levels == a.levels && g.log2_table == a.log2_table;
        for (uint32_t l = 0; same && l < g.levels; ++l) same = g.level_res[l] == a.level_res[l];
        if (s->use_mma && same) HY_TRY(dev_alloc(s, &s->both_table, s->geo_entries * 4 * tsz));
        // warp-specialised tcgen05 kernel: what AUTO runs when the two grids share their geometry (needs the interleaved table)
        s->ws_mma = s->use_mma && same && (desc->mlp_path == HYRF_MLP_WS || desc->mlp_path == HYRF_MLP_AUTO);
    }
    HY_TRY(dev_alloc_t(s, &s->gm, 2 * N));
    HY_TRY(dev_alloc_t(s, &s->gm_id, N));
    for (auto& P : s->pre) {
        HY_TRY(dev_alloc_t(s, &P.flag_words, (N + 31) / 32 + 32));
        HY_TRY(dev_alloc_t(s, &P.id_words, (N + 31) / 32 + 32));
        HY_TRY(dev_alloc_t(s, &P.word_rank, (N + 31) / 32 + 32));
        HY_TRY(dev_alloc_t(s, &P.vis_m, N));
        HY_TRY(dev_alloc_t(s, &P.block_counts, 4 * cull_blocks + 8));
        HY_TRY(dev_alloc_t(s, &P.vis_idx, N));
        HY_TRY(dev_alloc_t(s, &P.sort_a_key, N));
        HY_TRY(dev_alloc_t(s, &P.sort_a_val, N));
        HY_TRY(dev_alloc_t(s, &P.sort_b_key, N));
        HY_TRY(dev_alloc_t(s, &P.sort_b_val, N));
        HY_TRY(dev_alloc_t(s, &P.hist, hy_radix_hist_elems(N)));
        HY_TRY(dev_alloc_t(s, &P.scan, 2 * hy_scan_scratch_elems(N) + 64));
        HY_TRY(dev_alloc_t(s, &P.counters, 1));
        if ((e = cudaMallocHost(reinterpret_cast<void**>(&P.counters_host), sizeof(FrameCounters))) != cudaSuccess) {
            destroy(s);
            return hy_cuda_fail(e, "cudaMallocHost");
        }
        if ((e = cudaEventCreateWithFlags(&P.ev_free, cudaEventDisableTiming)) != cudaSuccess) {
            destroy(s);
            return hy_cuda_fail(e, "cudaEventCreate");
        }
    }
    hy_select_pre_set(s, 0);
    HY_TRY(dev_alloc_t(s, &s->rec, 3 * N));
    HY_TRY(dev_alloc_t(s, &s->rect, N));
    HY_TRY(dev_alloc_t(s, &s->tiles, N));
    HY_TRY(dev_alloc_t(s, &s->mtiles, N));
    HY_TRY(dev_alloc_t(s, &s->tt_sorted, N));
    HY_TRY(dev_alloc_t(s, &s->offs, N));
    HY_TRY(dev_alloc_t(s, &s->ranges, tiles));
    HY_TRY(dev_alloc_t(s, &s->mranges, tiles));
    HY_TRY(dev_alloc_t(s, &s->list_len, tiles));
    HY_TRY(dev_alloc_t(s, &s->tile_queue, tiles));
    HY_TRY(dev_alloc_t(s, &s->finalT, P));
    HY_TRY(dev_alloc_t(s, &s->bg_list, P));
    if ((e = cudaEventCreateWithFlags(&s->ev_counters, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&s->ev_start, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&s->ev_frame_done, cudaEventDisableTiming)) != cudaSuccess) {
        destroy(s);
        return hy_cuda_fail(e, "cudaEventCreate");
    }
    // S1 and the depth sort are short, latency-bound kernels that must slip in beside the field kernel (and, in a pipelined
    // stream of frames, beside the previous frame's rasterizer): their stream gets the highest priority, so the block
    // scheduler hands freed SM slots to their CTAs first
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    if ((e = cudaStreamCreateWithPriority(&s->sort_stream, cudaStreamNonBlocking, prio_hi)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&s->ev_culled, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&s->ev_sorted, cudaEventDisableTiming)) != cudaSuccess) {
        destroy(s);
        return hy_cuda_fail(e, "cudaStreamCreate / cudaEventCreate (sort)");
    }
    HY_TRY(ensure_entries(s, 4 * N + 65536));   // initial guess (macro-tile entries); grows on demand (hyrf_render)
#undef HY_TRY
    *out = s;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_stream(hyrf_scene* s, void* cuda_stream) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_stream: NULL scene");
    if (s->stream == reinterpret_cast<cudaStream_t>(cuda_stream)) return HYRF_OK;   // (cheap to call before every frame)
    cudaStreamSynchronize(s->stream);   // what is enqueued on the old stream reads and writes the scene's scratch
    s->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_upload_params(hyrf_scene* s, const hyrf_params* p) {
    if (!s || !p) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_params: NULL argument");
    if (!p->geo_table || !p->app_table || !p->bg_table || !p->geo_w || !p->app_w || !p->bg_w)
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_params: NULL parameter pointer");
    // the explicit part may be left out as a whole (it then comes through hyrf_upload_explicit_rvq), not in part
    const bool no_explicit = !p->pos && !p->rgb_logit && !p->scale_logit && !p->opacity_logit;
    if (!no_explicit && (!p->pos || !p->rgb_logit || !p->scale_logit || !p->opacity_logit))
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_params: explicit parameters must be all given or all NULL");
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    const cudaMemcpyKind kind = p->host_ptrs ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    const size_t N = s->N, esz = s->fp16 ? 2 : 4, tsz = s->u8 ? 1 : esz;
    if (s->u8) {   // (min, step) per level and feature travel with the kernel arguments
        if (!p->geo_q || !p->app_q || !p->bg_q) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_params: HYRF_U8 needs geo_q, app_q, bg_q");
        struct { GridDev* g; const float* q; } qs[3] = {{&s->geo_grid, p->geo_q}, {&s->app_grid, p->app_q}, {&s->bg_grid, p->bg_q}};
        for (auto& x : qs) {
            float host[HY_MAX_LEVELS * 4];
            const size_t bytes = (size_t)x.g->levels * 4 * sizeof(float);
            if (p->host_ptrs) memcpy(host, x.q, bytes);
            else if ((e = cudaMemcpy(host, x.q, bytes, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(q)");
            for (uint32_t l = 0; l < x.g->levels; ++l)
                for (int f = 0; f < 2; ++f) {
                    if (!isfinite(host[(l * 2 + f) * 2]) || !isfinite(host[(l * 2 + f) * 2 + 1])) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_params: non-finite quantisation parameter");
                    x.g->q[l][f] = make_float2(host[(l * 2 + f) * 2], host[(l * 2 + f) * 2 + 1]);
                }
        }
    }
    struct { void* dst; const void* src; size_t bytes; } copies[] = {
        {s->pos, p->pos, 3 * N * 4}, {s->rgb, p->rgb_logit, 3 * N * 4}, {s->scale, p->scale_logit, N * 4},
        {s->opac, p->opacity_logit, N * 4},
        {(void*)s->geo_grid.table, p->geo_table, s->geo_entries * 2 * tsz},
        {(void*)s->app_grid.table, p->app_table, s->app_entries * 2 * tsz},
        {(void*)s->bg_grid.table, p->bg_table, s->bg_entries * 2 * tsz},
        {(void*)s->geo_mlp.w, p->geo_w, mlp_weights(s->desc.geo_mlp) * esz},
        {(void*)s->app_mlp.w, p->app_w, mlp_weights(s->desc.app_mlp) * esz},
        {(void*)s->bg_mlp.w, p->bg_w, mlp_weights(s->desc.bg_mlp) * esz}};
    for (auto& c : copies)
        if (c.src && (e = cudaMemcpyAsync(c.dst, c.src, c.bytes, kind, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyAsync(params)");
    if (s->use_mma) {
        hyrf_status st = hy_field_mma_prepare(s);
        if (st != HYRF_OK) return st;
    }
    if (!no_explicit) {
        hyrf_status st = hy_prepare_morton(s);
        if (st != HYRF_OK) return st;
    }
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(upload)");
    s->fields_ready = true;
    if (!no_explicit) s->explicit_ready = true;
    s->ready = s->fields_ready && s->explicit_ready;
    return HYRF_OK;
}

// PAPER.md:227-229 (1)-(2): binary16 positions + R-VQ codes -> the scene's fp32 explicit arrays (decode.cu)
extern "C" hyrf_status hyrf_upload_explicit_rvq(hyrf_scene* s, const hyrf_explicit_rvq* q) {
    if (!s || !q) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_explicit_rvq: NULL argument");
    if (!q->pos_h || !q->codes || !q->codebooks) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_explicit_rvq: NULL pointer");
    if (q->stages < 1 || q->stages > 16) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_explicit_rvq: stages %u outside [1, 16]", q->stages);
    if (q->codebook_size < 1 || q->codebook_size > 65536)
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_explicit_rvq: codebook_size %u outside [1, 65536]", q->codebook_size);
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    const size_t N = s->N, S = q->stages, K = q->codebook_size;
    const size_t pos_b = 3 * N * sizeof(uint16_t), code_b = S * N * sizeof(uint16_t), book_b = S * K * 5 * sizeof(float);
    // staging: [first_bad | pad to 256][pos_h][codes][codebooks] (host sources), each part 256-byte aligned
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t stage_bytes = 256 + (q->host_ptrs ? up(pos_b) + up(code_b) + up(book_b) : 0);
    uint8_t* stage = nullptr;
    hyrf_status st = dev_alloc_t(s, &stage, stage_bytes);
    if (st != HYRF_OK) return st;
    uint32_t* first_bad = reinterpret_cast<uint32_t*>(stage);
    const uint16_t *pos_h = q->pos_h, *codes = q->codes;
    const float* books = q->codebooks;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    uint32_t bad = 0xFFFFFFFFu;
    auto done = [&](hyrf_status r) {
        if (ev0) cudaEventDestroy(ev0);
        if (ev1) cudaEventDestroy(ev1);
        dev_free(s, stage);
        return r;
    };
    s->explicit_ready = false;
    s->ready = false;
    if ((e = cudaMemsetAsync(first_bad, 0xFF, sizeof(uint32_t), s->stream)) != cudaSuccess) return done(hy_cuda_fail(e, "cudaMemsetAsync(first_bad)"));
    if (q->host_ptrs) {
        uint8_t* d_pos = stage + 256;
        uint8_t* d_codes = d_pos + up(pos_b);
        uint8_t* d_books = d_codes + up(code_b);
        if ((e = cudaMemcpyAsync(d_pos, q->pos_h, pos_b, cudaMemcpyHostToDevice, s->stream)) != cudaSuccess ||
            (e = cudaMemcpyAsync(d_codes, q->codes, code_b, cudaMemcpyHostToDevice, s->stream)) != cudaSuccess ||
            (e = cudaMemcpyAsync(d_books, q->codebooks, book_b, cudaMemcpyHostToDevice, s->stream)) != cudaSuccess)
            return done(hy_cuda_fail(e, "cudaMemcpyAsync(rvq)"));
        pos_h = reinterpret_cast<const uint16_t*>(d_pos);
        codes = reinterpret_cast<const uint16_t*>(d_codes);
        books = reinterpret_cast<const float*>(d_books);
    }
    if ((e = cudaEventCreate(&ev0)) != cudaSuccess || (e = cudaEventCreate(&ev1)) != cudaSuccess) return done(hy_cuda_fail(e, "cudaEventCreate"));
    cudaEventRecord(ev0, s->stream);
    if ((st = hy_launch_explicit_decode(s, pos_h, codes, books, (uint32_t)S, (uint32_t)K, first_bad)) != HYRF_OK) return done(st);
    cudaEventRecord(ev1, s->stream);
    if ((e = cudaMemcpyAsync(&bad, first_bad, sizeof(bad), cudaMemcpyDeviceToHost, s->stream)) != cudaSuccess) return done(hy_cuda_fail(e, "cudaMemcpyAsync(first_bad)"));
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return done(hy_cuda_fail(e, "cudaStreamSynchronize(decode)"));
    if (bad != 0xFFFFFFFFu)
        return done(hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_upload_explicit_rvq: a code of Gaussian %u is >= codebook_size %u", bad, (uint32_t)K));
    cudaEventElapsedTime(&s->decode_ms, ev0, ev1);
    if ((st = hy_prepare_morton(s)) != HYRF_OK) return done(st);
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return done(hy_cuda_fail(e, "cudaStreamSynchronize(upload)"));
    s->explicit_ready = true;
    s->ready = s->fields_ready && s->explicit_ready;
    return done(HYRF_OK);
}

extern "C" hyrf_status hyrf_set_raster_mode(hyrf_scene* s, int mode) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_raster_mode: NULL scene");
    if (mode < 0 || mode > 4) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_raster_mode: mode %d outside [0, 4]", mode);
    s->raster_mode = mode;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_raster_backward(hyrf_scene* s, const float* g_cfg, const float* g_T, float* grad, uint64_t grad_rows) {
    if (!s || !g_cfg || !g_T || !grad) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_raster_backward: NULL argument");
    if (!s->rendered || !s->list_final)
        return hy_fail(HYRF_ERR_NOT_READY, "hyrf_raster_backward: the last frame kept no per-tile lists (hyrf_set_retain_lists, or the debug export HYRF_DBG_TILE_LIST | HYRF_DBG_TILE_RANGES)");
    if (grad_rows < s->lastV)
        return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_raster_backward: grad holds %llu rows, the last frame has %u visible Gaussians", (unsigned long long)grad_rows, s->lastV);
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    uint32_t launches = 0;
    return hy_launch_raster_backward(s, g_cfg, g_T, grad, &launches);
}

extern "C" hyrf_status hyrf_last_raster_mode(hyrf_scene* s, int* mode) {
    if (!s || !mode) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_last_raster_mode: NULL argument");
    if (!s->rendered) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_last_raster_mode: no completed render");
    *mode = s->last_raster_mode;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_last_decode_time(hyrf_scene* s, float* ms) {
    if (!s || !ms) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_last_decode_time: NULL argument");
    if (s->decode_ms < 0.0f) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_last_decode_time: no hyrf_upload_explicit_rvq yet");
    *ms = s->decode_ms;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_destroy_scene(hyrf_scene* s) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_destroy_scene: NULL scene");
    cudaSetDevice(s->desc.device);
    destroy(s);
    return HYRF_OK;
}

namespace {

hyrf_status build_frame(const hyrf_scene* s, const hyrf_camera* cam, int32_t W, int32_t H, FrameDev* f) {
    for (int k = 0; k < 9; ++k) if (!isfinite(cam->R[k])) return hy_fail(HYRF_ERR_CAMERA, "camera R is not finite");
    for (int k = 0; k < 3; ++k) if (!isfinite(cam->t[k])) return hy_fail(HYRF_ERR_CAMERA, "camera t is not finite");
    if (!isfinite(cam->fx) || !isfinite(cam->fy) || !(cam->fx > 0.0f) || !(cam->fy > 0.0f) || !isfinite(cam->cx) || !isfinite(cam->cy))
        return hy_fail(HYRF_ERR_CAMERA, "camera intrinsics are not finite / positive");
    memcpy(f->R, cam->R, sizeof(f->R));
    memcpy(f->t, cam->t, sizeof(f->t));
    f->fx = cam->fx; f->fy = cam->fy; f->cx = cam->cx; f->cy = cam->cy;
    for (int k = 0; k < 3; ++k)   // DESIGN.md §2 "Camera": o = -R^T t
        f->o[k] = -(fmaf(cam->R[6 + k], cam->t[2], fmaf(cam->R[3 + k], cam->t[1], cam->R[k] * cam->t[0])));
    const double on = sqrt((double)f->o[0] * f->o[0] + (double)f->o[1] * f->o[1] + (double)f->o[2] * f->o[2]);
    if (!(on < (double)s->desc.bg_radius))
        return hy_fail(HYRF_ERR_CAMERA, "camera centre (|o| = %g) is not inside the background sphere (r = %g)", on, (double)s->desc.bg_radius);
    f->limx = (1.0f + s->desc.cull_tol) * ((float)W / (2.0f * cam->fx));
    f->limy = (1.0f + s->desc.cull_tol) * ((float)H / (2.0f * cam->fy));
    f->z_near = s->desc.z_near; f->tau_T = s->desc.tau_T; f->bg_radius = s->desc.bg_radius;
    for (int a = 0; a < 3; ++a) {
        f->aabb_c[a] = 0.5f * (s->desc.aabb_min[a] + s->desc.aabb_max[a]);
        f->aabb_h[a] = 0.5f * (s->desc.aabb_max[a] - s->desc.aabb_min[a]);
    }
    f->ablation = s->ablation;
    f->W = W; f->H = H;
    f->gx = (W + HY_TILE - 1) / HY_TILE; f->gy = (H + HY_TILE - 1) / HY_TILE;
    // small tile grids (<= 512 x 512 pixels) keep per-tile lists: with few tiles a macro tile's list is most of the scene
    // beyond that the binning works on macro tiles of 2^mshift x 2^mshift tiles (the rasterizer picks a tile's entries out of
    // its macro tile's list): the larger the splats, the coarser. Measured frame, 4 x 4 / 8 x 8 / 16 x 16 tiles: config 3
    // (10 tiles per visible Gaussian) 0.461 / 0.496 / - ms, config 4 (15) 0.808 / 0.888 / -, 500k @ 1080p (35) 0.527 /
    // 0.513 / -, 4M @ 1080p (35) 1.702 / 1.593 / -, 500k @ 4K (120) 1.215 / 1.167 / 1.168, 4M @ 4K (117) 2.984 / 2.284 /
    // 2.190; 2 x 2 was slower everywhere. The choice follows the previous frame (like the rasterizer's); bits do not depend on it.
    int msh = HY_MACRO_SHIFT;
    if (s->macro_shift) msh = s->macro_shift;
    else if (s->lastV != 0 && s->lastD > 96ull * s->lastV) msh = HY_MACRO_SHIFT + 2;
    else if (s->lastV != 0 && s->lastD > 24ull * s->lastV) msh = HY_MACRO_SHIFT + 1;
    f->mshift = (f->gx * f->gy <= 1024) ? 0 : msh;
    f->mgx = (f->gx + (1 << f->mshift) - 1) >> f->mshift; f->mgy = (f->gy + (1 << f->mshift) - 1) >> f->mshift;
    // screen strip (hyrf_set_strip): pixel rows [row0, row1) -> tile rows; the default is the whole image
    f->ty0 = 0; f->ty1 = f->gy;
    if (s->strip_row1 > s->strip_row0) {
        if (s->strip_row0 % HY_TILE != 0 || (s->strip_row1 % HY_TILE != 0 && s->strip_row1 < H) || s->strip_row0 >= H)
            return hy_fail(HYRF_ERR_INVALID_ARG, "strip rows [%d, %d) must start on a multiple of %d inside the image and end on one or at / beyond H = %d",
                           s->strip_row0, s->strip_row1, HY_TILE, H);
        f->ty0 = s->strip_row0 / HY_TILE;
        f->ty1 = s->strip_row1 >= H ? f->gy : s->strip_row1 / HY_TILE;
    }
    return HYRF_OK;
}

// hyrf_render_host_async leaves the device->host copy of the frame it has just enqueued PENDING; it is enqueued here,
// from the next call (once that frame's kernels are enqueued and the host would only wait for its counters) or from
// hyrf_host_sync. Two reasons. (1) The image travels in pieces of copy_chunk_bytes: while ONE 11 MB copy is in flight,
// kernels launched beside it start late (measured on B200: the cull stage of the next frame 0.029 -> 0.089 ms, its
// field kernel +0.016 ms; with 256 KB pieces the delay is gone). (2) 43 enqueues cost the host
// ~0.1 ms: here that time is hidden in a wait instead of standing between two frames.
hyrf_status hy_flush_pending_copy(hyrf_scene* s) {
    hyrf_scene::PendingCopy& pc = s->pending_copy;
    if (!pc.valid) return HYRF_OK;
    pc.valid = false;
    cudaError_t e;
    if ((e = cudaStreamWaitEvent(s->copy_stream, s->ev_rendered[pc.slot], 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent");
    const size_t chunk = s->copy_chunk_bytes ? s->copy_chunk_bytes : pc.bytes;
    for (size_t o = 0; o < pc.bytes; o += chunk) {
        const size_t nb = pc.bytes - o < chunk ? pc.bytes - o : chunk;
        if ((e = cudaMemcpyAsync((char*)pc.dst + o, (const char*)pc.src + o, nb, cudaMemcpyDeviceToHost, s->copy_stream)) != cudaSuccess)
            return hy_cuda_fail(e, "cudaMemcpyAsync(image)");
    }
    if ((e = cudaEventRecord(s->ev_copied[pc.slot], s->copy_stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord");
    return HYRF_OK;
}

hyrf_status render_impl(hyrf_scene* s, const hyrf_camera* cam, int32_t W, int32_t H, float* out_rgb) {
    if (!s || !cam || !out_rgb) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_render: NULL argument");
    if (!s->ready) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_render before the fields (hyrf_upload_params) and the explicit Gaussians (hyrf_upload_params or hyrf_upload_explicit_rvq) were uploaded");
    if (W < 1 || H < 1 || (uint32_t)W > s->desc.max_width || (uint32_t)H > s->desc.max_height)
        return hy_fail(HYRF_ERR_INVALID_ARG, "W x H = %d x %d outside [1, %u] x [1, %u]", W, H, s->desc.max_width, s->desc.max_height);
    FrameDev f;
    hyrf_status st = build_frame(s, cam, W, H, &f);
    if (st != HYRF_OK) return st;
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    const bool timing = s->timing;
    if (timing && !s->ev_valid) {
        for (auto& ev : s->ev) if ((e = cudaEventCreate(&ev)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventCreate");
        s->ev_valid = true;
    }
    uint32_t launches = 0;
    s->lastW = W; s->lastH = H;
    s->rendered = false;
    // S1 and the depth sort write the OTHER set of their buffers than the previous frame (scene.h PreSet)
    hy_select_pre_set(s, s->pre_cur ^ 1);
    hyrf_scene::PreSet& P = s->pre[s->pre_cur];
    const bool overlap = s->sort_overlap;
    const bool pipeline = (s->pipeline || s->pipeline_all) && overlap;
    cudaStream_t pst = overlap ? s->sort_stream : s->stream;   // where S1 and the depth sort run
    if (timing) {
        s->prev_timed = s->last_timed;
        s->ev_end = s->ev_end == 5 ? 6 : 5;
        cudaEventRecord(s->ev[0], s->stream);
    }
    s->last_timed = timing;
    if (overlap) {
        // the frame that last used this set (two frames ago) must have stopped reading it
        if (P.in_use && (e = cudaStreamWaitEvent(pst, P.ev_free, 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent(set free)");
        if (!pipeline) {
            // one frame at a time (hyrf_render / hyrf_render_host): S1 starts behind everything already enqueued on the
            // caller's stream. A pipelined stream of frames (hyrf_render_host_async) skips this: its cull and depth sort
            // run beside the previous frame's rasterizer.
            if ((e = cudaEventRecord(s->ev_start, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(start)");
            if ((e = cudaStreamWaitEvent(pst, s->ev_start, 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent(start)");
        }
    }

    // S1: visibility pre-culling
    hy_launch_cull(s, f, &launches, pst, P.scan);
    if (overlap) {
        if ((e = cudaEventRecord(s->ev_culled, pst)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(culled)");
        if ((e = cudaStreamWaitEvent(s->stream, s->ev_culled, 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent(culled)");
    }
    if (timing) cudaEventRecord(s->ev[1], s->stream);

    // S4c first half: order the visible Gaussians by (depth bits, id). The keys are the cull's (Z needs nothing from
    // the fields), so the five small, latency-bound sort kernels run on their own stream beside the field kernel,
    // which leaves a few SMs free for them (hy_launch_field_*), and join the frame before the binning.
    uint32_t *order_key = nullptr, *order = nullptr;
    // every visible Gaussian has Z > z_near > 0, so its key (the bits of Z) is above the bits of z_near: the sort works on
    // the difference, which needs fewer digits (radix.cu). Without pre-culling (ablation) any Z can occur: plain keys.
    uint32_t depth_key_sub = 0;
    int depth_key_bits = 32;
    if (!(f.ablation & HYRF_ABL_NO_CULL)) {
        memcpy(&depth_key_sub, &f.z_near, sizeof(uint32_t));
        // Z = r3 . p + t_z <= |r3| r_max + |t_z| (1 % and one float step above the three binary32 fmas that compute it):
        // the keys to sort lie in (bits(z_near), bits(bound)], a range that normally fits 27 bits = three digits
        const double r3 = sqrt((double)f.R[6] * f.R[6] + (double)f.R[7] * f.R[7] + (double)f.R[8] * f.R[8]);
        const double zb = (r3 * s->r_max + fabs((double)f.t[2])) * 1.01;
        if (zb < 1e37) {
            const float zf = nextafterf((float)zb, INFINITY);
            uint32_t top;
            memcpy(&top, &zf, sizeof(uint32_t));
            depth_key_bits = 1;
            while (depth_key_bits < 32 && (top > depth_key_sub ? top - depth_key_sub : 0u) >> depth_key_bits) ++depth_key_bits;
        }
    }
    if (overlap) {
        hy_launch_radix(s->sort_a_key, s->sort_a_val, s->sort_b_key, s->sort_b_val, s->N, &s->counters->V, depth_key_bits, P.hist,
                        P.scan, pst, &order_key, &order, &launches, /*iota_vals=*/true, depth_key_sub);
        if ((e = cudaEventRecord(s->ev_sorted, pst)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(sorted)");
    }
    // In a pipelined stream the sort has the previous frame's rasterizer to hide under, so the field kernel takes every
    // SM; otherwise it leaves some to the sort running beside it.
    s->field_full_grid = !overlap || (pipeline && s->frame_in_flight && cudaEventQuery(s->ev_frame_done) == cudaErrorNotReady);
    cudaGetLastError();

    // S2 + S3 + S4a: field query, aggregation, projection
    // (explicit-only ablation: no field is queried, so the CUDA-core kernel's early-out path serves both dtypes)
    const bool mma = s->use_mma && !(s->ablation & HYRF_ABL_NO_NEURAL);
    if ((st = !mma ? hy_launch_field_fma(s, f, &launches)
                   : (s->ws_mma ? hy_launch_field_ws(s, f, &launches) : hy_launch_field_mma(s, f, &launches))) != HYRF_OK) return st;
    if (timing) cudaEventRecord(s->ev[2], s->stream);

    // counters (V, D) start their way to the host now; the depth ordering below does not need them, so the copy
    // and the host's wake-up hide behind it
    // (written by a one-warp kernel straight into the pinned host block, not by a memcpy: a device-to-host memcpy would
    // queue on the copy engine behind the previous frame's 11 MB image copy of hyrf_render_host_async and hold this
    // stream — and the host — back until that has finished)
    hy_launch_counters_to_host(s->counters, s->counters_host, s->stream);
    ++launches;
    if ((e = cudaEventRecord(s->ev_counters, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(counters)");

    // S4b-c: the depth order joins here (or is computed here when serialised); build the per-tile lists in that order
    if (overlap) {
        if ((e = cudaStreamWaitEvent(s->stream, s->ev_sorted, 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent(sorted)");
    } else {
        hy_launch_radix(s->sort_a_key, s->sort_a_val, s->sort_b_key, s->sort_b_val, s->N, &s->counters->V, depth_key_bits, P.hist,
                        P.scan, s->stream, &order_key, &order, &launches, /*iota_vals=*/true, depth_key_sub);
    }
    const uint32_t n_tiles = (uint32_t)(f.gx * f.gy);
    uint32_t V = 0;
    uint64_t D = 0;
    // The binning works on MACRO tiles (4 x 4 tiles): ~3 list entries per Gaussian instead of ~10, and the rasterizer
    // picks each tile's subsequence out of its macro tile's depth-ordered list while staging. Per-TILE ranges and lists
    // are only materialised when the debug export asks for them: the ranges by a second, tile-level run of the same
    // binning, the lists by the rasterizer itself (what it consumed, in the order it consumed it).
    const uint32_t n_macro = (uint32_t)(f.mgx * f.mgy);
    const bool export_lists = ((s->debug_mask >> HYRF_DBG_TILE_LIST) | (s->debug_mask >> HYRF_DBG_TILE_RANGES)) & 1u;
    // per-tile lists are kept for the backward pass (hyrf_set_retain_lists) or written out whole for the debug export;
    // only the export needs every tile's list to its end, so a retained list stops where the tile's pixels all had
    // terminated (list_len) and the rasterizer keeps its early exit
    const bool want_lists = export_lists || s->retain_lists;
    const bool ordered = s->bin_ws && hy_bin_ordered_supported(s->N, n_macro) && (!want_lists || hy_bin_ordered_supported(s->N, n_tiles));
    if ((!ordered || want_lists) && (st = hy_flush_pending_copy(s)) != HYRF_OK) return st;   // these routes wait for the counters first
    if (ordered && want_lists) {
        // The export makes the rasterizer write every tile's list (D entries) into the pair buffer, and nothing there
        // checks a bound: learn D BEFORE anything is binned and grow first. (Without the export the frame is enqueued
        // blind and only re-binned on overflow: the binning itself clamps to the capacity.) The stream has joined the
        // depth sort by now, so synchronising it also covers the sort's use of the workspace that growing reallocates.
        if ((e = cudaEventSynchronize(s->ev_counters)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventSynchronize(counters)");
        const uint64_t need = s->counters_host->D > s->counters_host->Dm ? s->counters_host->D : s->counters_host->Dm;
        if (need >= 0xFFFFFFFFull) return hy_fail(HYRF_ERR_OOM, "tile-entry count %llu does not fit 32-bit offsets", (unsigned long long)need);
        if (need > s->d_capacity) {
            if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(grow)");
            if ((st = ensure_entries(s, (size_t)need)) != HYRF_OK) return st;
        }
    }
    if (ordered) {
        // everything is sized on the device, so the whole frame is enqueued before the host looks at the counters;
        // only a frame whose entry count outgrew the list buffer is re-binned after growing it
        for (int attempt = 0;; ++attempt) {
            if (attempt > 0 && (e = cudaMemsetAsync(&s->counters->n_bg, 0, 3 * sizeof(uint32_t), s->stream)) != cudaSuccess)
                return hy_cuda_fail(e, "cudaMemsetAsync(n_bg)");   // n_bg, bin_ticket, bin_done: the first attempt used them
            if (want_lists) {
                if ((st = hy_launch_bin_ordered(s, order, n_tiles, (uint32_t)f.gx, &launches, /*macro=*/false, 0)) != HYRF_OK) return st;
                if ((e = cudaMemsetAsync(&s->counters->bin_ticket, 0, 2 * sizeof(uint32_t), s->stream)) != cudaSuccess)
                    return hy_cuda_fail(e, "cudaMemsetAsync(bin_ticket)");
            }
            if ((st = hy_launch_bin_ordered(s, order, n_tiles, (uint32_t)f.gx, &launches, /*macro=*/true, (uint32_t)f.mshift)) != HYRF_OK) return st;
            // the per-tile lists are written by the rasterizer into the (by then dead) pair array of the macro run
            s->list_final = want_lists ? s->ent_val[0] : nullptr;
            if (timing) cudaEventRecord(s->ev[3], s->stream);
            s->list_partial = want_lists && !export_lists;
            if (s->list_partial && (e = cudaMemsetAsync(s->list_len, 0, (size_t)n_tiles * sizeof(uint32_t), s->stream)) != cudaSuccess)
                return hy_cuda_fail(e, "cudaMemsetAsync(list_len)");   // (tiles of another device's strip stay empty)
            hy_launch_raster(s, f, s->mranges, s->ent_key[1], /*macro=*/true, out_rgb, &launches, s->tile_queue,
                             want_lists ? s->ent_val[0] : nullptr, s->list_partial ? s->list_len : nullptr);                            // S5 (Eq. 1)
            if (timing) cudaEventRecord(s->ev[4], s->stream);
            if ((st = hy_launch_background(s, f, out_rgb, &launches)) != HYRF_OK) return st;   // S6 (Eq. 10-11, A.2)
            if (timing) cudaEventRecord(s->ev[s->ev_end], s->stream);
            if (attempt == 0 && (st = hy_flush_pending_copy(s)) != HYRF_OK) return st;   // (the previous frame's image: see there)
            if (attempt == 0 && (e = cudaEventSynchronize(s->ev_counters)) != cudaSuccess)
                return hy_cuda_fail(e, "cudaEventSynchronize(counters)");
            V = s->counters_host->V;
            D = s->counters_host->D;
            const uint64_t need = want_lists && D > s->counters_host->Dm ? D : s->counters_host->Dm;
            if (need >= 0xFFFFFFFFull) return hy_fail(HYRF_ERR_OOM, "tile-entry count %llu does not fit 32-bit offsets", (unsigned long long)need);
            if (need <= s->d_capacity) break;
            if (attempt > 0) return hy_fail(HYRF_ERR_OOM, "tile-entry scratch still too small after growing");
            if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(grow)");
            if ((st = ensure_entries(s, (size_t)need)) != HYRF_OK) return st;
        }
    } else {
        // radix route (very large tile grids): (tile, rank) pairs emitted in depth order, stable sort by tile id
        if ((e = cudaEventSynchronize(s->ev_counters)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventSynchronize(counters)");
        V = s->counters_host->V;
        D = s->counters_host->D;
        if (D >= 0xFFFFFFFFull || D > hy_radix_max_items())
            return hy_fail(HYRF_ERR_OOM, "tile-entry count %llu exceeds the supported maximum", (unsigned long long)D);
        if (D > s->d_capacity) {
            // growing frees the sort workspace the depth ordering is still using: wait for it first
            if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(grow)");
            // the depth order lives in the N-sized buffers, which are not reallocated
            if ((st = ensure_entries(s, (size_t)D)) != HYRF_OK) return st;
        }
        hy_launch_tiles_gather(s, order, V, &launches);
        hy_launch_scan(s->tt_sorted, s->offs, V, s->scan_scratch, s->stream, &launches);
        hy_launch_emit(s, order, V, &launches);
        int tile_bits = 1;
        while ((1u << tile_bits) < n_tiles) ++tile_bits;
        uint32_t *sorted_key = nullptr, *sorted_val = nullptr;
        hy_launch_radix(s->ent_key[0], s->ent_val[0], s->ent_key[1], s->ent_val[1], (size_t)D, nullptr, tile_bits, s->hist,
                        s->scan_scratch, s->stream, &sorted_key, &sorted_val, &launches);
        hy_launch_ranges(s, sorted_key, D, n_tiles, &launches);
        s->list_final = sorted_val;
        if (timing) cudaEventRecord(s->ev[3], s->stream);
        s->list_partial = false;
        hy_launch_raster(s, f, s->ranges, sorted_val, /*macro=*/false, out_rgb, &launches, nullptr, nullptr, nullptr);   // S5
        if (timing) cudaEventRecord(s->ev[4], s->stream);
        if ((st = hy_launch_background(s, f, out_rgb, &launches)) != HYRF_OK) return st;       // S6 (Eq. 10-11, A.2)
        if (timing) cudaEventRecord(s->ev[s->ev_end], s->stream);
    }

    if ((e = cudaGetLastError()) != cudaSuccess) return hy_cuda_fail(e, "kernel launch");
    // from here on nothing of this frame reads the cull / sort set any more (the rasterizer and the background work from
    // the records and lists): the frame after next may overwrite it
    if ((e = cudaEventRecord(P.ev_free, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(set free)");
    P.in_use = true;
    if ((e = cudaEventRecord(s->ev_frame_done, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord(frame done)");
    s->frame_in_flight = true;
    s->last_launches = launches;
    s->last_frame = f;
    s->lastV = V; s->lastD = D; s->lastDm = s->counters_host->Dm;
    s->rendered = true;
    return HYRF_OK;
}

}  // namespace

extern "C" hyrf_status hyrf_render(hyrf_scene* s, const hyrf_camera* cam, int32_t W, int32_t H, float* out_rgb) {
    return render_impl(s, cam, W, H, out_rgb);
}

extern "C" hyrf_status hyrf_render_host(hyrf_scene* s, const hyrf_camera* cam, int32_t W, int32_t H, float* out_host) {
    if (!s || !out_host) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_render_host: NULL argument");
    if (!s->image) {
        hyrf_status st = dev_alloc_t(s, &s->image, (size_t)s->desc.max_width * s->desc.max_height * 3);
        if (st != HYRF_OK) return st;
    }
    hyrf_status st = render_impl(s, cam, W, H, s->image);
    if (st != HYRF_OK) return st;
    cudaError_t e = cudaMemcpyAsync(out_host, s->image, (size_t)W * H * 3 * sizeof(float), cudaMemcpyDeviceToHost, s->stream);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyAsync(image)");
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(image)");
    return HYRF_OK;
}

// Pipelined host delivery: frame k renders into one of two library-owned device images on the scene's stream; its
// device->host copy runs on a second stream behind an event, so it overlaps the render of frame k+1.
extern "C" hyrf_status hyrf_render_host_async(hyrf_scene* s, const hyrf_camera* cam, int32_t W, int32_t H, float* out_host) {
    if (!s || !out_host) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_render_host_async: NULL argument");
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    hyrf_status st;
    if (!s->copy_stream) {
        if ((e = cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamCreate(copy)");
        for (int k = 0; k < 2; ++k) {
            if ((e = cudaEventCreateWithFlags(&s->ev_rendered[k], cudaEventDisableTiming)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventCreate");
            if ((e = cudaEventCreateWithFlags(&s->ev_copied[k], cudaEventDisableTiming)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventCreate");
        }
    }
    const size_t P3 = (size_t)s->desc.max_width * s->desc.max_height * 3;
    if (!s->image && (st = dev_alloc_t(s, &s->image, P3)) != HYRF_OK) return st;
    if (!s->image2 && (st = dev_alloc_t(s, &s->image2, P3)) != HYRF_OK) return st;
    const int slot = (s->host_slot ^= 1);
    float* img = slot ? s->image2 : s->image;
    // (normally the pending copy is the OTHER image's and goes out during this call; after a failed call it may be this one's)
    if (s->pending_copy.valid && s->pending_copy.slot == slot && (st = hy_flush_pending_copy(s)) != HYRF_OK) return st;
    // the copy that last read this image must have finished before it is rendered into again
    if (s->slot_used[slot] && (e = cudaStreamWaitEvent(s->stream, s->ev_copied[slot], 0)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamWaitEvent");
    s->pipeline = true;   // a stream of frames: this one's cull and depth sort may run beside the previous one's rasterizer
    st = render_impl(s, cam, W, H, img);
    s->pipeline = false;
    if (st != HYRF_OK) return st;
    if ((e = cudaEventRecord(s->ev_rendered[slot], s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaEventRecord");
    s->pending_copy = {out_host, img, (size_t)W * H * 3 * sizeof(float), slot, true};   // enqueued by hy_flush_pending_copy
    s->slot_used[slot] = true;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_host_sync(hyrf_scene* s) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_host_sync: NULL scene");
    cudaError_t e;
    hyrf_status st = hy_flush_pending_copy(s);
    if (st != HYRF_OK) return st;
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize");
    if (s->copy_stream && (e = cudaStreamSynchronize(s->copy_stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(copy)");
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_timing(hyrf_scene* s, int32_t enabled) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_timing: NULL scene");
    s->timing = enabled != 0;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_stage_times(hyrf_scene* s, float ms[6]) {
    if (!s || !ms) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_stage_times: NULL argument");
    if (!s->rendered || !s->timing || !s->ev_valid) return hy_fail(HYRF_ERR_NOT_READY, "no timed render yet");
    cudaError_t e = cudaEventSynchronize(s->ev[s->ev_end]);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaEventSynchronize");
    for (int k = 0; k < 5; ++k)
        if ((e = cudaEventElapsedTime(&ms[k], s->ev[k], s->ev[k == 4 ? s->ev_end : k + 1])) != cudaSuccess) return hy_cuda_fail(e, "cudaEventElapsedTime");
    if ((e = cudaEventElapsedTime(&ms[5], s->ev[0], s->ev[s->ev_end])) != cudaSuccess) return hy_cuda_fail(e, "cudaEventElapsedTime");
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_frame_gap(hyrf_scene* s, float* ms) {
    if (!s || !ms) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_frame_gap: NULL argument");
    if (!s->rendered || !s->timing || !s->ev_valid || !s->prev_timed) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_frame_gap needs two consecutive timed renders");
    cudaError_t e = cudaEventSynchronize(s->ev[s->ev_end]);
    if (e != cudaSuccess) return hy_cuda_fail(e, "cudaEventSynchronize");
    if ((e = cudaEventElapsedTime(ms, s->ev[s->ev_end == 5 ? 6 : 5], s->ev[0])) != cudaSuccess) return hy_cuda_fail(e, "cudaEventElapsedTime");
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_ablation(hyrf_scene* s, uint32_t mask) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_ablation: NULL scene");
    if (mask & ~15u) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_ablation: unknown bits in mask %u", mask);
    s->ablation = mask;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_sort_overlap(hyrf_scene* s, int on) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_sort_overlap: NULL scene");
    s->sort_overlap = on != 0;
    if (on > 1) s->ws_sort_sms = on < s->sm_count ? on : s->sm_count - 1;   // on > 1: SMs the warp-specialised field kernel leaves to the sort
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_retain_lists(hyrf_scene* s, int on) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_retain_lists: NULL scene");
    s->retain_lists = on != 0;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_bin_granularity(hyrf_scene* s, int shift) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_bin_granularity: NULL scene");
    if (shift != 0 && (shift < 1 || shift > 4)) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_bin_granularity: shift %d outside {0, 1 .. 4}", shift);
    s->macro_shift = shift;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_strip(hyrf_scene* s, int32_t row_begin, int32_t row_end) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_strip: NULL scene");
    if (row_begin < 0 || row_end < row_begin) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_strip: rows [%d, %d)", row_begin, row_end);
    s->strip_row0 = row_begin; s->strip_row1 = row_end;   // row_end == row_begin: the whole image again
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_set_pipelining(hyrf_scene* s, int on) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_set_pipelining: NULL scene");
    s->pipeline_all = on != 0;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_last_launch_count(hyrf_scene* s, uint32_t* launches) {
    if (!s || !launches) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_last_launch_count: NULL argument");
    *launches = s->last_launches;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_debug_enable(hyrf_scene* s, uint32_t mask) {
    if (!s) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_debug_enable: NULL scene");
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    cudaStreamSynchronize(s->stream);
    const size_t N = s->N, P = (size_t)s->desc.max_width * s->desc.max_height;
    hyrf_status st;
    if (((mask >> HYRF_DBG_STAGE2_RAW) & 1u) && !s->dbg_raw && (st = dev_alloc_t(s, &s->dbg_raw, 11 * N)) != HYRF_OK) return st;
    if (((mask >> HYRF_DBG_STAGE3_ATTRS) & 1u) && !s->dbg_attrs && (st = dev_alloc_t(s, &s->dbg_attrs, 11 * N)) != HYRF_OK) return st;
    if (((mask >> HYRF_DBG_BG_MASK) & 1u) && !s->bg_mask && (st = dev_alloc_t(s, &s->bg_mask, P)) != HYRF_OK) return st;
    if (((mask >> HYRF_DBG_FG) & 1u) && !s->fg && (st = dev_alloc_t(s, &s->fg, 3 * P)) != HYRF_OK) return st;
    s->debug_mask = mask;
    s->rendered = false;
    return HYRF_OK;
}

extern "C" hyrf_status hyrf_debug_fetch(hyrf_scene* s, uint32_t kind, void* host_dst, size_t cap, size_t* bytes) {
    if (!s || !bytes) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_debug_fetch: NULL argument");
    if (kind == HYRF_DBG_EXPLICIT) {   // what the uploads left in the scene: p_e[3], s_e, alpha_e, c_e[3], one row each
        if (!s->explicit_ready) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_debug_fetch: no explicit parameters uploaded");
        const size_t row = (size_t)s->N * sizeof(float);
        *bytes = 8 * row;
        if (!host_dst) return HYRF_OK;
        if (8 * row > cap) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_debug_fetch: need %zu bytes, cap %zu", 8 * row, cap);
        cudaError_t ce;
        if ((ce = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(ce, "cudaSetDevice");
        if ((ce = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(ce, "cudaStreamSynchronize(debug)");
        uint8_t* o = static_cast<uint8_t*>(host_dst);
        if ((ce = cudaMemcpy(o, s->pos, 3 * row, cudaMemcpyDeviceToHost)) != cudaSuccess ||
            (ce = cudaMemcpy(o + 3 * row, s->scale, row, cudaMemcpyDeviceToHost)) != cudaSuccess ||
            (ce = cudaMemcpy(o + 4 * row, s->opac, row, cudaMemcpyDeviceToHost)) != cudaSuccess ||
            (ce = cudaMemcpy(o + 5 * row, s->rgb, 3 * row, cudaMemcpyDeviceToHost)) != cudaSuccess)
            return hy_cuda_fail(ce, "cudaMemcpy(explicit)");
        return HYRF_OK;
    }
    if (!s->rendered) return hy_fail(HYRF_ERR_NOT_READY, "hyrf_debug_fetch: no completed render");
    cudaError_t e;
    if ((e = cudaSetDevice(s->desc.device)) != cudaSuccess) return hy_cuda_fail(e, "cudaSetDevice");
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(debug)");
    const size_t N = s->N, V = s->lastV, D = (size_t)s->lastD, P = (size_t)s->lastW * s->lastH;
    const size_t n_tiles = (size_t)((s->lastW + HY_TILE - 1) / HY_TILE) * ((s->lastH + HY_TILE - 1) / HY_TILE);
    const bool on = (kind < 32) && ((s->debug_mask >> kind) & 1u);
    const void* src = nullptr;
    size_t need = 0;
    switch (kind) {
        case HYRF_DBG_VIS_MASK: need = N; break;
        case HYRF_DBG_VIS_IDX: src = s->vis_idx; need = V * 4; break;
        case HYRF_DBG_STAGE2_RAW: if (!on) goto off; src = s->dbg_raw; need = V * 44; break;
        case HYRF_DBG_STAGE3_ATTRS: if (!on) goto off; src = s->dbg_attrs; need = V * 44; break;
        case HYRF_DBG_PROJ: need = V * 40; break;
        case HYRF_DBG_RECT: src = s->rect; need = V * 16; break;
        case HYRF_DBG_TILE_RANGES: if (!on) goto off; src = s->ranges; need = n_tiles * 8; break;
        case HYRF_DBG_TILE_LIST: if (!on || !s->list_final) goto off; need = D * 4; break;
        case HYRF_DBG_FINAL_T: src = s->finalT; need = P * 4; break;
        case HYRF_DBG_BG_MASK: if (!on) goto off; src = s->bg_mask; need = P; break;
        case HYRF_DBG_COUNTERS: need = 40; break;
        case HYRF_DBG_FG: if (!on) goto off; src = s->fg; need = P * 12; break;
        default: return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_debug_fetch: unknown kind %u", kind);
    }
    *bytes = need;
    if (!host_dst) return HYRF_OK;
    if (need > cap) return hy_fail(HYRF_ERR_INVALID_ARG, "hyrf_debug_fetch: need %zu bytes, cap %zu", need, cap);
    if (need == 0) return HYRF_OK;
    if (kind == HYRF_DBG_COUNTERS) {
        uint64_t c[5] = {N, V, D, n_tiles, s->lastDm};
        memcpy(host_dst, c, sizeof(c));
        return HYRF_OK;
    }
    if (kind == HYRF_DBG_VIS_MASK) {   // visibility bits by id -> one byte per Gaussian
        std::vector<uint32_t> words((N + 31) / 32);
        if ((e = cudaMemcpy(words.data(), s->id_words, words.size() * 4, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(id_words)");
        uint8_t* o = static_cast<uint8_t*>(host_dst);
        for (size_t i = 0; i < N; ++i) o[i] = (words[i >> 5] >> (i & 31)) & 1u;
        return HYRF_OK;
    }
    if (kind == HYRF_DBG_PROJ) {   // records -> (u, v, depth, A, B, C, opacity, r, g, b)
        std::vector<float> rec(12 * V);
        if ((e = cudaMemcpy(rec.data(), s->rec, rec.size() * 4, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(rec)");
        float* o = static_cast<float*>(host_dst);
        for (size_t j = 0; j < V; ++j) {
            const float* r = &rec[12 * j];
            float* d = o + 10 * j;
            d[0] = r[0]; d[1] = r[1]; d[2] = r[9]; d[3] = r[2]; d[4] = r[3]; d[5] = r[4]; d[6] = r[5]; d[7] = r[6]; d[8] = r[7]; d[9] = r[8];
        }
        return HYRF_OK;
    }
    if (kind == HYRF_DBG_TILE_LIST) {   // visible ranks -> Gaussian ids
        std::vector<uint32_t> idx(V);
        if (V && (e = cudaMemcpy(idx.data(), s->vis_idx, V * 4, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(vis_idx)");
        uint32_t* o = static_cast<uint32_t*>(host_dst);
        if ((e = cudaMemcpy(o, s->list_final, D * 4, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(list)");
        for (size_t q = 0; q < D; ++q) o[q] = o[q] < V ? idx[o[q]] : 0xFFFFFFFFu;
        return HYRF_OK;
    }
    if ((e = cudaMemcpy(host_dst, src, need, cudaMemcpyDeviceToHost)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpy(debug)");
    return HYRF_OK;
off:
    return hy_fail(HYRF_ERR_NOT_READY, "hyrf_debug_fetch: kind %u was not enabled with hyrf_debug_enable before the render", kind);
}
