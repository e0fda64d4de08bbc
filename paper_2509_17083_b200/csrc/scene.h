// scene.h — host-side scene object and the kernel launchers behind the C-ABI (include/hyrf.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/hyrf.h"
#include "common.cuh"

struct MlpDev {
    const void* w;        // as uploaded: layers concatenated, row-major [out][in], float or __half
    uint32_t in_dim, hidden, n_hidden, out_dim;
};

// Device counters of one frame (one cache line).
struct FrameCounters {
    uint32_t V;           // visible Gaussians after S1
    uint32_t pad0;
    unsigned long long D; // tile entries (sum of tiles touched)
    uint32_t n_bg;        // pixels whose residual transmittance passes tau_T (S6 work list)
    uint32_t bin_ticket;  // block tickets of bin_offsets_kernel
    uint32_t bin_done;    // finished CTAs of bin_prefix_kernel
    uint32_t pad[1];
    unsigned long long Dm; // macro-tile entries (sum of 4x4-tile blocks touched): what the binning actually moves
    uint32_t pad2[6];
};

struct hyrf_scene {
    hyrf_scene_desc desc;
    std::vector<uint32_t> res_geo, res_app, res_bg;
    bool ready = false;          // fields_ready && explicit_ready
    bool fields_ready = false;   // tables and decoder weights uploaded (hyrf_upload_params)
    bool explicit_ready = false; // explicit Gaussians uploaded (hyrf_upload_params or hyrf_upload_explicit_rvq)
    float decode_ms = -1.0f;     // decode kernel of the last hyrf_upload_explicit_rvq
    bool fp16 = false;         // decoder weights / activations in fp16 (param_dtype F16 or U8)
    bool u8 = false;           // grid tables are 8-bit min-max codes (param_dtype U8)
    bool use_mma = false;
    bool warp_mma = false;     // decoders on warp-level mma.sync (field_warp_kernel) instead of tcgen05 (field_mma.cu)
    cudaStream_t stream = 0;
    uint32_t N = 0;
    int sm_count = 0;          // cudaDevAttrMultiProcessorCount of desc.device (148 on a full B200)
    bool field_attr_set = false;   // cudaFuncSetAttribute of the tensor-core field kernels done for this scene's device
    bool field_ws_attr_set = false;
    bool ws_mma = false;       // decoders on tcgen05 with warp-specialised gather / decoder roles (field_ws.cu)
    double r_max = INFINITY;   // max |position| over the Gaussians (hy_prepare_morton): bounds every camera-space depth
    int ws_sort_sms = 16;      // SMs the warp-specialised field kernel leaves to the depth sort running beside it (swept 12..40 on configs 3, 4, 5: DESIGN.md section 11)

    // persistent parameters
    float* pos = nullptr;      // [3][N]
    float* rgb = nullptr;      // [3][N]
    float* scale = nullptr;    // [N]
    float* opac = nullptr;     // [N]
    GridDev geo_grid{}, app_grid{}, bg_grid{};
    size_t geo_entries = 0, app_entries = 0, bg_entries = 0;
    MlpDev geo_mlp{}, app_mlp{}, bg_mlp{};
    void* mma_w = nullptr;     // fp16 weights re-laid out for the tensor-core path (field_mma.cu)
    void* both_table = nullptr;  // geo + app tables interleaved [entry][4] half, when the two grids share their geometry
    float4* gm = nullptr;      // [N][2] Morton-ordered records (pos.xyz, scale | opacity, rgb), built at upload (cull.cu)
    uint32_t* gm_id = nullptr; // [N] id of the m-th Gaussian in Morton order

    // What S1 and the depth sort write exists twice: a stream of frames (hyrf_render_host_async) runs frame k+1's cull and
    // sort on `sort_stream` beside frame k's rasterizer. The members below with the same names alias the set of the frame
    // being enqueued (and, afterwards, of the last frame: what the debug fetches read).
    struct PreSet {
        uint32_t *flag_words = nullptr, *id_words = nullptr, *word_rank = nullptr, *vis_m = nullptr, *block_counts = nullptr,
                 *vis_idx = nullptr, *sort_a_key = nullptr, *sort_a_val = nullptr, *sort_b_key = nullptr, *sort_b_val = nullptr;
        uint32_t *hist = nullptr, *scan = nullptr;        // radix / scan workspace of the depth sort and the cull's scans
        FrameCounters *counters = nullptr, *counters_host = nullptr;
        cudaEvent_t ev_free = nullptr;                    // main stream: the frame that used this set no longer reads it
        bool in_use = false;
    } pre[2];
    int pre_cur = 0;
    bool pipeline = false;            // the frame being enqueued belongs to a pipelined stream (no ordering behind the previous frame's tail)
    size_t copy_chunk_bytes = 256u << 10; // hyrf_render_host_async: the image goes to the host in pieces of this size (api.cu)
    struct PendingCopy { float* dst; const float* src; size_t bytes; int slot; bool valid; } pending_copy = {nullptr, nullptr, 0, 0, false};
    bool pipeline_all = false;        // hyrf_set_pipelining: every hyrf_render is enqueued that way
    bool frame_in_flight = false;     // a previous frame's end event has been recorded
    bool field_full_grid = false;     // this frame's field kernel takes every SM (nothing runs beside it, or the sort hides elsewhere)
    cudaEvent_t ev_start = nullptr, ev_frame_done = nullptr;

    // per-frame scratch sized from N
    uint32_t* flag_words = nullptr;   // [ceil(N/32)] visibility bits, Morton order
    uint32_t* id_words = nullptr;     // [ceil(N/32)] visibility bits, id order (also the VIS_MASK debug export)
    uint32_t* word_rank = nullptr;    // [ceil(N/32)] visible rank of the first bit of each id word
    uint32_t* vis_m = nullptr;        // [N] Morton indices of the visible Gaussians (the field kernels' work list)
    uint32_t* block_counts = nullptr; // cull block counts / scanned
    uint32_t* vis_idx = nullptr;      // [N]
    float4* rec = nullptr;            // [N][3] projected records
    uint4* rect = nullptr;            // [N] (x0, x1, y0, y1)
    uint32_t* tiles = nullptr;        // [N] tiles touched
    uint32_t* mtiles = nullptr;       // [N] macro tiles (4x4-tile blocks) touched
    uint32_t* sort_a_key = nullptr;   // [N] ping-pong buffers of the depth sort; the field kernel writes (depth bits, rank) into a
    uint32_t* sort_a_val = nullptr;
    uint32_t* sort_b_key = nullptr;
    uint32_t* sort_b_val = nullptr;
    uint32_t* tt_sorted = nullptr;    // [N] tiles touched in depth order
    uint32_t* offs = nullptr;         // [N] exclusive scan of tt_sorted
    uint32_t* scan_scratch = nullptr; // pyramid for the device-wide scan
    size_t scan_scratch_elems = 0;
    uint32_t* bin_ws = nullptr;       // ordered binning: count matrix [chunks][tiles] + totals + look-back words
    uint32_t bin_frame = 0;           // tag of the look-back words (bin_ordered.cu)
    uint32_t* hist = nullptr;         // [256][radix blocks] block histograms
    size_t hist_elems = 0;
    FrameCounters* counters = nullptr;       // device
    FrameCounters* counters_host = nullptr;  // pinned

    // per-frame scratch sized from D (grown on demand)
    size_t d_capacity = 0;
    uint32_t* ent_key[2] = {nullptr, nullptr};  // tile id per entry
    uint32_t* ent_val[2] = {nullptr, nullptr};  // visible rank per entry
    uint32_t* list_final = nullptr;             // points at the sorted ent_val of the last frame

    // per-frame scratch sized from max W x H
    uint2* ranges = nullptr;  // [tiles] per-tile ranges (debug export; produced by the tile-level binning)
    uint32_t* list_len = nullptr; // [tiles] retained lists: entries of each tile's list the rasterizer wrote (list_partial)
    bool bin_attr_set = false;    // bin_ordered.cu's function attributes set for this scene's device
    bool retain_lists = false;    // hyrf_set_retain_lists
    bool list_partial = false;    // the last frame's per-tile lists end at list_len (retained), not at their ranges (exported)
    uint2* mranges = nullptr; // [macro tiles] ranges into the macro-tile lists the rasterizer walks
    uint32_t* tile_queue = nullptr;  // [tiles] tile ids, longest list first (bin_ordered.cu -> raster.cu)
    float* fg = nullptr;      // [H][W][3] (debug only)
    float* finalT = nullptr;  // [H][W]
    float* image = nullptr;   // [H][W][3] for hyrf_render_host
    float* image2 = nullptr;  // second image of hyrf_render_host_async's double buffer
    cudaStream_t copy_stream = nullptr;       // device->host copies of hyrf_render_host_async
    cudaEvent_t ev_rendered[2] = {}, ev_copied[2] = {};
    bool slot_used[2] = {false, false};
    int host_slot = 0;
    uint8_t* bg_mask = nullptr;
    uint32_t* bg_list = nullptr;  // [H*W] pixels S6 has to shade, appended by the rasterizer

    FrameDev last_frame{};            // camera and frame constants of the last render (hyrf_backward)
    float* bwd_gT = nullptr;          // backward scratch: dL/dT [H][W], dL/d(projected record) [V][9], SSIM maps
    float* bwd_grec = nullptr;
    float* bwd_ssim = nullptr;
    uint32_t last_backward_launches = 0;
    int32_t strip_row0 = 0, strip_row1 = 0;   // hyrf_set_strip: pixel rows this device renders (equal: the whole image)

    // debug / measurement
    uint32_t ablation = 0;            // hyrf_ablation bits
    int macro_shift = 0;              // hyrf_set_bin_granularity: 0 auto, else macro tiles of 2^shift x 2^shift tiles
    int raster_mode = 0;              // hyrf_set_raster_mode: 0 auto, 1 tile-level lists only, 2 per-warp lists
    int last_raster_mode = 0;         // what the last hy_launch_raster picked
    uint32_t debug_mask = 0;
    float* dbg_raw = nullptr;         // [N][11]
    float* dbg_attrs = nullptr;       // [N][11]
    bool timing = false;
    cudaEvent_t ev[7] = {};           // [0..4] stage starts; [5], [6] frame ends, alternating by frame (ev_end)
    int ev_end = 5;                   // which of ev[5] / ev[6] closes the last frame
    bool last_timed = false;
    bool prev_timed = false;          // the frame before the last one was timed too (hyrf_frame_gap)
    cudaEvent_t ev_counters = nullptr;
    cudaStream_t sort_stream = nullptr;                  // the depth sort runs here, beside the field kernel
    bool sort_overlap = true;                            // hyrf_set_sort_overlap
    cudaEvent_t ev_culled = nullptr, ev_sorted = nullptr;
    bool ev_valid = false;
    uint32_t last_launches = 0;
    uint32_t lastV = 0;
    uint64_t lastD = 0, lastDm = 0;
    int32_t lastW = 0, lastH = 0;
    bool rendered = false;
};

// error reporting shared by all translation units
hyrf_status hy_fail(hyrf_status st, const char* fmt, ...);
hyrf_status hy_cuda_fail(cudaError_t e, const char* what);

// ---- launchers (each returns the number of kernels it enqueued through *launches) -------------------------
// decode of the compressed explicit Gaussians at upload (decode.cu); *first_bad must hold 0xFFFFFFFF
hyrf_status hy_launch_explicit_decode(hyrf_scene* s, const uint16_t* pos_h, const uint16_t* codes,
                                      const float* codebooks, uint32_t S, uint32_t K, uint32_t* first_bad);
// S1 (cull.cu): visibility bits, stable compactions -> vis_m (Morton work list), vis_idx + rank lookup (id order)
hyrf_status hy_prepare_morton(hyrf_scene* s);
void hy_launch_cull(hyrf_scene* s, const FrameDev& f, uint32_t* launches, cudaStream_t st, uint32_t* scan_scratch);
// S2 + S3 + S4a (field.cu): per visible Gaussian query both fields, aggregate, project
hyrf_status hy_launch_field(hyrf_scene* s, const FrameDev& f, uint32_t* launches);
// device-wide exclusive scan of n u32 (scan.cu); scratch must hold hy_scan_scratch_elems(n)
size_t hy_scan_scratch_elems(size_t n);
void hy_launch_scan(const uint32_t* in, uint32_t* out, size_t n, uint32_t* scratch, cudaStream_t st,
                    uint32_t* launches);
// stable LSD radix sort of (key, val) pairs on bits [0, key_bits) (radix.cu). n_dev: device count (may be null ->
// n_cap). Result ends in (*out_key, *out_val) which is either buffer pair. iota_vals: val_a is not read, the value of
// item i is i.
size_t hy_radix_hist_elems(size_t n_cap);
size_t hy_radix_max_items();
void hy_launch_radix(uint32_t* key_a, uint32_t* val_a, uint32_t* key_b, uint32_t* val_b, size_t n_cap,
                     const uint32_t* n_dev, int key_bits, uint32_t* hist, uint32_t* scan_scratch, cudaStream_t st,
                     uint32_t** out_key, uint32_t** out_val, uint32_t* launches, bool iota_vals = false,
                     uint32_t key_sub = 0);
// S4b-c (bin.cu)
void hy_launch_tiles_gather(hyrf_scene* s, const uint32_t* order, uint32_t V, uint32_t* launches);
void hy_launch_emit(hyrf_scene* s, const uint32_t* order, uint32_t V, uint32_t* launches);
void hy_launch_ranges(hyrf_scene* s, const uint32_t* keys, uint64_t D, uint32_t n_tiles, uint32_t* launches);
// S4b-c in one ordered counting pass (bin_ordered.cu), for frames of a bounded tile count; no host-side V or D
bool hy_bin_ordered_supported(uint32_t N, uint32_t n_tiles);
size_t hy_bin_ordered_ws_elems(uint32_t N, size_t cap, uint32_t max_tiles);
hyrf_status hy_launch_bin_ordered(hyrf_scene* s, const uint32_t* order, uint32_t n_tiles, uint32_t gx,
                                  uint32_t* launches, bool macro, uint32_t shift);
// S5 (raster.cu)
void hy_launch_raster(hyrf_scene* s, const FrameDev& f, const uint2* ranges, const uint32_t* list, bool macro,
                      float* out_rgb, uint32_t* launches, const uint32_t* tile_queue, uint32_t* dbg_list, uint32_t* dbg_len);
void hy_launch_raster_warp(hyrf_scene* s, const FrameDev& f, const uint2* ranges, const uint32_t* list, bool macro,
                           float* out_rgb, uint32_t* launches, const uint32_t* tile_queue, uint32_t* dbg_list, uint32_t* dbg_len);
void hy_launch_raster_pair(hyrf_scene* s, const FrameDev& f, const uint2* ranges, const uint32_t* list, bool macro,
                           float* out_rgb, uint32_t* launches, const uint32_t* tile_queue, uint32_t* dbg_list, uint32_t* dbg_len,
                           bool all = false);
// backward of S5 for the last frame (raster_backward.cu); needs the per-tile lists (s->ranges, s->list_final)
hyrf_status hy_launch_raster_backward(hyrf_scene* s, const float* g_cfg, const float* g_T, float* grad,
                                      uint32_t* launches);
// S6 (background.cu)
hyrf_status hy_launch_background(hyrf_scene* s, const FrameDev& f, float* out_rgb, uint32_t* launches);
