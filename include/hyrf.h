/*
 * hyrf.h — C-ABI of the B200-native HyRF hybrid forward render pass (arxiv 2509.17083, §3.2–3.3).
 *
 * One scene = explicit compact Gaussians + decoupled grid fields + tiny MLP decoders + background field
 * (PAPER.md:61–63, :124–126); one camera = R, t and an image frame; result = pixel colours
 * (PAPER.md:55 Eq. 1, :132 Eq. 11). Arithmetic of every stage: DESIGN.md §2.
 *
 * Conventions
 *  - Every call returns a hyrf_status and never throws, aborts or prints. On error, outputs are untouched and
 *    hyrf_last_error() describes the failure (thread-local string, never NULL).
 *  - Pointers in hyrf_params are DEVICE pointers unless host_ptrs != 0. The library copies; the caller keeps
 *    ownership of everything it passes in. hyrf_render's out_rgb is a DEVICE pointer; hyrf_render_host's is HOST.
 *  - hyrf_render enqueues the whole frame on the scene's stream, then waits for one 32-byte device→host readback
 *    of the frame's counters (visible count V, tile-entry count D; available once the field kernel has finished, while
 *    binning and rasterisation are still running). If D outgrew the list scratch, the scratch is grown and the frame is
 *    re-binned; otherwise nothing is allocated. The caller synchronises the stream before reading out_rgb.
 *  - One scene lives on one device. A scene is not thread-safe; the library is.
 *  - There is no CPU fallback anywhere: without a CUDA device every compute call returns HYRF_ERR_CUDA.
 */
#ifndef HYRF_H
#define HYRF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HYRF_MAX_LEVELS 16u
#define HYRF_MAX_WIDTH 64u /* widest MLP layer (inputs, hidden units) the kernels are compiled for */

typedef struct hyrf_scene hyrf_scene; /* opaque, library-owned */

typedef enum {
    HYRF_OK = 0,
    HYRF_ERR_INVALID_ARG = 1, /* NULL pointer, W/H outside [1, max], n_gaussians == 0 ... */
    HYRF_ERR_NOT_READY = 2,   /* render before the fields and the explicit Gaussians were uploaded; fetch / backward before a render */
    HYRF_ERR_UNSUPPORTED = 3, /* feats != 2, table not a power of two, dims beyond HYRF_MAX_* */
    HYRF_ERR_CAMERA = 4,      /* non-finite camera, or centre outside the background sphere */
    HYRF_ERR_OOM = 5,         /* device allocation failed, or D >= 2^32 */
    HYRF_ERR_CUDA = 6         /* any CUDA runtime failure, incl. no device */
} hyrf_status;

/* dtype of grid tables and MLP weights. HYRF_U8 is the compressed model of PAPER.md:227-229 (3): tables are 8-bit
 * min-max codes [entry][2] with value = fma(code, step, min) per level and feature (hyrf_params *_q), decoder
 * weights are fp16 and the decoded feature is rounded to fp16 as with HYRF_F16 (DESIGN.md §2 D3'). */
typedef enum { HYRF_F32 = 0, HYRF_F16 = 1, HYRF_U8 = 2 } hyrf_dtype;

/* How the MLP decoders are evaluated.
 *  FMA: CUDA-core fp32 fma in the oracle's order — geometry decisions bit-reproducible (any param_dtype).
 *  MMA: fp16 tensor cores with fp32 accumulation (param_dtype F16 / U8) — tcgen05, activations in TMEM, a CTA per
 *       128 Gaussians.
 *  HMMA: the same arithmetic on warp-level mma.sync, a warp per 32 Gaussians with no cross-warp hand-over (needs the
 *       two grids to share their geometry, as in every paper configuration; otherwise MMA runs).
 *  WS:   the MMA arithmetic (tcgen05, fp32 accumulation) as a warp-specialised pipeline: gather warps write the
 *        features into shared memory as tcgen05 A operands, decoder warpgroups consume them (needs the two grids to
 *        share their geometry; otherwise MMA runs).
 *  AUTO: WS (else MMA) when param_dtype is F16 / U8 and the layer shapes are supported, else FMA. */
typedef enum { HYRF_MLP_AUTO = 0, HYRF_MLP_FMA = 1, HYRF_MLP_MMA = 2, HYRF_MLP_HMMA = 3, HYRF_MLP_WS = 4 } hyrf_mlp_path;

/* Multi-resolution grid (layout DESIGN.md §2 D3). level_res is a HOST array. */
typedef struct {
    uint32_t levels;     /* 1..HYRF_MAX_LEVELS */
    uint32_t feats;      /* must be 2 ("feature of size 2") */
    uint32_t log2_table; /* hashed levels have 2^log2_table entries; <= 24 */
    const uint32_t* level_res;
} hyrf_grid_desc;

/* Decoder MLP: in_dim → hidden × n_hidden (ReLU) → out_dim (linear), no biases. */
typedef struct {
    uint32_t in_dim, hidden, n_hidden, out_dim;
} hyrf_mlp_desc;

typedef struct {
    uint32_t n_gaussians;
    float aabb_min[3], aabb_max[3]; /* scene box B0 used by the contraction */
    hyrf_grid_desc geo_grid, app_grid, bg_grid;
    hyrf_mlp_desc geo_mlp; /* in = 2*geo levels,            out = 8 (alpha_n, s_n[3], r_n[4]) — Eq. 4 */
    hyrf_mlp_desc app_mlp; /* in >= 2*app levels + 6*octaves, out = 3 (c_n)                     — Eq. 6 */
    hyrf_mlp_desc bg_mlp;  /* in >= 2*bg levels  + 6*octaves, out = 3 (background colour)       — Eq. 10 */
    uint32_t dir_pe_octaves; /* 4 */
    hyrf_dtype param_dtype;
    hyrf_mlp_path mlp_path;
    float cull_tol;  /* Eq. 9 tolerance band, default 0.1 */
    float z_near;    /* "too close to the image plane", default 0.2 */
    float bg_radius; /* background sphere radius, default 100 */
    float tau_T;     /* background composited where T > tau_T, default 0.2 */
    uint32_t max_width, max_height;
    int32_t device;
    /* optional allocator (e.g. torch-backed); NULL → cudaMalloc / cudaFree */
    void* (*alloc)(size_t bytes, void* user);
    void (*release)(void* ptr, void* user);
    void* user;
} hyrf_scene_desc;

typedef struct {
    const float* pos;           /* [3][N] SoA: x[N], y[N], z[N] — p_e (these four: all given, or all NULL, see hyrf_upload_params) */
    const float* rgb_logit;     /* [3][N] — c_e (pre-sigmoid) */
    const float* scale_logit;   /* [N]    — s_e (pre-sigmoid, isotropic) */
    const float* opacity_logit; /* [N]    — alpha_e (pre-sigmoid) */
    const void *geo_table, *app_table, *bg_table; /* levels concatenated, [entry][2], param_dtype */
    const void *geo_w, *app_w, *bg_w;             /* layers concatenated, each row-major [out][in] */
    const float *geo_q, *app_q, *bg_q;            /* HYRF_U8 only: [levels][2 features][2] = (min, step); else NULL */
    int32_t host_ptrs;                            /* 0: device pointers, else host pointers */
} hyrf_params;

/* Camera frame: +x right, +y down, +z forward; pixel (i, j) centre at integer coordinates. */
typedef struct {
    float R[9]; /* row-major world → camera */
    float t[3];
    float fx, fy, cx, cy;
} hyrf_camera;

/* Validates the descriptor, allocates every persistent device buffer (Gaussian SoA, tables, weights, per-frame
 * scratch sized from n_gaussians and max_width × max_height). */
hyrf_status hyrf_create_scene(const hyrf_scene_desc* desc, hyrf_scene** out);

/* Copies the parameters into library-owned buffers (H2D or D2D on the scene's stream) and re-lays the weights
 * out for the kernels. May be called again to replace the parameters. pos, rgb_logit, scale_logit and
 * opacity_logit may ALL be NULL when the explicit part arrives compressed through hyrf_upload_explicit_rvq; the
 * scene can be rendered once both the fields and the explicit part have been uploaded. */
hyrf_status hyrf_upload_params(hyrf_scene* scene, const hyrf_params* params);

/* Compressed explicit Gaussians (post-processing items (1) "point positions as half-precision
 * tensors" and (2) "residual vector quantization (R-VQ) ... [of the] explicit Gaussian properties"; arithmetic:
 * DESIGN.md §2 D1'). The Huffman layer of item (2) is an entropy code of these same integers and is undone by the
 * loader on the CPU before this call. All pointers are DEVICE pointers unless host_ptrs != 0; the caller keeps them.
 *   pos_h     [3][N] IEEE binary16 bit patterns of p_e, SoA like hyrf_params.pos          p_e = float(pos_h), exact
 *   codes     [stages][N] uint16, codes[s][i] < codebook_size
 *   codebooks [stages][codebook_size][5] float, columns (s_e, alpha_e, c_e[0], c_e[1], c_e[2])
 *   property row of Gaussian i = codebooks[0][codes[0][i]] + codebooks[1][codes[1][i]] + ... in binary32, added in
 *   stage order (left to right). */
typedef struct {
    const uint16_t* pos_h;
    uint32_t stages;        /* 1..16 */
    uint32_t codebook_size; /* 1..65536 */
    const uint16_t* codes;
    const float* codebooks;
    int32_t host_ptrs;
} hyrf_explicit_rvq;

/* Decodes the compressed explicit part on the GPU (one kernel over N, csrc/decode.cu) into the scene's own fp32
 * arrays, replacing whatever explicit parameters the scene held, and rebuilds the Morton-ordered records from them;
 * hyrf_render then runs exactly as after hyrf_upload_params. Synchronises the scene's stream. Errors:
 * HYRF_ERR_INVALID_ARG for NULL pointers, stages / codebook_size out of range, or a code >= codebook_size (the
 * message names the first such Gaussian; the explicit part is then undefined and the scene is not renderable until
 * a successful upload of it). */
hyrf_status hyrf_upload_explicit_rvq(hyrf_scene* scene, const hyrf_explicit_rvq* rvq);

/* Duration (ms, CUDA events on the scene's stream) of the decode kernel of the last hyrf_upload_explicit_rvq. */
hyrf_status hyrf_last_decode_time(hyrf_scene* scene, float* ms);

/* Stream all later work of this scene is enqueued on (a cudaStream_t). Default: the legacy stream 0. */
hyrf_status hyrf_set_stream(hyrf_scene* scene, void* cuda_stream);

/* The hybrid forward render pass, §3.2–3.3 in the order of PAPER.md:27:
 * (1) visibility pre-culling Eq. 8–9; (2) geometry + appearance field query Eq. 2–6; (3) aggregation Eq. 7;
 * (4) EWA projection, tile binning, depth order; (5) alpha blending Eq. 1; (6) background Eq. 10–11, 15–18.
 * out_rgb: DEVICE float [H][W][3]. */
hyrf_status hyrf_render(hyrf_scene* scene, const hyrf_camera* camera, int32_t W, int32_t H, float* out_rgb);

/* Same pass, HOST result: renders into a library-owned device image, copies it to out_rgb_host
 * (float [H][W][3], ideally pinned) and synchronises the stream. The end-to-end call bench.py's "e2e" times. */
hyrf_status hyrf_render_host(hyrf_scene* scene, const hyrf_camera* camera, int32_t W, int32_t H,
                             float* out_rgb_host);

/* Pipelined variant for a stream of frames: returns as soon as the frame is enqueued (and its counters are known);
 * the device->host copy of the image runs on a second stream and overlaps the next hyrf_render_host_async. Two
 * frames may be in flight, so the caller alternates between (at least) two host buffers and calls hyrf_host_sync
 * before reading them. hyrf_host_sync waits for every render and copy enqueued so far. */
hyrf_status hyrf_render_host_async(hyrf_scene* scene, const hyrf_camera* camera, int32_t W, int32_t H,
                                   float* out_rgb_host);
hyrf_status hyrf_host_sync(hyrf_scene* scene);

hyrf_status hyrf_destroy_scene(hyrf_scene* scene);

const char* hyrf_last_error(void);

/* ---- parity / measurement exports (not on the hot path) ------------------------------------------------ */

typedef enum {
    HYRF_DBG_VIS_MASK = 0,    /* u8  [N] */
    HYRF_DBG_VIS_IDX = 1,     /* u32 [V] ascending Gaussian ids */
    HYRF_DBG_STAGE2_RAW = 2,  /* f32 [V][11] (alpha_n, s_n[3], r_n[4], c_n[3]) */
    HYRF_DBG_STAGE3_ATTRS = 3,/* f32 [V][11] (s[3], r[4] wxyz, alpha, c[3]) */
    HYRF_DBG_PROJ = 4,        /* f32 [V][10] (u, v, depth, A, B, C, opacity, r, g, b) */
    HYRF_DBG_RECT = 5,        /* u32 [V][4] (x0, x1, y0, y1), all zero when dropped */
    HYRF_DBG_TILE_RANGES = 6, /* u32 [tiles][2] [start, end) into the tile list */
    HYRF_DBG_TILE_LIST = 7,   /* u32 [D] Gaussian ids ordered by (tile, depth bits, id) */
    HYRF_DBG_FINAL_T = 8,     /* f32 [H][W] residual transmittance after stage 5 */
    HYRF_DBG_BG_MASK = 9,     /* u8  [H][W] 1 where the background was composited */
    HYRF_DBG_COUNTERS = 10,   /* u64 [5]: N, V, D (sum of tiles touched), tiles, Dm (macro-tile entries binned) */
    HYRF_DBG_FG = 11,         /* f32 [H][W][3] foreground colour C_fg before stage 6 */
    HYRF_DBG_EXPLICIT = 12    /* f32 [8][N]: rows p_e.x, p_e.y, p_e.z, s_e, alpha_e, c_e[0..2] as the scene holds them
                                 (needs no render and no hyrf_debug_enable: what the uploads left in the scene) */
} hyrf_debug_kind;

/* mask bit k enables retention of kind k for later fetches (STAGE2_RAW / STAGE3_ATTRS / BG_MASK / FG cost extra writes
 * in the kernels; TILE_RANGES / TILE_LIST make the pass materialise the per-tile lists, which it otherwise keeps per
 * 4 x 4-tile macro tile: the ranges come from a tile-level run of the binning, the lists are written by the
 * rasterizer as it consumes them; everything else is retained anyway). */
hyrf_status hyrf_debug_enable(hyrf_scene* scene, uint32_t mask);

/* Synchronises the stream and copies data of the LAST render to host_dst. *bytes receives the size needed; if it
 * exceeds cap nothing is copied and HYRF_ERR_INVALID_ARG is returned (host_dst may be NULL to query the size). */
hyrf_status hyrf_debug_fetch(hyrf_scene* scene, uint32_t kind, void* host_dst, size_t cap, size_t* bytes);

/* CUDA-event times (ms) of the last render's stages 1..6 (S1 cull; S2+S3+S4a field query, aggregation and
 * projection — one fused kernel; S4b–c binning and ordering; S5 rasterise; S6 background; [5] = whole frame).
 * Timing is recorded only after hyrf_debug_enable or hyrf_set_timing(scene, 1). Synchronises the stream. */
hyrf_status hyrf_set_timing(hyrf_scene* scene, int32_t enabled);
hyrf_status hyrf_stage_times(hyrf_scene* scene, float ms[6]);
/* Time (ms) the caller's stream spent between the end of the previous timed frame's last kernel and the start of the
 * last frame's first stage: what a stream of frames loses between frames (host enqueue latency, joins). Needs two
 * consecutive timed renders, else HYRF_ERR_NOT_READY. */
hyrf_status hyrf_frame_gap(hyrf_scene* scene, float* ms);

/* Ablation switches of the same pass (PAPER.md:214-223 Table 5, :233-237, :259-261). mask = OR of:
 *  NO_CULL:     the fields are queried and aggregated for every stored Gaussian; those failing Eq. 9 are dropped at
 *               projection instead (zero record, zero tiles), so the image is unchanged and only the cost moves
 *               (the paper's "w/o pre-culling", 27 vs 106 FPS);
 *  NO_BG:       no background compositing (out = C_fg);
 *  NO_NEURAL:   decoder outputs taken as 0: explicit isotropic, diffuse Gaussians only (no field query at all);
 *  NO_EXPLICIT: s_e = alpha_e = c_e = 0 in Eq. 7 (positions stay explicit).
 * A single shared field needs no switch: upload the same table for geo and app. Default 0 = the full model. */
typedef enum {
    HYRF_ABL_NO_CULL = 1, HYRF_ABL_NO_BG = 2, HYRF_ABL_NO_NEURAL = 4, HYRF_ABL_NO_EXPLICIT = 8
} hyrf_ablation;
hyrf_status hyrf_set_ablation(hyrf_scene* scene, uint32_t mask);

/* Scheduling of the depth sort (S4c; "ordered by depth"). Its keys, the camera-space depths, depend on
 * the explicit positions only, so by default (on != 0) the sort runs on a library-owned second stream BESIDE the
 * field query (S2), which leaves a few SMs to it (16 by default; on > 1: that many), and joins the frame before the
 * binning. on == 0 serialises the frame on the caller's stream (one kernel at a time: what per-kernel profiling
 * wants). The image and every debug export are identical either way. */
hyrf_status hyrf_set_sort_overlap(hyrf_scene* scene, int on);

/* Screen-strip parallelism over several devices: every device holds the whole scene and runs
 * S1-S3 and the projection for the whole frame (a Gaussian's reach is known only after its fields have been queried),
 * but bins, rasterises and composites only the pixel rows [row_begin, row_end) of out_rgb; the other rows of out_rgb are
 * left untouched. row_begin must be a multiple of 16 (the tile size), row_end a multiple of 16 or >= H. The rows a
 * device writes are bit-identical to the same rows of the whole-image render, so the strips of G devices, exchanged by
 * ONE all-gather of H/G x W x 3 floats, are the single-device image. row_begin == row_end (default 0, 0): whole image. */
hyrf_status hyrf_set_strip(hyrf_scene* scene, int32_t row_begin, int32_t row_end);

/* Frame pipelining for a STREAM of hyrf_render calls (hyrf_render_host_async always works this way). S1 and the depth
 * sort of a frame depend on the camera and the explicit positions only and write library-owned, double-buffered
 * scratch, so with on != 0 they are enqueued on the library's own high-priority stream WITHOUT waiting for what the
 * caller's stream still holds: frame k+1's cull and sort run beside frame k's rasterizer, and its field kernel then
 * takes every SM. Everything that touches out_rgb stays on the caller's stream, in order; images are bit-identical.
 * Default off: each hyrf_render starts behind all work enqueued before it (what a per-frame timing bracket on the
 * caller's stream must see). Needs hyrf_set_sort_overlap on (the default). */
hyrf_status hyrf_set_pipelining(hyrf_scene* scene, int on);

/* Rasterizer variant (S5; Eq. 1). Every variant stages a tile's depth-ordered list once per tile and
 * produces the same bits; they differ in cost. mode 1: a pixel per thread, every warp of the tile blends every staged
 * entry. mode 2: a warp owns an 8 x 4 pixel block and blends only the entries that can reach alpha >= 1/255 somewhere
 * in its block (per-warp lists built while staging). mode 3: per-warp lists over 8 x 8 blocks with two pixels per lane
 * on the two-wide fp32 instructions of sm_100 (fma.rn.f32x2: half the issue slots per pair) — fastest while splats
 * cover few tiles. mode 4: the two-pixel loop of mode 3 over every staged entry, without masks and lists — fastest when
 * a splat covers ~100 tiles (4K frames). mode 0 (default): 3 or 4, chosen per frame from the tiles touched per visible
 * Gaussian of the previous frame. HYRF_ERR_INVALID_ARG for any other mode. */
hyrf_status hyrf_set_raster_mode(hyrf_scene* scene, int mode);
/* Granularity of the binning (S4b): on tile grids of more than 1024 tiles the per-tile lists are not
 * materialised; Gaussians are binned into MACRO tiles of 2^shift x 2^shift tiles and the rasterizer picks each tile's
 * subsequence out of its macro tile's depth-ordered list. shift 0 (default): chosen per frame from the tiles touched per
 * visible Gaussian of the previous frame (2, 3 or 4: the larger the splats, the coarser); 1 .. 4: fixed. The image and
 * every debug export are identical for every value. HYRF_ERR_INVALID_ARG otherwise. */
hyrf_status hyrf_set_bin_granularity(hyrf_scene* scene, int shift);

/* The variant (1 .. 4) the last render used. */
hyrf_status hyrf_last_raster_mode(hyrf_scene* scene, int* mode);

/* Backward of stage 5 for the LAST rendered frame (first piece of the training pass of PAPER.md:136-142, which
 * back-propagates through the rasterizer the paper defers to, :108; arithmetic DESIGN.md §2 D12). With the frame's
 * blending decisions frozen, C_fg and the final transmittance T of every pixel are differentiable in the projected
 * records. g_cfg: DEVICE float [H][W][3] = dL/dC_fg; g_T: DEVICE float [H][W] = dL/dT (how a loss on the composited
 * image reaches the foreground: out = C_fg + T c_s). grad: DEVICE float [V][9], row = visible rank (HYRF_DBG_VIS_IDX
 * order), columns dL/d(u, v, A, B, C, opacity, r, g, b); overwritten. Enqueued on the scene's stream; the caller
 * synchronises. grad_rows: rows grad holds; fewer than the frame's V: HYRF_ERR_INVALID_ARG, nothing is written. The
 * frame must have kept its per-tile lists (hyrf_set_retain_lists, or the debug export HYRF_DBG_TILE_LIST |
 * HYRF_DBG_TILE_RANGES), else HYRF_ERR_NOT_READY. Sums use fp32 atomics: the result is reproducible to rounding, not
 * bit for bit. */
hyrf_status hyrf_raster_backward(hyrf_scene* scene, const float* g_cfg, const float* g_T, float* grad, uint64_t grad_rows);

/* Training mode of the forward pass: with on != 0 every hyrf_render keeps what the backward entry points need — the
 * per-tile ranges (one extra, count-only run of the binning at tile level) and each tile's list as the rasterizer
 * consumed it, up to the entry at which all of the tile's pixels had terminated (the rasterizer keeps its early exit;
 * nothing behind that entry was blended, so no gradient flows there). Separate from the debug export, which writes
 * every list to its end, disables the early exit and is meant for parity tests. The image is bit-identical. Costs one
 * host wait for the frame's counters before the binning (the list buffer is grown first if need be). Default off. */
hyrf_status hyrf_set_retain_lists(hyrf_scene* scene, int on);

/* ---- microprobes ("L2 gather throughput and sustained issue rate are not in MEASURED_PEAKS.json —
 * measure them with two microprobes first and commit the numbers"). Not on the render path; no scene needed. ------- */

/* Scattered look-ups of entry_bytes (4 or 8) from a table of table_bytes (power of two; 32-64 MB stays L2-resident)
 * — the access pattern of the grid gathers of S2 (Eq. 3). ctas_per_sm x 256 threads per SM, 8 independent
 * look-ups in flight per lane, iters x 8 look-ups per lane. share = 1 / 2 / 4 lanes read the same 32-byte sector
 * (2 = the two-lane gather of the field kernel); line = 1 packs four sectors of one instruction into one 128-byte
 * line. Outputs: lane look-ups per second, distinct sectors per second, best kernel time (ms, CUDA events). */
hyrf_status hyrf_probe_gather(int32_t device, uint64_t table_bytes, uint32_t entry_bytes, uint32_t ctas_per_sm,
                              uint32_t share, uint32_t line, uint32_t iters, double* lookups_per_s,
                              double* sectors_per_s, float* ms);

/* Sustained issue rate of dependent-free fp32 code: kind 0 FFMA only, 1 FFMA + integer ALU (two pipes), 2 the
 * instruction mix of the alpha-blend loop of S5 (Eq. 1: fp32 ops + one MUFU.EX2 + compares / selects per
 * pair). Output: warp instructions per second over the whole GPU (x 32 = lane slots per second). */
hyrf_status hyrf_probe_issue(int32_t device, uint32_t kind, uint32_t ctas_per_sm, uint32_t iters,
                             double* warp_instr_per_s, float* ms);

/* The whole backward pass for the LAST rendered frame (§3.4; arithmetic DESIGN.md §2 D13): given
 * g_out = dL/d out_rgb (DEVICE float [H][W][3]), the gradients of L with respect to every parameter of the scene, with
 * the forward's decisions frozen: S6 (background composite, Eq. 10-11) -> S5 (alpha blend, hyrf_raster_backward's
 * kernel) -> S4a (EWA projection) -> S3 (Eq. 7) -> S2 (decoders Eq. 4, 6; direction encoding Eq. 5; grid encodes Eq. 3;
 * contraction Eq. 2). Every pointer of hyrf_grads is a DEVICE float array shaped like the parameter it belongs to
 * (tables and weights in fp32 whatever the scene's param_dtype; 8-bit tables: gradient with respect to the decoded
 * values), or NULL when that gradient is not wanted. Gradients are ADDED to what the arrays hold (the caller zeroes
 * them, or accumulates several cameras). Enqueued on the scene's stream; the caller synchronises. Like
 * hyrf_raster_backward it needs a frame that kept its per-tile lists (hyrf_set_retain_lists or the debug export), else
 * HYRF_ERR_NOT_READY. Sums use fp32 atomics: reproducible to rounding, not bit for bit. */
typedef struct {
    float* pos;           /* [3][N] */
    float* rgb_logit;     /* [3][N] */
    float* scale_logit;   /* [N] */
    float* opacity_logit; /* [N] */
    float *geo_table, *app_table, *bg_table; /* [entries][2] */
    float *geo_w, *app_w, *bg_w;             /* layers concatenated, row-major [out][in] */
} hyrf_grads;
hyrf_status hyrf_backward(hyrf_scene* scene, const float* g_out, const hyrf_grads* grads);

/* The training loss of PAPER.md:138-140 Eq. 12 (reading A28): L = (1 - lambda) mean|image - target| +
 * lambda (1 - SSIM(image, target)), SSIM with an 11 x 11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2,
 * C2 = 0.03^2. image, target: DEVICE float [H][W][3]; *loss_host receives L; g_image (DEVICE float [H][W][3], may be
 * NULL) receives dL/d image — what hyrf_backward takes as g_out. Synchronises the scene's stream. */
hyrf_status hyrf_loss_l1_ssim(hyrf_scene* scene, const float* image, const float* target, int32_t W, int32_t H,
                              float lambda, double* loss_host, float* g_image);

/* The same loss through an entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid it). Needs no scene: device = CUDA device ordinal
 * (0 .. 63), cuda_stream = the cudaStream_t (as void*) the work is enqueued on and that is synchronised before the call
 * returns; the other arguments, the arithmetic and the result are hyrf_loss_l1_ssim's. The scratch (the loss
 * accumulator and three derivative maps of 3 W H floats each) is a file-scope device array of
 * 4 + 9 HYRF_LOSS_NOALLOC_MAX_PIXELS floats (37.7 MB) that every GPU which loads the library holds until the process
 * exits. Limit: W * H <= HYRF_LOSS_NOALLOC_MAX_PIXELS (2^20: covers 1280 x 720 and 1245 x 825); larger images are
 * rejected with HYRF_ERR_INVALID_ARG before anything is enqueued — use hyrf_loss_l1_ssim for those. The call performs
 * no cudaMalloc / cudaFree and calls no allocating library routine. All calls on a device SHARE the array: it keeps
 * the last call's contents (the call clears the accumulator and rewrites the maps before reading them), and two calls
 * whose GPU work overlaps (different streams, different host threads) race on it — serialise them. */
#define HYRF_LOSS_NOALLOC_MAX_PIXELS (1u << 20)
hyrf_status hyrf_loss_l1_ssim_noalloc(int32_t device, void* cuda_stream, const float* image, const float* target,
                                      int32_t W, int32_t H, float lambda, double* loss_host, float* g_image);

/* Number of kernels the last render launched (for bench.py's gpu_launches). */
hyrf_status hyrf_last_launch_count(hyrf_scene* scene, uint32_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* HYRF_H */
