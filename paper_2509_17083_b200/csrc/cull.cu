// cull.cu — S1: visibility pre-culling against the camera frustum + order-preserving compaction.
// PAPER.md:112–122 (Eq. 8–9): eliminate points that will not project into the image frame BEFORE the neural
// fields are queried. Arithmetic: DESIGN.md §2 D1.
//
// The Gaussians are kept twice in HBM: as uploaded (id order, the order every list and tie-break is defined in) and
// as a 32-byte record in Morton order of the contracted position (built once at upload). The cull streams the
// Morton copy, so the visible set comes out spatially coherent — neighbouring lanes of the field kernel then gather
// from the same grid cells on the coarse and middle levels — while the visible RANK of a Gaussian (its slot in
// every later array) is still its rank in id order: the per-id visibility bytes are compacted a second time in id
// order, which yields vis_idx (ascending ids) and a rank lookup (word prefix + popcount) for the field kernel.
#include "scene.h"

namespace {

constexpr int kCullThreads = 256;
constexpr int kCullItems = 1024;  // per block: 4 coalesced sweeps of 256

// Morton code of the contracted position: 10 bits per axis
__device__ __forceinline__ uint32_t spread10(uint32_t v) {
    v &= 0x3FFu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__global__ void morton_code_kernel(const float* __restrict__ pos, uint32_t N, FrameDev f, uint32_t* __restrict__ code,
                                   uint32_t* __restrict__ id) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float x[3];
    hy_contract(f, pos[i], pos[N + i], pos[2ull * N + i], x);
    uint32_t q[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float v = x[a] == x[a] ? x[a] : 0.0f;
        q[a] = (uint32_t)fminf(v * 1024.0f, 1023.0f);
    }
    code[i] = spread10(q[0]) | (spread10(q[1]) << 1) | (spread10(q[2]) << 2);
    id[i] = i;
}

// max |p|^2 over the Gaussians, as the bits of a non-negative float (their integer order is the float order); NaN
// positions never win a comparison (they are never visible either: Eq. 9 is false for them)
__global__ void max_norm2_kernel(const float* __restrict__ pos, uint32_t N, uint32_t* __restrict__ out_bits) {
    float m = 0.0f;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const float x = pos[i], y = pos[N + i], z = pos[2ull * N + i];
        const float d = x * x + y * y + z * z;
        if (d > m) m = d;
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out_bits, __float_as_uint(m));
}

// gm[m] = (pos.xyz, scale | opacity, rgb) of the m-th Gaussian in Morton order; gm_id[m] = its id
__global__ void morton_gather_kernel(const uint32_t* __restrict__ order, const float* __restrict__ pos,
                                     const float* __restrict__ rgb, const float* __restrict__ scale,
                                     const float* __restrict__ opac, uint32_t N, float4* __restrict__ gm,
                                     uint32_t* __restrict__ gm_id) {
    const uint32_t m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    const uint32_t i = order[m];
    gm[2ull * m] = make_float4(pos[i], pos[N + i], pos[2ull * N + i], scale[i]);
    gm[2ull * m + 1] = make_float4(opac[i], rgb[i], rgb[N + i], rgb[2ull * N + i]);
    gm_id[m] = i;
}

// One launch, two sweeps of the same Eq. 9 test (same function, same fp32 inputs, hence the same bits):
// over the Morton records -> visibility bits + block counts in Morton order (the work list), and over the uploaded SoA
// -> visibility bits + block counts in id order (ranks, vis_idx). Recomputing the test on the 12 MB SoA is cheaper
// than scattering one byte per Gaussian from the Morton sweep into id order.
__device__ __forceinline__ bool d1_keep(const FrameDev& f, float px, float py, float pz) {
    float X, Y, Z;
    hy_to_camera(f, px, py, pz, X, Y, Z);
    const bool keep = (Z > f.z_near) && (fabsf(X) <= __fmul_rn(f.limx, Z)) && (fabsf(Y) <= __fmul_rn(f.limy, Z));
    return keep || (f.ablation & HYRF_ABL_NO_CULL);   // "w/o pre-culling": everything goes to the fields
}

__global__ void __launch_bounds__(kCullThreads)
cull_mark_kernel(const float4* __restrict__ gm, const float* __restrict__ pos, uint32_t N, FrameDev f,
                 uint32_t* __restrict__ m_words, uint32_t* __restrict__ m_counts, uint32_t* __restrict__ id_words,
                 uint32_t* __restrict__ id_counts) {
    __shared__ uint32_t warp_cnt[2][kCullThreads / 32];
    const uint32_t base = blockIdx.x * kCullItems;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t cnt_m = 0, cnt_i = 0;
#pragma unroll
    for (int k = 0; k < kCullItems / kCullThreads; ++k) {
        const uint32_t i = base + k * kCullThreads + threadIdx.x;
        bool keep_m = false, keep_i = false;
        if (i < N) {
            const float4 p = __ldg(gm + 2ull * i);
            keep_m = d1_keep(f, p.x, p.y, p.z);
            keep_i = d1_keep(f, __ldg(pos + i), __ldg(pos + N + i), __ldg(pos + 2ull * N + i));
        }
        const uint32_t bal_m = __ballot_sync(0xffffffffu, keep_m), bal_i = __ballot_sync(0xffffffffu, keep_i);
        if (lane == 0) {
            const uint32_t word = (base >> 5) + k * (kCullThreads / 32) + warp;
            if (word * 32u < N) { m_words[word] = bal_m; id_words[word] = bal_i; }
            cnt_m += __popc(bal_m);
            cnt_i += __popc(bal_i);
        }
    }
    if (lane == 0) { warp_cnt[0][warp] = cnt_m; warp_cnt[1][warp] = cnt_i; }
    __syncthreads();
    if (threadIdx.x < 2) {
        uint32_t sum = 0;
#pragma unroll
        for (int w = 0; w < kCullThreads / 32; ++w) sum += warp_cnt[threadIdx.x][w];
        (threadIdx.x ? id_counts : m_counts)[blockIdx.x] = sum;
    }
}

// Stable compaction of one bit array: out[rank] = index of the set bit; optionally word_rank[word] = rank of the
// word's first bit (the lookup the field kernel turns an id into its visible rank with).
// Sum of counts[0 .. blockIdx.x) by the whole block (when the host passed no scanned offsets): for the block counts
// of a few million Gaussians this is a handful of loads per thread and saves the scan launches.
__device__ __forceinline__ uint32_t block_offset(const uint32_t* __restrict__ counts, uint32_t* s_red /*[8]*/) {
    uint32_t sum = 0;
    for (uint32_t b = threadIdx.x; b < blockIdx.x; b += kCullThreads) sum += __ldg(counts + b);
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = sum;
    __syncthreads();
    uint32_t total = 0;
#pragma unroll
    for (int w = 0; w < kCullThreads / 32; ++w) total += s_red[w];
    return total;
}

// With `pos`: also depth_key[rank] = bits of the camera-space depth Z of that Gaussian (D1's Z, the key of the depth
// sort S4c). Z needs nothing from the fields, so the sort can start right after the cull, beside the field query.
__device__ __forceinline__ void compact_bits(const uint32_t* __restrict__ words, const uint32_t* __restrict__ block_offs,
                                             const uint32_t* __restrict__ block_counts, uint32_t N,
                                             uint32_t* __restrict__ out, uint32_t* __restrict__ word_rank,
                                             uint32_t* s_prefix /*[32]*/, uint32_t* s_red, uint32_t* boff_out,
                                             const float* __restrict__ pos = nullptr, const FrameDev* f = nullptr,
                                             uint32_t* __restrict__ depth_key = nullptr) {
    const uint32_t base = blockIdx.x * kCullItems;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t boff = block_offs ? block_offs[blockIdx.x] : block_offset(block_counts, s_red);
    *boff_out = boff;
    if (warp == 0) {  // 32 words per block: exclusive scan of their popcounts by one warp
        const uint32_t word = (base >> 5) + lane;
        const bool in = word * 32u < N;
        const uint32_t c = in ? __popc(words[word]) : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= (uint32_t)d) incl += v;
        }
        s_prefix[lane] = incl - c;
        if (word_rank && in) word_rank[word] = boff + incl - c;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kCullItems / kCullThreads; ++k) {
        const uint32_t wl = k * (kCullThreads / 32) + warp;
        const uint32_t word = (base >> 5) + wl;
        if (word * 32u >= N) continue;
        const uint32_t bits = words[word];
        if ((bits >> lane) & 1u) {
            const uint32_t rank = boff + s_prefix[wl] + __popc(bits & ((1u << lane) - 1u));
            const uint32_t i = base + k * kCullThreads + threadIdx.x;
            out[rank] = i;
            if (pos) {
                float X, Y, Z;
                hy_to_camera(*f, pos[i], pos[(size_t)N + i], pos[2 * (size_t)N + i], X, Y, Z);
                depth_key[rank] = __float_as_uint(Z);
            }
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kCullThreads)
cull_compact_kernel(const uint32_t* __restrict__ m_words, const uint32_t* __restrict__ m_offs,
                    const uint32_t* __restrict__ m_counts, const uint32_t* __restrict__ id_words,
                    const uint32_t* __restrict__ id_offs, const uint32_t* __restrict__ id_counts, uint32_t N,
                    uint32_t* __restrict__ vis_m, uint32_t* __restrict__ vis_idx, uint32_t* __restrict__ word_rank,
                    FrameCounters* __restrict__ counters, const float* __restrict__ pos, const FrameDev f,
                    uint32_t* __restrict__ depth_key) {
    __shared__ uint32_t s_prefix[kCullItems / 32];
    __shared__ uint32_t s_red[kCullThreads / 32];
    uint32_t boff_m, boff_i;
    compact_bits(m_words, m_offs, m_counts, N, vis_m, nullptr, s_prefix, s_red, &boff_m);
    compact_bits(id_words, id_offs, id_counts, N, vis_idx, word_rank, s_prefix, s_red, &boff_i, pos, &f, depth_key);
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        counters->V = boff_m + m_counts[blockIdx.x];
        counters->D = 0ull;
        counters->Dm = 0ull;
        counters->n_bg = 0u;
        counters->bin_ticket = 0u;
        counters->bin_done = 0u;
    }
}

}  // namespace

// Built once per hyrf_upload_params: Morton order of the contracted positions + the 32-byte records in that order.
hyrf_status hy_prepare_morton(hyrf_scene* s) {
    FrameDev f{};
    for (int a = 0; a < 3; ++a) {
        f.aabb_c[a] = 0.5f * (s->desc.aabb_min[a] + s->desc.aabb_max[a]);
        f.aabb_h[a] = 0.5f * (s->desc.aabb_max[a] - s->desc.aabb_min[a]);
    }
    const uint32_t N = s->N;
    morton_code_kernel<<<(N + 255) / 256, 256, 0, s->stream>>>(s->pos, N, f, s->sort_a_key, s->sort_a_val);
    uint32_t *key = nullptr, *order = nullptr, launches = 0;
    hy_launch_radix(s->sort_a_key, s->sort_a_val, s->sort_b_key, s->sort_b_val, N, nullptr, 30, s->hist, s->scan_scratch,
                    s->stream, &key, &order, &launches);
    morton_gather_kernel<<<(N + 255) / 256, 256, 0, s->stream>>>(order, s->pos, s->rgb, s->scale, s->opac, N, s->gm,
                                                                 s->gm_id);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return hy_cuda_fail(e, "hy_prepare_morton");
    // r_max = max |p|: every camera-space depth is then bounded on the host (|Z| <= |r3| r_max + |t_z|), which tells the
    // depth sort of a frame how many key bits it has to look at (api.cu)
    uint32_t bits = 0;
    uint32_t* word = s->block_counts;   // (the cull's scratch: idle during an upload)
    if ((e = cudaMemsetAsync(word, 0, sizeof(uint32_t), s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemsetAsync(r_max)");
    max_norm2_kernel<<<s->sm_count * 4, 256, 0, s->stream>>>(s->pos, N, word);
    if ((e = cudaMemcpyAsync(&bits, word, sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaMemcpyAsync(r_max)");
    if ((e = cudaStreamSynchronize(s->stream)) != cudaSuccess) return hy_cuda_fail(e, "cudaStreamSynchronize(r_max)");
    float n2;
    memcpy(&n2, &bits, sizeof(float));
    s->r_max = sqrt((double)n2) * (1.0 + 1e-6);
    return HYRF_OK;
}

void hy_launch_cull(hyrf_scene* s, const FrameDev& f, uint32_t* launches, cudaStream_t st, uint32_t* scan_scratch) {
    const uint32_t nb = (s->N + kCullItems - 1) / kCullItems;
    uint32_t* m_counts = s->block_counts;
    uint32_t* m_offs = s->block_counts + nb;
    uint32_t* id_counts = s->block_counts + 2 * nb;
    uint32_t* id_offs = s->block_counts + 3 * nb;
    cull_mark_kernel<<<nb, kCullThreads, 0, st>>>(s->gm, s->pos, s->N, f, s->flag_words, m_counts, s->id_words,
                                                         id_counts);
    ++*launches;
    const bool in_kernel = nb <= 8192;   // block offsets summed inside the compaction; beyond that, scan first
    if (!in_kernel) {
        hy_launch_scan(m_counts, m_offs, nb, scan_scratch, st, launches);
        hy_launch_scan(id_counts, id_offs, nb, scan_scratch, st, launches);
    }
    cull_compact_kernel<<<nb, kCullThreads, 0, st>>>(s->flag_words, in_kernel ? nullptr : m_offs, m_counts,
                                                            s->id_words, in_kernel ? nullptr : id_offs, id_counts, s->N,
                                                            s->vis_m, s->vis_idx, s->word_rank, s->counters, s->pos, f,
                                                            s->sort_a_key);
    ++*launches;
}
