// field_mma.cu — S2 + S3 + S4a fused, tensor-core path for fp16 parameters (BASELINE configs 3–5):
//   contraction (Eq. 2) -> grid encodes (Eq. 3) -> direction PE (Eq. 5) -> decoders (Eq. 4, 6, "fully-fused
//   MLP, 2 hidden layers x 64") -> aggregation (Eq. 7) -> EWA projection.
// B200 design: a CTA owns a tile of 128 visible Gaussians = the 128 TMEM lanes. 256 threads: warps 0–3 gather the
// geometry field, warps 4–7 the appearance field + PE. The gathers are bound by L1TEX wavefronts (one per distinct
// 128-B line per instruction, profiles/r1a_README.md), so a warp takes 16 Gaussians at a time with TWO lanes per
// Gaussian: lane l and lane l^16 fetch the x and x+1 corners, which share a line 31/32 of the time, in the same
// instruction — 4 wavefronts per (Gaussian, level) instead of 8. Features go registers -> TMEM
// (tcgen05.st, fp16 pairs) as the A operand; the weights sit in shared memory as the B operand (K-major core
// matrices); tcgen05.mma accumulates fp32 in TMEM; the epilogue (tcgen05.ld, ReLU, round to fp16, tcgen05.st)
// feeds the next layer without touching shared or global memory. Only the 48-byte projected record leaves the SM.
// The two decoders run as independent chains with their own mbarrier. Accumulation order inside an MMA is
// unspecified, so this path is compared with the oracle by tolerance, not bit for bit.
#include "field_common.cuh"
#include "field_tc_common.cuh"
#include "tcgen05.cuh"


namespace {

constexpr int kThreads = 256;
constexpr int kTile = 128;
constexpr int kTmemCols = 256;
constexpr uint32_t kColDg = 0, kColDa = 64, kColAg = 128, kColAa = 160;
// raw row-major [out][in] fp16 weights -> packed operand block
__global__ void pack_weights_kernel(const __half* __restrict__ geo, const __half* __restrict__ app,
                                    __half* __restrict__ packed) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= kPackedBytes / 2) return;
    packed[i] = __float2half(0.0f);
    struct Op { uint32_t off, N, Kp, n_real, k_real, src; bool app; };
    const Op ops[6] = {{kOffG1, 64, 32, 64, 32, 0, false},        {kOffG2, 64, 64, 64, 64, 64 * 32, false},
                       {kOffG3, 16, 64, 8, 64, 64 * 32 + 64 * 64, false}, {kOffA1, 64, 64, 64, 56, 0, true},
                       {kOffA2, 64, 64, 64, 64, 64 * 56, true},   {kOffA3, 16, 64, 3, 64, 64 * 56 + 64 * 64, true}};
    for (int o = 0; o < 6; ++o) {
        const Op& op = ops[o];
        const uint32_t lo = op.off / 2, hi = lo + op.N * op.Kp;
        if (i < lo || i >= hi) continue;
        const uint32_t r = i - lo;
        const uint32_t grp = r / (op.Kp * 8), rem = r % (op.Kp * 8);
        const uint32_t kc = rem / 64, n = grp * 8 + (rem % 64) / 8, k = kc * 8 + (rem % 8);
        if (n < op.n_real && k < op.k_real) packed[i] = (op.app ? app : geo)[op.src + n * op.k_real + k];
    }
}

// D3 for one level with two lanes per Gaussian: this lane blends the four corners whose x bit is xb; the partner
// lane (lane ^ 16) takes the other four; the sum of both (fp32) is rounded to a packed half2 feature pair.
template <bool U8>
__device__ __forceinline__ uint32_t gather_level_pair(const GridDev& g, uint32_t l, const float x[3], uint32_t xb) {
    const uint32_t N = g.res[l];
    const float Nf = (float)N;
    uint32_t ci[3];
    float w[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float u = __fmul_rn(x[a], Nf);
        int i = (int)floorf(u);
        i = min(i, (int)N - 1);
        ci[a] = (uint32_t)i;
        w[a] = __fsub_rn(u, (float)i);
    }
    const uint32_t vx = ci[0] + xb;
    uint32_t idx[4];
    if ((g.dense_mask >> l) & 1u) {
        const uint32_t n1 = N + 1u;
        const uint32_t b = vx + n1 * (ci[1] + n1 * ci[2]);
        idx[0] = b; idx[1] = b + n1; idx[2] = b + n1 * n1; idx[3] = b + n1 * n1 + n1;
    } else {
        const uint32_t hy0 = ci[1] * 2654435761u, hy1 = hy0 + 2654435761u;
        const uint32_t hz0 = ci[2] * 805459861u, hz1 = hz0 + 805459861u;
        idx[0] = (vx ^ hy0 ^ hz0) & g.table_mask; idx[1] = (vx ^ hy1 ^ hz0) & g.table_mask;
        idx[2] = (vx ^ hy0 ^ hz1) & g.table_mask; idx[3] = (vx ^ hy1 ^ hz1) & g.table_mask;
    }
    float2 v[4];
    if (U8) {   // D3': value = fma(code, step, min)
        const uchar2* tab = reinterpret_cast<const uchar2*>(g.table) + g.offset[l];
        const float2 q0 = g.q[l][0], q1 = g.q[l][1];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uchar2 c = __ldg(tab + idx[k]);
            v[k] = make_float2(__fmaf_rn((float)c.x, q0.y, q0.x), __fmaf_rn((float)c.y, q1.y, q1.x));
        }
    } else {
        const __half2* tab = reinterpret_cast<const __half2*>(g.table) + g.offset[l];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = __half22float2(__ldg(tab + idx[k]));
    }
    const float ax = xb ? w[0] : __fsub_rn(1.0f, w[0]);
    const float wy0 = __fsub_rn(1.0f, w[1]), wz0 = __fsub_rn(1.0f, w[2]);
    float a0 = 0.0f, a1 = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float wt = __fmul_rn(__fmul_rn(ax, (k & 1) ? w[1] : wy0), (k & 2) ? w[2] : wz0);
        a0 = __fmaf_rn(wt, v[k].x, a0);
        a1 = __fmaf_rn(wt, v[k].y, a1);
    }
    a0 = __fadd_rn(a0, __shfl_xor_sync(0xffffffffu, a0, 16));
    a1 = __fadd_rn(a1, __shfl_xor_sync(0xffffffffu, a1, 16));
    return pack_h2(a0, a1);
}

// both lanes of a pair end up with both fields' rounded feature pairs
template <bool U8>
__device__ __forceinline__ void gather_level_pair2(const GridDev& g, const GridDev& ga, const void* __restrict__ both,
                                                   uint32_t l, const float x[3], uint32_t xb, uint32_t& geo, uint32_t& app) {
    float g0, g1, a0, a1;
    gather_level_half2<U8>(g, ga, both, l, x, xb, g0, g1, a0, a1);
    g0 = __fadd_rn(g0, __shfl_xor_sync(0xffffffffu, g0, 16));
    g1 = __fadd_rn(g1, __shfl_xor_sync(0xffffffffu, g1, 16));
    a0 = __fadd_rn(a0, __shfl_xor_sync(0xffffffffu, a0, 16));
    a1 = __fadd_rn(a1, __shfl_xor_sync(0xffffffffu, a1, 16));
    geo = pack_h2(g0, g1);
    app = pack_h2(a0, a1);
}

// geo / app tables [entry][2] half -> one table [entry][4] half
__global__ void interleave_tables_kernel(const uint32_t* __restrict__ geo, const uint32_t* __restrict__ app, size_t n,
                                         uint2* __restrict__ both) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) both[i] = make_uint2(geo[i], app[i]);
}

// 8-bit tables: [entry][2] codes x 2 -> [entry][4] codes
__global__ void interleave_tables_u8_kernel(const uint16_t* __restrict__ geo, const uint16_t* __restrict__ app, size_t n,
                                            uint32_t* __restrict__ both) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) both[i] = (uint32_t)geo[i] | ((uint32_t)app[i] << 16);
}

template <bool U8>
__global__ void __launch_bounds__(kThreads, 2)
field_mma_kernel(const FieldArgs A, const uint4* __restrict__ packed_w, const void* __restrict__ both) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[2];
    __shared__ uint32_t tmem_slot;
    __shared__ float s_col[kTile][3];
    __shared__ uint32_t s_exch[2][4][16][16];   // [field sent][warp & 3][level][row & 15], interleaved-table path

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t chain = warp >> 2;                 // 0: geometry, 1: appearance
    const uint32_t row = threadIdx.x & (kTile - 1);   // Gaussian within the tile == TMEM lane
    for (uint32_t i = threadIdx.x; i < kPackedBytes / 16; i += kThreads)
        reinterpret_cast<uint4*>(smem)[i] = __ldg(packed_w + i);
    tc::fence_proxy_async_smem();
    if (warp == 0) tc::tmem_alloc<kTmemCols>(&tmem_slot);
    if (threadIdx.x == 32) {
        tc::mbar_init(&mbar[0], 1);
        tc::mbar_init(&mbar[1], 1);
        tc::fence_mbar_init();
    }
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    const uint32_t lane_base = ((warp & 3u) * 32u) << 16;
    const uint32_t tD = tmem + (chain ? kColDa : kColDg);
    const uint32_t tA = tmem + (chain ? kColAa : kColAg);
    const uint32_t sb = tc::smem_u32(smem);
    const uint32_t off1 = chain ? kOffA1 : kOffG1, off2 = chain ? kOffA2 : kOffG2, off3 = chain ? kOffA3 : kOffG3;
    const uint32_t k1 = chain ? 64u : 32u;            // padded K of layer 1
    constexpr uint32_t idesc64 = tc::idesc_f16_f32(128, 64), idesc16 = tc::idesc_f16_f32(128, 16);
    uint64_t* bar = &mbar[chain];
    uint32_t phase = 0;
    const bool leader = row == 0;
    const uint32_t V = A.counters->V;
    const GridDev& grid = chain ? A.app : A.geo;

    for (uint32_t tile = blockIdx.x; tile * kTile < V; tile += gridDim.x) {
        const uint32_t j = tile * kTile + row;
        const bool valid = j < V;
        Explicit ex{};
        float px = 0.0f, py = 0.0f, pz = 0.0f;
        uint32_t a[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) a[i] = 0u;
        float x[3] = {0.5f, 0.5f, 0.5f};
        if (valid) {
            ex = fetch_visible(A, j);
            px = ex.px; py = ex.py; pz = ex.pz;
            hy_contract(A.f, px, py, pz, x);
        }
        if (both) {
            // Interleaved tables: a warp gathers BOTH fields for 16 of its 32 rows (rows 16*chain .. 16*chain+15 of
            // the quadrant it shares with warp ^ 4), two lanes per Gaussian. Each lane keeps the word of its own
            // row and field; the words the partner warp needs go through shared memory.
            const uint32_t lane = threadIdx.x & 31u, xb = lane >> 4;
            const int src = (int)((chain << 4) | (lane & 15u));
            float xs[3];
            xs[0] = __shfl_sync(0xffffffffu, x[0], src);
            xs[1] = __shfl_sync(0xffffffffu, x[1], src);
            xs[2] = __shfl_sync(0xffffffffu, x[2], src);
            const bool own = xb == chain;
#pragma unroll
            for (int l = 0; l < 16; ++l) {
                uint32_t wg, wa;
                gather_level_pair2<U8>(A.geo, A.app, both, l, xs, xb, wg, wa);
                if (own) a[l] = chain ? wa : wg;
                else s_exch[chain][warp & 3u][l][lane & 15u] = chain ? wg : wa;
            }
            __syncthreads();
            if (!own) {
#pragma unroll
                for (int l = 0; l < 16; ++l) a[l] = s_exch[chain ^ 1u][warp & 3u][l][lane & 15u];
            }
        } else {   // separate tables: two lanes per Gaussian; half h covers rows 16h..16h+15 of this warp
            const uint32_t lane = threadIdx.x & 31u, xb = lane >> 4;
#pragma unroll
            for (uint32_t h = 0; h < 2; ++h) {
                const int src = (int)((h << 4) | (lane & 15u));
                float xs[3];
                xs[0] = __shfl_sync(0xffffffffu, x[0], src);
                xs[1] = __shfl_sync(0xffffffffu, x[1], src);
                xs[2] = __shfl_sync(0xffffffffu, x[2], src);
                const bool own = xb == h;
#pragma unroll
                for (int l = 0; l < 16; ++l) {
                    const uint32_t p = gather_level_pair<U8>(grid, l, xs, xb);
                    a[l] = own ? p : a[l];
                }
            }
        }
        if (valid) {
            if (chain) {
                dir_pe_packed(A.f, px, py, pz, a + 16);   // D4
            }
        }
        if (!valid) {
#pragma unroll
            for (int l = 0; l < 16; ++l) a[l] = 0u;
        }
        // ---- layer 1: A <- features, D = A W1^T ----
        tc::st_x16(tA + lane_base, a);
        if (chain) tc::st_x16(tA + lane_base + 16, a + 16);
        tc::wait_st();
        tc::fence_before_sync();
        asm volatile("bar.sync %0, 128;" ::"r"(1 + chain) : "memory");
        if (leader) {
            tc::fence_after_sync();
            for (uint32_t s = 0; s < k1 / 16; ++s)
                tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off1 + s * 256, 128, k1 * 16), idesc64, s);
            tc::commit(bar);
        }
        tc::mbar_wait(bar, phase); phase ^= 1;
        tc::fence_after_sync();
        // ---- layer 2: A <- relu(D) in fp16, D = A W2^T ----
        {
            uint32_t d[32];
            tc::ld_x32(tD + lane_base, d); tc::wait_ld();
            relu_pack32(d, a);
            tc::ld_x32(tD + lane_base + 32, d); tc::wait_ld();
            relu_pack32(d, a + 16);
        }
        tc::st_x16(tA + lane_base, a);
        tc::st_x16(tA + lane_base + 16, a + 16);
        tc::wait_st();
        tc::fence_before_sync();
        asm volatile("bar.sync %0, 128;" ::"r"(1 + chain) : "memory");
        if (leader) {
            tc::fence_after_sync();
            for (uint32_t s = 0; s < 4; ++s)
                tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off2 + s * 256, 128, 1024), idesc64, s);
            tc::commit(bar);
        }
        tc::mbar_wait(bar, phase); phase ^= 1;
        tc::fence_after_sync();
        // ---- output layer: A <- relu(D) in fp16, D[:, 0:16] = A W3^T ----
        {
            uint32_t d[32];
            tc::ld_x32(tD + lane_base, d); tc::wait_ld();
            relu_pack32(d, a);
            tc::ld_x32(tD + lane_base + 32, d); tc::wait_ld();
            relu_pack32(d, a + 16);
        }
        tc::st_x16(tA + lane_base, a);
        tc::st_x16(tA + lane_base + 16, a + 16);
        tc::wait_st();
        tc::fence_before_sync();
        asm volatile("bar.sync %0, 128;" ::"r"(1 + chain) : "memory");
        if (leader) {
            tc::fence_after_sync();
            for (uint32_t s = 0; s < 4; ++s)
                tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off3 + s * 256, 128, 1024), idesc16, s);
            tc::commit(bar);
        }
        tc::mbar_wait(bar, phase); phase ^= 1;
        tc::fence_after_sync();
        float raw[11];
        if (chain) {
            uint32_t o[4];
            tc::ld_x4(tD + lane_base, o); tc::wait_ld();
            s_col[row][0] = __uint_as_float(o[0]); s_col[row][1] = __uint_as_float(o[1]); s_col[row][2] = __uint_as_float(o[2]);
        } else {
            uint32_t o[8];
            tc::ld_x8(tD + lane_base, o); tc::wait_ld();
#pragma unroll
            for (int i = 0; i < 8; ++i) raw[i] = __uint_as_float(o[i]);
        }
        tc::fence_before_sync();
        __syncthreads();
        if (!chain && valid) {
            raw[8] = s_col[row][0]; raw[9] = s_col[row][1]; raw[10] = s_col[row][2];
            aggregate_project<true>(A, ex, raw);
        }
        __syncthreads();
        tc::fence_after_sync();
    }
    tc::fence_before_sync();
    __syncthreads();
    if (warp == 0) tc::tmem_dealloc<kTmemCols>(tmem);
}


// ---- software-pipelined variant for the interleaved tables ----------------------------------------------------------
// Same decoders, same arithmetic. The difference is WHEN the gathers are issued: the grid look-ups of tile t+1 are
// cut into three chunks that sit in the three windows where the warps of tile t would otherwise wait for their
// tcgen05.mma to complete (commit -> mbarrier). The decoder chain of a tile is ~5 us of mostly latency; hidden this way
// the kernel's time approaches that of the gathers alone.
template <bool U8>
__global__ void __launch_bounds__(kThreads, 2)
field_mma_pipe_kernel(const FieldArgs A, const uint4* __restrict__ packed_w, const void* __restrict__ both) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) uint64_t mbar[2];
    __shared__ uint32_t tmem_slot;
    __shared__ float s_col[kTile][3];
    __shared__ uint32_t s_exch[2][4][16][16];   // [field sent][warp & 3][level][row & 15]

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t chain = warp >> 2;                 // 0: geometry, 1: appearance
    const uint32_t row = threadIdx.x & (kTile - 1);   // Gaussian within the tile == TMEM lane
    for (uint32_t i = threadIdx.x; i < kPackedBytes / 16; i += kThreads)
        reinterpret_cast<uint4*>(smem)[i] = __ldg(packed_w + i);
    tc::fence_proxy_async_smem();
    if (warp == 0) tc::tmem_alloc<kTmemCols>(&tmem_slot);
    if (threadIdx.x == 32) {
        tc::mbar_init(&mbar[0], 1);
        tc::mbar_init(&mbar[1], 1);
        tc::fence_mbar_init();
    }
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    const uint32_t lane_base = ((warp & 3u) * 32u) << 16;
    const uint32_t tD = tmem + (chain ? kColDa : kColDg);
    const uint32_t tA = tmem + (chain ? kColAa : kColAg);
    const uint32_t sb = tc::smem_u32(smem);
    const uint32_t off1 = chain ? kOffA1 : kOffG1, off2 = chain ? kOffA2 : kOffG2, off3 = chain ? kOffA3 : kOffG3;
    const uint32_t k1 = chain ? 64u : 32u;            // padded K of layer 1
    constexpr uint32_t idesc64 = tc::idesc_f16_f32(128, 64), idesc16 = tc::idesc_f16_f32(128, 16);
    uint64_t* bar = &mbar[chain];
    uint32_t phase = 0;
    const bool leader = row == 0;
    const uint32_t V = A.counters->V;
    // gather role of this lane: rows 16*chain .. 16*chain+15 of the quadrant, two lanes per Gaussian
    const uint32_t xb = lane >> 4;
    const bool own = xb == chain;
    const int src = (int)((chain << 4) | (lane & 15u));
    uint32_t(*exch_out)[16] = s_exch[chain][warp & 3u];
    uint32_t(*exch_in)[16] = s_exch[chain ^ 1u][warp & 3u];

    auto fetch = [&](uint32_t tile, Explicit& e, bool& v, float xs[3]) {
        const uint32_t j = tile * kTile + row;
        v = j < V;
        float x[3] = {0.5f, 0.5f, 0.5f};
        e = Explicit{};
        if (v) {
            e = fetch_visible(A, j);
            hy_contract(A.f, e.px, e.py, e.pz, x);
        }
        xs[0] = __shfl_sync(0xffffffffu, x[0], src);
        xs[1] = __shfl_sync(0xffffffffu, x[1], src);
        xs[2] = __shfl_sync(0xffffffffu, x[2], src);
    };
#define HY_GATHER(L0, L1, XS, F)                                            \
    _Pragma("unroll") for (int l = (L0); l < (L1); ++l) {                   \
        uint32_t wg, wa;                                                    \
        gather_level_pair2<U8>(A.geo, A.app, both, l, XS, xb, wg, wa);                \
        if (own) F[l] = chain ? wa : wg;                                    \
        else exch_out[l][lane & 15u] = chain ? wg : wa;                     \
    }
    auto epilogue_to_A = [&]() {   // A <- relu(D) in fp16, 64 columns in two halves
        uint32_t d[32], pk[16];
        tc::ld_x32(tD + lane_base, d); tc::wait_ld();
        relu_pack32(d, pk);
        tc::st_x16(tA + lane_base, pk);
        tc::ld_x32(tD + lane_base + 32, d); tc::wait_ld();
        relu_pack32(d, pk);
        tc::st_x16(tA + lane_base + 16, pk);
        tc::wait_st();
        tc::fence_before_sync();
        asm volatile("bar.sync %0, 128;" ::"r"(1 + chain) : "memory");
    };

    uint32_t tile = blockIdx.x;
    if (tile * kTile < V) {
        Explicit ex;
        bool valid;
        float xs[3];
        uint32_t f[16];
        // prologue: the first tile's gathers are not hidden behind anything
        fetch(tile, ex, valid, xs);
        HY_GATHER(0, 16, xs, f)
        __syncthreads();
        if (!own) {
#pragma unroll
            for (int l = 0; l < 16; ++l) f[l] = exch_in[l][lane & 15u];
        }
        __syncthreads();
        for (;;) {
            const uint32_t next_tile = tile + gridDim.x;
            const bool has_next = next_tile * kTile < V;
            // ---- layer 1: A <- features (+ direction encoding), D = A W1^T ----
            {
                uint32_t a[16];
#pragma unroll
                for (int l = 0; l < 16; ++l) a[l] = valid ? f[l] : 0u;
                tc::st_x16(tA + lane_base, a);
                if (chain) {
#pragma unroll
                    for (int l = 0; l < 16; ++l) a[l] = 0u;
                    if (valid) {
                        dir_pe_packed(A.f, ex.px, ex.py, ex.pz, a);   // D4
                    }
                    tc::st_x16(tA + lane_base + 16, a);
                }
                tc::wait_st();
                tc::fence_before_sync();
                asm volatile("bar.sync %0, 128;" ::"r"(1 + chain) : "memory");
            }
            if (leader) {
                tc::fence_after_sync();
                for (uint32_t s = 0; s < k1 / 16; ++s)
                    tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off1 + s * 256, 128, k1 * 16), idesc64, s);
                tc::commit(bar);
            }
            // window 1: next tile's records, contraction, levels 0-5
            Explicit exn{};
            bool vn = false;
            float xsn[3] = {0.5f, 0.5f, 0.5f};
            uint32_t fn[16];
#pragma unroll
            for (int l = 0; l < 16; ++l) fn[l] = 0u;
            if (has_next) {
                fetch(next_tile, exn, vn, xsn);
                HY_GATHER(0, 6, xsn, fn)
            }
            tc::mbar_wait(bar, phase); phase ^= 1;
            tc::fence_after_sync();
            // ---- layer 2 ----
            epilogue_to_A();
            if (leader) {
                tc::fence_after_sync();
                for (uint32_t s = 0; s < 4; ++s)
                    tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off2 + s * 256, 128, 1024), idesc64, s);
                tc::commit(bar);
            }
            if (has_next) { HY_GATHER(6, 11, xsn, fn) }   // window 2
            tc::mbar_wait(bar, phase); phase ^= 1;
            tc::fence_after_sync();
            // ---- output layer ----
            epilogue_to_A();
            if (leader) {
                tc::fence_after_sync();
                for (uint32_t s = 0; s < 4; ++s)
                    tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + off3 + s * 256, 128, 1024), idesc16, s);
                tc::commit(bar);
            }
            if (has_next) { HY_GATHER(11, 16, xsn, fn) }  // window 3
            tc::mbar_wait(bar, phase); phase ^= 1;
            tc::fence_after_sync();
            float raw[11];
            if (chain) {
                uint32_t o[4];
                tc::ld_x4(tD + lane_base, o); tc::wait_ld();
                s_col[row][0] = __uint_as_float(o[0]); s_col[row][1] = __uint_as_float(o[1]); s_col[row][2] = __uint_as_float(o[2]);
            } else {
                uint32_t o[8];
                tc::ld_x8(tD + lane_base, o); tc::wait_ld();
#pragma unroll
                for (int i = 0; i < 8; ++i) raw[i] = __uint_as_float(o[i]);
            }
            tc::fence_before_sync();
            __syncthreads();
            if (!chain && valid) {
                raw[8] = s_col[row][0]; raw[9] = s_col[row][1]; raw[10] = s_col[row][2];
                aggregate_project<true>(A, ex, raw);
            }
            if (has_next && !own) {
#pragma unroll
                for (int l = 0; l < 16; ++l) fn[l] = exch_in[l][lane & 15u];
            }
            __syncthreads();
            tc::fence_after_sync();
            if (!has_next) break;
            tile = next_tile;
            ex = exn;
            valid = vn;
#pragma unroll
            for (int l = 0; l < 16; ++l) f[l] = fn[l];
        }
    }
#undef HY_GATHER
    tc::fence_before_sync();
    __syncthreads();
    if (warp == 0) tc::tmem_dealloc<kTmemCols>(tmem);
}


// ---- warp-autonomous variant (mma.sync) ------------------------------------------------------------------------------
// The decoders are 33 kFLOP per Gaussian: < 2 % of the tensor pipe either way. What the tcgen05 kernels above pay for
// is not throughput but hand-overs: TMEM round trips (tcgen05.st / ld + waits), one elected issuer, 128-thread
// barriers and an mbarrier wait per layer — ~7 us of latency per 128-Gaussian tile that only a second CTA and the
// gather windows can hide (0.112 ms of the 0.204 ms with the gathers removed). Here a WARP owns 32
// Gaussians end to end and never synchronises with another warp: gathers with two lanes per Gaussian (as above, two
// passes of 16), features -> the warp's own 6 KB of shared memory -> mma.sync m16n8k16 A fragments; the accumulator
// fragment of one layer IS the A fragment of the next after ReLU + rounding (registers only); weights are read from
// shared memory as pre-packed B fragments (one LDS.128 feeds four HMMA: two k-steps x the warp's two 16-row tiles);
// the 11 outputs return to one lane per Gaussian through shared memory for Eq. 7 and the projection. The 16 warps of
// an SM drift apart, so one warp's gathers (L1TEX) overlap another's decoders (tensor pipe, issue slots) by themselves.
constexpr uint32_t kWG1 = 0, kWG2 = 256, kWG3 = 768, kWA1 = 832, kWA2 = 1344, kWA3 = 1856, kWPackedU4 = 1920;   // uint4 offsets
constexpr uint32_t kRowG = 20, kRowA = 28;   // words per feature row: 16 (+4 pad) and 16 + 12 PE; both strides are conflict-free for fragment loads
constexpr uint32_t kWarpWords = 32 * kRowG + 32 * kRowA;
constexpr int kWThreads = 512;   // one CTA per SM: 16 warps share one copy of the weights
constexpr uint32_t kWarpSmemBytes = kWPackedU4 * 16 + (kWThreads / 32) * kWarpWords * 4;

// raw row-major [out][in] fp16 weights -> B fragments of mma.sync.m16n8k16 (col-major B = rows of W), two k-steps per
// uint4: lane (g = lane / 4, t = lane % 4) of n-tile j holds W[8j + g][16s + 2t, +1] and W[8j + g][16s + 8 + 2t, +1]
__global__ void pack_weights_hmma_kernel(const __half* __restrict__ geo, const __half* __restrict__ app,
                                         uint32_t* __restrict__ packed) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;   // one 32-bit word (two halves) each
    if (i >= kWPackedU4 * 4) return;
    struct Op { uint32_t off, NT, KP, n_real, k_real, src; bool app; };
    const Op ops[6] = {{kWG1, 8, 1, 64, 32, 0, false}, {kWG2, 8, 2, 64, 64, 64 * 32, false}, {kWG3, 1, 2, 8, 64, 64 * 32 + 64 * 64, false},
                       {kWA1, 8, 2, 64, 56, 0, true},  {kWA2, 8, 2, 64, 64, 64 * 56, true},  {kWA3, 1, 2, 3, 64, 64 * 56 + 64 * 64, true}};
    const uint32_t u4 = i >> 2, c = i & 3u;
    uint32_t out = 0;
    for (int o = 0; o < 6; ++o) {
        const Op& op = ops[o];
        if (u4 < op.off || u4 >= op.off + op.NT * op.KP * 32) continue;
        const uint32_t r = u4 - op.off, lane = r & 31u, jp = r >> 5, j = jp / op.KP, p = jp % op.KP;
        const uint32_t n = 8 * j + (lane >> 2), k = 16 * (2 * p + (c >> 1)) + 8 * (c & 1u) + 2 * (lane & 3u);
        const __half* W = (op.app ? app : geo) + op.src;
        const __half lo = (n < op.n_real && k < op.k_real) ? W[n * op.k_real + k] : __float2half(0.0f);
        const __half hi = (n < op.n_real && k + 1 < op.k_real) ? W[n * op.k_real + k + 1] : __float2half(0.0f);
        out = (uint32_t)__half_as_ushort(lo) | ((uint32_t)__half_as_ushort(hi) << 16);
    }
    packed[i] = out;
}

__device__ __forceinline__ void hmma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// one layer for the warp's two 16-row tiles: acc[t][j] = A_t (16 x 16 KS) W_j^T
template <int NT, int KS>
__device__ __forceinline__ void hmma_layer(const uint4* __restrict__ w, uint32_t lane, const uint32_t (&a)[2][KS][4],
                                           float (&acc)[2][NT][4]) {
#pragma unroll
    for (int j = 0; j < NT; ++j) {
#pragma unroll
        for (int t = 0; t < 2; ++t) acc[t][j][0] = acc[t][j][1] = acc[t][j][2] = acc[t][j][3] = 0.0f;
#pragma unroll
        for (int p = 0; p < KS / 2; ++p) {
            const uint4 b = w[(j * (KS / 2) + p) * 32 + lane];
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                hmma16816(acc[t][j], a[t][2 * p], b.x, b.y);
                hmma16816(acc[t][j], a[t][2 * p + 1], b.z, b.w);
            }
        }
    }
}

// ReLU + round to fp16: the accumulator fragments of n-tiles 2s, 2s+1 are the A fragment of k-step s
__device__ __forceinline__ void relu_to_A(const float (&acc)[2][8][4], uint32_t (&a)[2][4][4]) {
#pragma unroll
    for (int t = 0; t < 2; ++t)
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            a[t][s][0] = pack_h2(fmaxf(acc[t][2 * s][0], 0.0f), fmaxf(acc[t][2 * s][1], 0.0f));
            a[t][s][1] = pack_h2(fmaxf(acc[t][2 * s][2], 0.0f), fmaxf(acc[t][2 * s][3], 0.0f));
            a[t][s][2] = pack_h2(fmaxf(acc[t][2 * s + 1][0], 0.0f), fmaxf(acc[t][2 * s + 1][1], 0.0f));
            a[t][s][3] = pack_h2(fmaxf(acc[t][2 * s + 1][2], 0.0f), fmaxf(acc[t][2 * s + 1][3], 0.0f));
        }
}

template <bool U8>
__global__ void __launch_bounds__(kWThreads, 1)
field_warp_kernel(const FieldArgs A, const uint4* __restrict__ packed_w, const void* __restrict__ both) {
    extern __shared__ __align__(16) uint8_t smem[];
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    uint4* sw = reinterpret_cast<uint4*>(smem);
    for (uint32_t i = threadIdx.x; i < kWPackedU4; i += kWThreads) sw[i] = __ldg(packed_w + i);
    __syncthreads();
    uint32_t* fG = reinterpret_cast<uint32_t*>(smem + kWPackedU4 * 16) + warp * kWarpWords;   // [32][kRowG]; later out[32][12] floats
    uint32_t* fA = fG + 32 * kRowG;                                                           // [32][kRowA]
    float* out = reinterpret_cast<float*>(fG);
    const uint32_t V = A.counters->V;
    const uint32_t xb = lane >> 4, r16 = lane & 15u;
    const uint32_t g = lane >> 2, tg = lane & 3u;
    const uint32_t nwarps = gridDim.x * (kWThreads / 32);
    for (uint32_t wt = blockIdx.x * (kWThreads / 32) + warp; wt * 32u < V; wt += nwarps) {
        const uint32_t j = wt * 32u + lane;
        const bool valid = j < V;
        float x[3] = {0.5f, 0.5f, 0.5f};
        Explicit ex{};
        if (valid) {
            ex = fetch_visible(A, j);
            hy_contract(A.f, ex.px, ex.py, ex.pz, x);
        }
        // ---- grid encodes: two passes of 16 Gaussians, lanes l and l ^ 16 share one ----
#pragma unroll 1
        for (uint32_t h = 0; h < 2; ++h) {
            const int src = (int)(16u * h + r16);
            const float xs[3] = {__shfl_sync(0xffffffffu, x[0], src), __shfl_sync(0xffffffffu, x[1], src),
                                 __shfl_sync(0xffffffffu, x[2], src)};
            uint32_t* dst = xb ? fA + (16u * h + r16) * kRowA : fG + (16u * h + r16) * kRowG;
#pragma unroll
            for (int l = 0; l < 16; ++l) {   // fully unrolled: the loads of several levels are in flight together
                float g0, g1, a0, a1;
                gather_level_half2<U8>(A.geo, A.app, both, l, xs, xb, g0, g1, a0, a1);
                // the low lane keeps the geometry pair, the high lane the appearance pair: each sends what the other keeps
                const float s0 = xb ? g0 : a0, s1 = xb ? g1 : a1;
                const float k0 = xb ? a0 : g0, k1 = xb ? a1 : g1;
                const float f0 = __fadd_rn(k0, __shfl_xor_sync(0xffffffffu, s0, 16));
                const float f1 = __fadd_rn(k1, __shfl_xor_sync(0xffffffffu, s1, 16));
                dst[l] = pack_h2(f0, f1);
            }
        }
        // ---- direction encoding (Eq. 5), one lane per Gaussian ----
        {
            uint32_t pe2[12];
#pragma unroll
            for (int i = 0; i < 12; ++i) pe2[i] = 0u;
            if (valid) {
                dir_pe_packed(A.f, ex.px, ex.py, ex.pz, pe2);   // D4
            }
            uint4* d4 = reinterpret_cast<uint4*>(fA + lane * kRowA + 16);   // 112-byte rows: 16-byte aligned
            d4[0] = make_uint4(pe2[0], pe2[1], pe2[2], pe2[3]);
            d4[1] = make_uint4(pe2[4], pe2[5], pe2[6], pe2[7]);
            d4[2] = make_uint4(pe2[8], pe2[9], pe2[10], pe2[11]);
        }
        __syncwarp();
        float acc[2][8][4], o3[2][1][4];
        uint32_t a64[2][4][4];
        // ---- geometry decoder (Eq. 4): 32 -> 64 -> 64 -> 8 ----
        {
            uint32_t a32[2][2][4];
#pragma unroll
            for (int t = 0; t < 2; ++t)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const uint32_t* r0 = fG + (16 * t + g) * kRowG + 8 * s + tg;
                    a32[t][s][0] = r0[0]; a32[t][s][1] = r0[8 * kRowG]; a32[t][s][2] = r0[4]; a32[t][s][3] = r0[8 * kRowG + 4];
                }
            __syncwarp();   // fG is free from here: it becomes `out`
            hmma_layer<8, 2>(sw + kWG1, lane, a32, acc);
        }
        relu_to_A(acc, a64);
        hmma_layer<8, 4>(sw + kWG2, lane, a64, acc);
        relu_to_A(acc, a64);
        hmma_layer<1, 4>(sw + kWG3, lane, a64, o3);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            *reinterpret_cast<float2*>(out + (16 * t + g) * 12 + 2 * tg) = make_float2(o3[t][0][0], o3[t][0][1]);
            *reinterpret_cast<float2*>(out + (16 * t + g + 8) * 12 + 2 * tg) = make_float2(o3[t][0][2], o3[t][0][3]);
        }
        // ---- appearance decoder (Eq. 6): 32 + 24 -> 64 -> 64 -> 3 ----
#pragma unroll
        for (int t = 0; t < 2; ++t)
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const uint32_t* r0 = fA + (16 * t + g) * kRowA + 8 * s + tg;
                a64[t][s][0] = r0[0]; a64[t][s][1] = r0[8 * kRowA];
                if (s < 3) { a64[t][s][2] = r0[4]; a64[t][s][3] = r0[8 * kRowA + 4]; }
                else { a64[t][s][2] = 0u; a64[t][s][3] = 0u; }   // inputs 56..63 do not exist
            }
        hmma_layer<8, 4>(sw + kWA1, lane, a64, acc);
        relu_to_A(acc, a64);
        hmma_layer<8, 4>(sw + kWA2, lane, a64, acc);
        relu_to_A(acc, a64);
        hmma_layer<1, 4>(sw + kWA3, lane, a64, o3);
        if (tg < 2) {
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                *reinterpret_cast<float2*>(out + (16 * t + g) * 12 + 8 + 2 * tg) = make_float2(o3[t][0][0], o3[t][0][1]);
                *reinterpret_cast<float2*>(out + (16 * t + g + 8) * 12 + 8 + 2 * tg) = make_float2(o3[t][0][2], o3[t][0][3]);
            }
        }
        __syncwarp();
        // ---- Eq. 7 + projection, one lane per Gaussian ----
        float raw[11];
        {
            const float4* o4 = reinterpret_cast<const float4*>(out + lane * 12);
            const float4 q0 = o4[0], q1 = o4[1], q2 = o4[2];
            raw[0] = q0.x; raw[1] = q0.y; raw[2] = q0.z; raw[3] = q0.w; raw[4] = q1.x; raw[5] = q1.y; raw[6] = q1.z; raw[7] = q1.w;
            raw[8] = q2.x; raw[9] = q2.y; raw[10] = q2.z;
        }
        __syncwarp();   // `out` is fG again for the next tile
        if (valid) aggregate_project<true>(A, ex, raw);
    }
}

}  // namespace

bool hy_field_mma_supported(const hyrf_scene_desc& d) {
    return (d.param_dtype == HYRF_F16 || d.param_dtype == HYRF_U8) && d.geo_grid.levels == 16 && d.app_grid.levels == 16 && d.dir_pe_octaves == 4 &&
           d.geo_mlp.in_dim == 32 && d.geo_mlp.hidden == 64 && d.geo_mlp.n_hidden == 2 && d.app_mlp.in_dim == 56 &&
           d.app_mlp.hidden == 64 && d.app_mlp.n_hidden == 2;
}

// re-lay the uploaded weights out as tcgen05 B operands (called from hyrf_upload_params)
hyrf_status hy_field_mma_prepare(hyrf_scene* s) {
    pack_weights_kernel<<<(kPackedBytes / 2 + 255) / 256, 256, 0, s->stream>>>(
        reinterpret_cast<const __half*>(s->geo_mlp.w), reinterpret_cast<const __half*>(s->app_mlp.w),
        reinterpret_cast<__half*>(s->mma_w));
    pack_weights_hmma_kernel<<<(kWPackedU4 * 4 + 255) / 256, 256, 0, s->stream>>>(
        reinterpret_cast<const __half*>(s->geo_mlp.w), reinterpret_cast<const __half*>(s->app_mlp.w),
        reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(s->mma_w) + kPackedBytes));
    if (s->both_table) {
        const size_t n = s->geo_entries;
        if (s->u8)
            interleave_tables_u8_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(
                reinterpret_cast<const uint16_t*>(s->geo_grid.table), reinterpret_cast<const uint16_t*>(s->app_grid.table),
                n, reinterpret_cast<uint32_t*>(s->both_table));
        else
            interleave_tables_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(
                reinterpret_cast<const uint32_t*>(s->geo_grid.table), reinterpret_cast<const uint32_t*>(s->app_grid.table),
                n, reinterpret_cast<uint2*>(s->both_table));
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return hy_cuda_fail(e, "pack_weights_kernel");
    return HYRF_OK;
}

size_t hy_field_mma_packed_bytes() { return kPackedBytes + kWPackedU4 * 16; }   // tcgen05 operand block, then the mma.sync fragments

hyrf_status hy_launch_field_mma(hyrf_scene* s, const FrameDev& f, uint32_t* launches) {
    FieldArgs A;
    hy_fill_field_args(s, f, &A);
    bool& attr_set = s->field_attr_set;   // per scene (one device each; a scene is used by one thread at a time)
    if (!attr_set) {
        const void* ks[4] = {(const void*)field_mma_kernel<false>, (const void*)field_mma_kernel<true>,
                             (const void*)field_mma_pipe_kernel<false>, (const void*)field_mma_pipe_kernel<true>};
        for (const void* k : ks) {
            cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
            if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(field_mma)");
        }
        const void* kw[2] = {(const void*)field_warp_kernel<false>, (const void*)field_warp_kernel<true>};
        for (const void* k : kw) {
            cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kWarpSmemBytes);
            if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(field_warp)");
        }
        attr_set = true;
    }
    const int need = (int)((s->N + kTile - 1) / kTile);
    // CTA slots left to the depth sort running beside this kernel (hyrf_set_sort_overlap): with none, the persistent
    // CTAs hold every register of every SM and the sort waits for the kernel to end. Config 3, frame time against the
    // slots left free: 0 -> 0.586, 16 -> 0.563, 32 -> 0.551, 48 -> 0.561 ms (serial: 0.620 ms).
    const int gap = s->field_full_grid ? 0 : (32 * s->sm_count) / 148;
    const int slots = s->sm_count * 2 - gap;
    const int grid = need < slots ? need : slots;
    const uint4* w = reinterpret_cast<const uint4*>(s->mma_w);
    if (s->both_table && s->warp_mma) {
        const int needw = (int)((s->N + kWThreads - 1) / kWThreads);
        const int slotsw = s->sm_count - gap / 2;
        const int gridw = needw < slotsw ? needw : slotsw;
        const uint4* ww = reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(s->mma_w) + kPackedBytes);
        if (s->u8) field_warp_kernel<true><<<gridw, kWThreads, kWarpSmemBytes, s->stream>>>(A, ww, s->both_table);
        else field_warp_kernel<false><<<gridw, kWThreads, kWarpSmemBytes, s->stream>>>(A, ww, s->both_table);
    } else if (s->both_table) {
        if (s->u8) field_mma_pipe_kernel<true><<<grid, kThreads, kSmemBytes, s->stream>>>(A, w, s->both_table);
        else field_mma_pipe_kernel<false><<<grid, kThreads, kSmemBytes, s->stream>>>(A, w, s->both_table);
    } else {
        if (s->u8) field_mma_kernel<true><<<grid, kThreads, kSmemBytes, s->stream>>>(A, w, nullptr);
        else field_mma_kernel<false><<<grid, kThreads, kSmemBytes, s->stream>>>(A, w, nullptr);
    }
    ++*launches;
    return HYRF_OK;
}
