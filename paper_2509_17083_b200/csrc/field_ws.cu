// field_ws.cu — S2 + S3 + S4a fused, tensor-core path, WARP-SPECIALISED (HYRF_MLP_WS): the same arithmetic as
// field_mma.cu's kernels (contraction Eq. 2 -> grid encodes Eq. 3 -> direction PE Eq. 5 -> decoders Eq. 4, 6 ->
// aggregation Eq. 7 -> EWA projection), organised as a producer / consumer pipeline inside one
// persistent CTA per SM.
//
// Why: the stage is bound by the LATENCY of its table gathers, not by any throughput (profiles/r1h: L1TEX 45-50 %,
// issue slots 46 %, top stall long_scoreboard, 14 warps resident). In field_mma.cu every warp alternates between
// gathering and decoding and carries both phases' state (128 registers, 16 warps per SM), so few loads are in
// flight. Here the roles are separate warps:
//   * 12 GATHER warps do nothing but table look-ups (two lanes per Gaussian, 16 Gaussians per instruction, the
//     dense / hashed choice of a level a template constant where the scene allows). Their only state is the
//     contracted position and a rolling window of 4 levels (16 loads per lane in flight: field_tc_common.cuh's
//     level_issue / level_consume). Features are written straight into shared memory in the K-major core-matrix
//     layout of a tcgen05 A operand (one 16-byte store per 4 levels).
//   * 2 DECODER warpgroups (128 threads = the 128 TMEM lanes each) take turns on tiles of 128 Gaussians: fetch the
//     explicit records and contract the positions two tiles ahead (the gather warps' input), then, when a tile's
//     features are complete, issue layer 1 with BOTH operands from shared memory (tcgen05.mma SS form: no register or
//     TMEM staging of the features), run the hidden layers with the activations in TMEM as in field_mma.cu, and
//     finish with Eq. 7 and the projection. Geometry and appearance chains interleave, so one chain's epilogue
//     covers the other's MMA latency.
// Hand-overs are mbarriers: ready[kNP] (positions of a tile available), full[kNF] (a tile's features written;
// 8 sixteen-row groups arrive), free[kNF] (the layer-1 MMAs that read a feature buffer have completed: tcgen05.commit),
// and one mbarrier per chain and warpgroup for the MMA completions.
#include "field_common.cuh"
#include "field_tc_common.cuh"
#include "tcgen05.cuh"

namespace {

constexpr int kTile = 128;
#ifndef HY_WS_GATHER_WARPS
#define HY_WS_GATHER_WARPS 12
#endif
#ifndef HY_WS_NF
#define HY_WS_NF 2
#endif
constexpr int kGatherWarps = HY_WS_GATHER_WARPS;        // a multiple of 4: decoder warp w then owns TMEM lanes 32 (w % 4) ..
constexpr int kDecWGs = 2;
constexpr int kWsThreads = (kGatherWarps + 4 * kDecWGs) * 32;   // 640
constexpr int kNF = HY_WS_NF;                           // feature buffers in flight
constexpr int kNP = 4;                                  // position / explicit-record buffers in flight
constexpr uint32_t kWsTmemCols = 512;
constexpr uint32_t kWgCols = 256;                       // per decoder warpgroup: D_geo 0, D_app 64, A_geo 128, A_app 160
// dynamic shared memory (bytes)
constexpr uint32_t kFeatBytes = 16384;                  // geometry features [128 x 32] fp16 | appearance features [128 x 32]
constexpr uint32_t kPeBytes = 8192;                     // direction encoding [128 x 32] fp16 (24 used), per decoder warpgroup
constexpr uint32_t kXBytes = 3 * kTile * 4, kExBytes = 9 * kTile * 4;
constexpr uint32_t kSmFeat = kPackedBytes;
constexpr uint32_t kSmPe = kSmFeat + kNF * kFeatBytes;
constexpr uint32_t kSmX = kSmPe + kDecWGs * kPeBytes;
constexpr uint32_t kSmEx = kSmX + kNP * kXBytes;
constexpr uint32_t kWsSmemBytes = kSmEx + kNP * kExBytes;   // 122,880

// byte offset of row r, 16-byte chunk c (8 consecutive K) in a [128 x 32] K-major core-matrix operand
__device__ __forceinline__ uint32_t row_chunk(uint32_t r, uint32_t c) { return (r >> 3) * 512u + c * 128u + (r & 7u) * 16u; }

// ND: levels 0 .. ND-1 are dense and the rest hashed, known at compile time; ND < 0: per-level run-time choice
template <bool U8, int ND>
__global__ void __launch_bounds__(kWsThreads, 1)
field_ws_kernel(const FieldArgs A, const uint4* __restrict__ packed_w, const void* __restrict__ both) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ __align__(8) uint64_t bar_ready[kNP], bar_full[kNF], bar_free[kNF], bar_g[kDecWGs], bar_a[kDecWGs];
    __shared__ uint32_t tmem_slot;

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    for (uint32_t i = threadIdx.x; i < kPackedBytes / 16; i += kWsThreads)
        reinterpret_cast<uint4*>(smem)[i] = __ldg(packed_w + i);
    // the direction-encoding operands keep zeros in their padding columns (inputs 56..63 of the appearance decoder)
    for (uint32_t i = threadIdx.x; i < kDecWGs * kPeBytes / 16; i += kWsThreads)
        reinterpret_cast<uint4*>(smem + kSmPe)[i] = make_uint4(0u, 0u, 0u, 0u);
    tc::fence_proxy_async_smem();
    if (warp == 0) tc::tmem_alloc<kWsTmemCols>(&tmem_slot);
    if (threadIdx.x == 32) {
        for (int i = 0; i < kNP; ++i) tc::mbar_init(&bar_ready[i], kTile);
        for (int i = 0; i < kNF; ++i) { tc::mbar_init(&bar_full[i], kTile / 16); tc::mbar_init(&bar_free[i], 1); }
        for (int i = 0; i < kDecWGs; ++i) { tc::mbar_init(&bar_g[i], 1); tc::mbar_init(&bar_a[i], 1); }
        tc::fence_mbar_init();
    }
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = tmem_slot;
    const uint32_t V = A.counters->V;
    const uint32_t n_tiles = (V + kTile - 1) / kTile;
    const uint32_t n_local = n_tiles > blockIdx.x ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;   // tiles b, b + grid, ...
    float* const sm_x = reinterpret_cast<float*>(smem + kSmX);
    uint32_t* const sm_ex = reinterpret_cast<uint32_t*>(smem + kSmEx);

    if (warp < kGatherWarps) {
        // ================================ gather warps ================================
        // unit u = (local tile u / 8, rows 16 (u % 8) .. + 15); lanes l and l ^ 16 share a Gaussian: the low lane takes
        // the corners at x, the high lane those at x + 1 (same 128-byte line 31 times in 32); after one exchange
        // the low lane holds the geometry features, the high lane the appearance features
        const uint32_t xb = lane >> 4, r16 = lane & 15u;
        for (uint32_t u = warp; u < n_local * 8u; u += kGatherWarps) {
            const uint32_t i = u >> 3, row = 16u * (u & 7u) + r16;
            const uint32_t sp = i % kNP, sf = i % kNF;
            tc::mbar_wait(&bar_ready[sp], (i / kNP) & 1u);
            const float* xs_in = sm_x + sp * (3 * kTile);
            const float xs[3] = {xs_in[row], xs_in[kTile + row], xs_in[2 * kTile + row]};
            if (i >= (uint32_t)kNF) tc::mbar_wait(&bar_free[sf], ((i / kNF) + 1u) & 1u);
            uint8_t* const dst = smem + kSmFeat + sf * kFeatBytes + (xb ? kFeatBytes / 2 : 0u) + row_chunk(row, 0);
            // software pipeline over the 16 levels: the loads of four levels are in flight while the oldest is blended
            LevelBuf buf[4];
#pragma unroll
            for (uint32_t q = 0; q < 4; ++q) level_issue<U8>(A.geo, both, q, ND < 0 ? ((A.geo.dense_mask >> q) & 1u) : (int)q < ND, xs, xb, buf[q]);
#pragma unroll 1
            for (uint32_t c = 0; c < 4; ++c) {
                uint32_t w4[4];
#pragma unroll
                for (uint32_t q = 0; q < 4; ++q) {
                    const uint32_t l = 4u * c + q;
                    float g0, g1, a0, a1;
                    level_consume<U8>(A.geo, A.app, l, buf[q], g0, g1, a0, a1);
                    if (c < 3) {
                        const uint32_t ln = l + 4u;
                        level_issue<U8>(A.geo, both, ln, ND < 0 ? ((A.geo.dense_mask >> ln) & 1u) : (int)ln < ND, xs, xb, buf[q]);
                    }
                    const float k0 = xb ? a0 : g0, k1 = xb ? a1 : g1, s0 = xb ? g0 : a0, s1 = xb ? g1 : a1;
                    w4[q] = pack_h2(__fadd_rn(k0, __shfl_xor_sync(0xffffffffu, s0, 16)),
                                    __fadd_rn(k1, __shfl_xor_sync(0xffffffffu, s1, 16)));
                }
                *reinterpret_cast<uint4*>(dst + c * 128u) = make_uint4(w4[0], w4[1], w4[2], w4[3]);
            }
            tc::fence_proxy_async_smem();   // these generic-proxy stores are read by the tensor core (async proxy)
            __syncwarp();
            if (lane == 0) tc::mbar_arrive(&bar_full[sf]);
        }
    } else {
        // ================================ decoder warpgroups ================================
        const uint32_t d = (warp - kGatherWarps) >> 2;
        const uint32_t row = threadIdx.x - (uint32_t)(kGatherWarps * 32) - d * kTile;   // Gaussian within the tile == TMEM lane
        const uint32_t lane_base = ((warp & 3u) * 32u) << 16;
        const uint32_t tDg = tmem + d * kWgCols, tDa = tDg + 64, tAg = tDg + 128, tAa = tDg + 160;
        const uint32_t sb = tc::smem_u32(smem);
        constexpr uint32_t idesc64 = tc::idesc_f16_f32(128, 64), idesc16 = tc::idesc_f16_f32(128, 16);
        uint64_t *const bg = &bar_g[d], *const ba = &bar_a[d];
        uint32_t phg = 0, pha = 0;
        const bool leader = row == 0;
        const uint32_t bar_id = 1u + d;

        // positions (for the gather warps) and explicit records (for this thread, later) of local tile i
        auto prep = [&](uint32_t i) {
            const uint32_t j = (blockIdx.x + i * gridDim.x) * kTile + row;
            const uint32_t sp = i % kNP;
            float x[3] = {0.5f, 0.5f, 0.5f};
            Explicit e{};
            e.j = 0xFFFFFFFFu;
            if (j < V) {
                e = fetch_visible(A, j);
                hy_contract(A.f, e.px, e.py, e.pz, x);
            }
            float* xo = sm_x + sp * (3 * kTile);
            xo[row] = x[0]; xo[kTile + row] = x[1]; xo[2 * kTile + row] = x[2];
            uint32_t* eo = sm_ex + sp * (9 * kTile) + row;
            eo[0] = __float_as_uint(e.px); eo[kTile] = __float_as_uint(e.py); eo[2 * kTile] = __float_as_uint(e.pz);
            eo[3 * kTile] = __float_as_uint(e.s_e); eo[4 * kTile] = __float_as_uint(e.a_e);
            eo[5 * kTile] = __float_as_uint(e.c_e0); eo[6 * kTile] = __float_as_uint(e.c_e1); eo[7 * kTile] = __float_as_uint(e.c_e2);
            eo[8 * kTile] = e.j;
            tc::mbar_arrive(&bar_ready[sp]);
        };
        // A <- relu(D) in fp16 (64 columns in two halves), then the warpgroup meets
        auto epilogue_to_A = [&](uint32_t tD, uint32_t tA) {
            uint32_t dd[32], pk[16];
            tc::ld_x32(tD + lane_base, dd); tc::wait_ld();
            relu_pack32(dd, pk);
            tc::st_x16(tA + lane_base, pk);
            tc::ld_x32(tD + lane_base + 32, dd); tc::wait_ld();
            relu_pack32(dd, pk);
            tc::st_x16(tA + lane_base + 16, pk);
            tc::wait_st();
            tc::fence_before_sync();
            asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
        };
        auto hidden_mma = [&](uint32_t tD, uint32_t tA, uint32_t w_off, uint32_t idesc, uint64_t* bar) {
            tc::fence_after_sync();
#pragma unroll
            for (uint32_t s = 0; s < 4; ++s)
                tc::mma_f16_ts(tD, tA + s * 8, tc::smem_desc_kmajor_noswizzle(sb + w_off + s * 256, 128, 1024), idesc, s);
            tc::commit(bar);
        };
        auto decode = [&](uint32_t i) {
            const uint32_t sp = i % kNP, sf = i % kNF;
            Explicit ex;
            {
                const uint32_t* ei = sm_ex + sp * (9 * kTile) + row;
                ex.px = __uint_as_float(ei[0]); ex.py = __uint_as_float(ei[kTile]); ex.pz = __uint_as_float(ei[2 * kTile]);
                ex.s_e = __uint_as_float(ei[3 * kTile]); ex.a_e = __uint_as_float(ei[4 * kTile]);
                ex.c_e0 = __uint_as_float(ei[5 * kTile]); ex.c_e1 = __uint_as_float(ei[6 * kTile]); ex.c_e2 = __uint_as_float(ei[7 * kTile]);
                ex.j = ei[8 * kTile];
            }
            const bool valid = ex.j != 0xFFFFFFFFu;
            {   // D4 -> this warpgroup's direction-encoding operand (K = 24 of 32; the rest stays zero)
                uint32_t pe2[12];
#pragma unroll
                for (int k = 0; k < 12; ++k) pe2[k] = 0u;
                if (valid) dir_pe_packed(A.f, ex.px, ex.py, ex.pz, pe2);
                uint8_t* pe = smem + kSmPe + d * kPeBytes + row_chunk(row, 0);
                *reinterpret_cast<uint4*>(pe) = make_uint4(pe2[0], pe2[1], pe2[2], pe2[3]);
                *reinterpret_cast<uint4*>(pe + 128) = make_uint4(pe2[4], pe2[5], pe2[6], pe2[7]);
                *reinterpret_cast<uint4*>(pe + 256) = make_uint4(pe2[8], pe2[9], pe2[10], pe2[11]);
                tc::fence_proxy_async_smem();
            }
            tc::fence_before_sync();   // (also orders the previous tile's tcgen05.ld of the outputs before the next MMAs)
            asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
            if (leader) {
                // ---- layer 1, both chains, operands from shared memory ----
                tc::mbar_wait(&bar_full[sf], (i / kNF) & 1u);
                tc::fence_after_sync();
                const uint32_t fg = sb + kSmFeat + sf * kFeatBytes, fa = fg + kFeatBytes / 2, pe = sb + kSmPe + d * kPeBytes;
#pragma unroll
                for (uint32_t s = 0; s < 2; ++s)   // geometry: K = 32
                    tc::mma_f16_ss(tDg, tc::smem_desc_kmajor_noswizzle(fg + s * 256, 128, 512),
                                   tc::smem_desc_kmajor_noswizzle(sb + kOffG1 + s * 256, 128, 512), idesc64, s);
                tc::commit(bg);
#pragma unroll
                for (uint32_t s = 0; s < 2; ++s)   // appearance: K = 32 features ...
                    tc::mma_f16_ss(tDa, tc::smem_desc_kmajor_noswizzle(fa + s * 256, 128, 512),
                                   tc::smem_desc_kmajor_noswizzle(sb + kOffA1 + s * 256, 128, 1024), idesc64, s);
#pragma unroll
                for (uint32_t s = 0; s < 2; ++s)   // ... + K = 32 direction encoding
                    tc::mma_f16_ss(tDa, tc::smem_desc_kmajor_noswizzle(pe + s * 256, 128, 512),
                                   tc::smem_desc_kmajor_noswizzle(sb + kOffA1 + (2 + s) * 256, 128, 1024), idesc64, 1u);
                tc::commit(ba);
                tc::commit(&bar_free[sf]);   // the feature buffer may be refilled once these MMAs have read it
            }
            // ---- layer 2 ----
            tc::mbar_wait(bg, phg); phg ^= 1u; tc::fence_after_sync();
            epilogue_to_A(tDg, tAg);
            if (leader) hidden_mma(tDg, tAg, kOffG2, idesc64, bg);
            tc::mbar_wait(ba, pha); pha ^= 1u; tc::fence_after_sync();
            epilogue_to_A(tDa, tAa);
            if (leader) hidden_mma(tDa, tAa, kOffA2, idesc64, ba);
            // ---- output layer ----
            tc::mbar_wait(bg, phg); phg ^= 1u; tc::fence_after_sync();
            epilogue_to_A(tDg, tAg);
            if (leader) hidden_mma(tDg, tAg, kOffG3, idesc16, bg);
            tc::mbar_wait(ba, pha); pha ^= 1u; tc::fence_after_sync();
            epilogue_to_A(tDa, tAa);
            if (leader) hidden_mma(tDa, tAa, kOffA3, idesc16, ba);
            float raw[11];
            {
                uint32_t o[8];
                tc::mbar_wait(bg, phg); phg ^= 1u; tc::fence_after_sync();
                tc::ld_x8(tDg + lane_base, o); tc::wait_ld();
#pragma unroll
                for (int k = 0; k < 8; ++k) raw[k] = __uint_as_float(o[k]);
                tc::mbar_wait(ba, pha); pha ^= 1u; tc::fence_after_sync();
                tc::ld_x4(tDa + lane_base, o); tc::wait_ld();
                raw[8] = __uint_as_float(o[0]); raw[9] = __uint_as_float(o[1]); raw[10] = __uint_as_float(o[2]);
            }
            if (valid) aggregate_project<true>(A, ex, raw);
        };

        uint32_t i = d;
        if (i < n_local) prep(i);
        for (; i < n_local; i += kDecWGs) {
            if (i + kDecWGs < n_local) prep(i + kDecWGs);   // two tiles ahead: the gather warps never wait for positions
            decode(i);
        }
    }
    tc::fence_before_sync();
    __syncthreads();
    if (warp == 0) tc::tmem_dealloc<kWsTmemCols>(tmem);
}

}  // namespace

// every level below n_dense dense, every other hashed?
static int contiguous_dense(const GridDev& g) {
    int nd = 0;
    while (nd < (int)g.levels && ((g.dense_mask >> nd) & 1u)) ++nd;
    return (g.dense_mask >> nd) == 0u ? nd : -1;
}

hyrf_status hy_launch_field_ws(hyrf_scene* s, const FrameDev& f, uint32_t* launches) {
    FieldArgs A;
    hy_fill_field_args(s, f, &A);
    if (!s->field_ws_attr_set) {
        const void* ks[4] = {(const void*)field_ws_kernel<false, 5>, (const void*)field_ws_kernel<true, 5>,
                             (const void*)field_ws_kernel<false, -1>, (const void*)field_ws_kernel<true, -1>};
        for (const void* k : ks) {
            cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kWsSmemBytes);
            if (e != cudaSuccess) return hy_cuda_fail(e, "cudaFuncSetAttribute(field_ws)");
        }
        s->field_ws_attr_set = true;
    }
    const int need = (int)((s->N + kTile - 1) / kTile);
    // One CTA per SM holds (nearly) every register of it: with the depth sort beside this kernel (hyrf_set_sort_overlap)
    // a few SMs are left to the sort's CTAs.
    const int gap = s->field_full_grid ? 0 : s->ws_sort_sms;
    const int slots = s->sm_count - gap > 1 ? s->sm_count - gap : 1;
    const int grid = need < slots ? need : slots;
    const uint4* w = reinterpret_cast<const uint4*>(s->mma_w);
    const bool nd5 = contiguous_dense(s->geo_grid) == 5;   // every BASELINE configuration with 16 levels and 2^19 entries
    if (s->u8) {
        if (nd5) field_ws_kernel<true, 5><<<grid, kWsThreads, kWsSmemBytes, s->stream>>>(A, w, s->both_table);
        else field_ws_kernel<true, -1><<<grid, kWsThreads, kWsSmemBytes, s->stream>>>(A, w, s->both_table);
    } else {
        if (nd5) field_ws_kernel<false, 5><<<grid, kWsThreads, kWsSmemBytes, s->stream>>>(A, w, s->both_table);
        else field_ws_kernel<false, -1><<<grid, kWsThreads, kWsSmemBytes, s->stream>>>(A, w, s->both_table);
    }
    ++*launches;
    return HYRF_OK;
}
