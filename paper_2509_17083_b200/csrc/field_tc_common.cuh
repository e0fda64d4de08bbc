// field_tc_common.cuh — pieces shared by the tensor-core field kernels (field_mma.cu: every warp gathers and decodes;
// field_ws.cu: warp-specialised producer / consumer): the packed tcgen05 B-operand block of the decoder weights, the
// K-major core-matrix index, and the two-lane gather of one level of the interleaved geometry + appearance table
// (Eq. 3; DESIGN.md §2 D3, §5).
#pragma once
#include "field_common.cuh"

namespace {

// packed weight block (bytes): geo W1 [64 x 32], W2 [64 x 64], W3 [16 x 64]; app W1 [64 x 64], W2, W3
constexpr uint32_t kOffG1 = 0, kOffG2 = 4096, kOffG3 = 12288, kOffA1 = 14336, kOffA2 = 22528, kOffA3 = 30720;
constexpr uint32_t kPackedBytes = 32768;
constexpr uint32_t kSmemBytes = kPackedBytes;   // two CTAs (2 x 256 TMEM columns) per SM by registers; the rest of the 228 KB is L1

// element (n, k) of an [N x Kp] K-major operand stored as 8x8 core matrices: half-index inside the operand
__host__ __device__ inline uint32_t core_index(uint32_t n, uint32_t k, uint32_t Kp) {
    return (n >> 3) * (Kp * 8) + (k >> 3) * 64 + (n & 7) * 8 + (k & 7);
}

__device__ __forceinline__ uint32_t pack_h2(float lo, float hi) {
    __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&h);
}

// The same level for BOTH fields at once, when the two grids share their geometry (levels, resolutions, table size —
// true of every paper configuration): the tables are interleaved at upload into one array of 8-byte entries
// (geo f0, geo f1, app f0, app f1), so one index computation and one load serve both fields and the x / x+1
// corners of both fields sit in one 16-byte span. Halves the sector look-ups and the index arithmetic.
// DMODE: 1 = the level is known dense at compile time, 0 = known hashed, -1 = decided by the grid's dense_mask at run time
// (both index paths then sit in the instruction stream under a predicate).
template <bool U8, int DMODE = -1>
__device__ __forceinline__ void gather_level_half2(const GridDev& g, const GridDev& ga, const void* __restrict__ both,
                                                   uint32_t l, const float x[3], uint32_t xb,
                                                   float& g0, float& g1, float& a0, float& a1) {
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
    if (DMODE == 1 || (DMODE < 0 && ((g.dense_mask >> l) & 1u))) {
        const uint32_t n1 = N + 1u;
        const uint32_t b = vx + n1 * (ci[1] + n1 * ci[2]);
        idx[0] = b; idx[1] = b + n1; idx[2] = b + n1 * n1; idx[3] = b + n1 * n1 + n1;
    } else {
        const uint32_t hy0 = ci[1] * 2654435761u, hy1 = hy0 + 2654435761u;
        const uint32_t hz0 = ci[2] * 805459861u, hz1 = hz0 + 805459861u;
        idx[0] = (vx ^ hy0 ^ hz0) & g.table_mask; idx[1] = (vx ^ hy1 ^ hz0) & g.table_mask;
        idx[2] = (vx ^ hy0 ^ hz1) & g.table_mask; idx[3] = (vx ^ hy1 ^ hz1) & g.table_mask;
    }
    float2 vgs[4], vas[4];
    if (U8) {   // 4-byte entries (geo c0 c1 | app c0 c1), D3': value = fma(code, step, min)
        const uchar4* tab = reinterpret_cast<const uchar4*>(both) + g.offset[l];
        const float2 qg0 = g.q[l][0], qg1 = g.q[l][1], qa0 = ga.q[l][0], qa1 = ga.q[l][1];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uchar4 c = __ldg(tab + idx[k]);
            vgs[k] = make_float2(__fmaf_rn((float)c.x, qg0.y, qg0.x), __fmaf_rn((float)c.y, qg1.y, qg1.x));
            vas[k] = make_float2(__fmaf_rn((float)c.z, qa0.y, qa0.x), __fmaf_rn((float)c.w, qa1.y, qa1.x));
        }
    } else {
        const uint2* tab = reinterpret_cast<const uint2*>(both) + g.offset[l];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint2 v = __ldg(tab + idx[k]);
            vgs[k] = __half22float2(*reinterpret_cast<const __half2*>(&v.x));
            vas[k] = __half22float2(*reinterpret_cast<const __half2*>(&v.y));
        }
    }
    const float ax = xb ? w[0] : __fsub_rn(1.0f, w[0]);
    const float wy0 = __fsub_rn(1.0f, w[1]), wz0 = __fsub_rn(1.0f, w[2]);
    g0 = 0.0f; g1 = 0.0f; a0 = 0.0f; a1 = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float wt = __fmul_rn(__fmul_rn(ax, (k & 1) ? w[1] : wy0), (k & 2) ? w[2] : wz0);
        const float2 vg = vgs[k], va = vas[k];
        g0 = __fmaf_rn(wt, vg.x, g0); g1 = __fmaf_rn(wt, vg.y, g1);
        a0 = __fmaf_rn(wt, va.x, a0); a1 = __fmaf_rn(wt, va.y, a1);
    }
}


// The same look-up cut in two, for software pipelining (field_ws.cu): level_issue computes the cell, the four corner
// indices of this lane's x side and the blend weights and ISSUES the four loads; level_consume, called a few levels
// later, blends them. Between the two only the loaded words (8 registers) and three weights are live, so a warp keeps
// several levels' loads in flight. Arithmetic and operation order are those of gather_level_half2.
struct LevelBuf {
    uint2 v[4];        // corner (y, z) = (k & 1, k >> 1): (geo f0 f1 | app f0 f1) halves, or 4 codes in .x (8-bit tables)
    float ax, wy, wz;  // this lane's x weight (w_x or 1 - w_x), w_y, w_z
};

template <bool U8>
__device__ __forceinline__ void level_issue(const GridDev& g, const void* __restrict__ both, uint32_t l, bool dense,
                                            const float x[3], uint32_t xb, LevelBuf& b) {
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
    if (dense) {
        const uint32_t n1 = N + 1u;
        const uint32_t bb = vx + n1 * (ci[1] + n1 * ci[2]);
        idx[0] = bb; idx[1] = bb + n1; idx[2] = bb + n1 * n1; idx[3] = bb + n1 * n1 + n1;
    } else {
        const uint32_t hy0 = ci[1] * 2654435761u, hy1 = hy0 + 2654435761u;
        const uint32_t hz0 = ci[2] * 805459861u, hz1 = hz0 + 805459861u;
        idx[0] = (vx ^ hy0 ^ hz0) & g.table_mask; idx[1] = (vx ^ hy1 ^ hz0) & g.table_mask;
        idx[2] = (vx ^ hy0 ^ hz1) & g.table_mask; idx[3] = (vx ^ hy1 ^ hz1) & g.table_mask;
    }
    // The level's base pointer is pinned in a register pair (the empty asm keeps the compiler from folding the level
    // offset into each index), so every address is ONE wide multiply-add (IMAD.WIDE.U32 idx, 8, base) instead of a
    // three- or four-instruction 64-bit add chain: the gather warps are issue-bound once their loads are pipelined.
    if (U8) {
        const uint32_t* tab = reinterpret_cast<const uint32_t*>(both) + g.offset[l];
        asm volatile("" : "+l"(tab));
#pragma unroll
        for (int k = 0; k < 4; ++k) b.v[k] = make_uint2(__ldg(tab + idx[k]), 0u);
    } else {
        const uint2* tab = reinterpret_cast<const uint2*>(both) + g.offset[l];
        asm volatile("" : "+l"(tab));
#pragma unroll
        for (int k = 0; k < 4; ++k) b.v[k] = __ldg(tab + idx[k]);
    }
    b.ax = xb ? w[0] : __fsub_rn(1.0f, w[0]);
    b.wy = w[1];
    b.wz = w[2];
}

template <bool U8>
__device__ __forceinline__ void level_consume(const GridDev& g, const GridDev& ga, uint32_t l, const LevelBuf& b,
                                              float& g0, float& g1, float& a0, float& a1) {
    const float wy0 = __fsub_rn(1.0f, b.wy), wz0 = __fsub_rn(1.0f, b.wz);
    g0 = 0.0f; g1 = 0.0f; a0 = 0.0f; a1 = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float2 vg, va;
        if (U8) {   // D3': value = fma(code, step, min)
            const uint32_t c = b.v[k].x;
            const float2 qg0 = g.q[l][0], qg1 = g.q[l][1], qa0 = ga.q[l][0], qa1 = ga.q[l][1];
            vg = make_float2(__fmaf_rn((float)(c & 0xFFu), qg0.y, qg0.x), __fmaf_rn((float)((c >> 8) & 0xFFu), qg1.y, qg1.x));
            va = make_float2(__fmaf_rn((float)((c >> 16) & 0xFFu), qa0.y, qa0.x), __fmaf_rn((float)(c >> 24), qa1.y, qa1.x));
        } else {
            vg = __half22float2(*reinterpret_cast<const __half2*>(&b.v[k].x));
            va = __half22float2(*reinterpret_cast<const __half2*>(&b.v[k].y));
        }
        const float wt = __fmul_rn(__fmul_rn(b.ax, (k & 1) ? b.wy : wy0), (k & 2) ? b.wz : wz0);
        g0 = __fmaf_rn(wt, vg.x, g0); g1 = __fmaf_rn(wt, vg.y, g1);
        a0 = __fmaf_rn(wt, va.x, a0); a1 = __fmaf_rn(wt, va.y, a1);
    }
}

// D4 for the fp16 decoders: direction of p from the camera centre, 4 octaves of (sin, cos) per axis, rounded to fp16 and
// packed in input order (6k + a = sin, 6k + 3 + a = cos) -> 12 words. By octave doubling: one sincospi per axis, then
// sin 2t = 2 sin t cos t, cos 2t = 1 - 2 sin^2 t; three doublings amplify the 1-ulp start error to ~1e-6, far below
// the fp16 rounding that follows.
__device__ __forceinline__ void dir_pe_packed(const FrameDev& f, float px, float py, float pz, uint32_t pe2[12]) {
    const float dx = __fsub_rn(px, f.o[0]), dy = __fsub_rn(py, f.o[1]), dz = __fsub_rn(pz, f.o[2]);
    const float n = __fsqrt_rn(__fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx))));
    const float d[3] = {__fdiv_rn(dx, n), __fdiv_rn(dy, n), __fdiv_rn(dz, n)};
    float pe[24];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        float sn, cs;
        sincospif(d[ax], &sn, &cs);
        pe[ax] = sn; pe[3 + ax] = cs;
#pragma unroll
        for (int k = 1; k < 4; ++k) {
            const float s2 = 2.0f * sn * cs, c2 = 1.0f - 2.0f * sn * sn;
            sn = s2; cs = c2;
            pe[6 * k + ax] = sn; pe[6 * k + 3 + ax] = cs;
        }
    }
#pragma unroll
    for (int i = 0; i < 12; ++i) pe2[i] = pack_h2(pe[2 * i], pe[2 * i + 1]);
}

// ReLU + round to fp16 of 32 fp32 accumulator columns -> 16 packed A columns
__device__ __forceinline__ void relu_pack32(const uint32_t* d, uint32_t* a) {
#pragma unroll
    for (int i = 0; i < 16; ++i)
        a[i] = pack_h2(fmaxf(__uint_as_float(d[2 * i]), 0.0f), fmaxf(__uint_as_float(d[2 * i + 1]), 0.0f));
}

}  // namespace
