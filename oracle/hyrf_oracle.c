/*
 * hyrf_oracle.c — CPU oracle for HyRF's hybrid forward render pass (arxiv 2509.17083).
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file. It shares no code with the CUDA path
 * (paper_2509_17083_b200/csrc); both were written from DESIGN.md §2, which restates the paper.
 *
 * Plain, slow, scalar C. The pass is an algorithm with built-in decisions (centre-only cull, 3-sigma tile
 * rectangle, alpha < 1/255 skip, T < 1e-4 stop, tau_T test), not a fast route to a separately defined exact
 * result, so the oracle follows the algorithm step by step in the paper's order. Arithmetic is IEEE binary32
 * with the rounding points of DESIGN.md §2 (compile with -ffp-contract=off; every fused multiply-add is an
 * explicit fmaf), because floating point decides integers here (visibility, tile rectangles, list order) and
 * both sides must take those decisions in the same precision.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py against closed forms, invariants,
 * library routines and brute force. What is NOT pinned: agreement with the authors' own renderer — the paper
 * prints no worked values ("parity unpinned" for the whole pass, and for the hash/level conventions of [27]
 * that the paper only cites, A12).
 *
 * OpenMP parallelism is over independent items only (Gaussians, tiles' pixels), so results do not depend on
 * the thread count.
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define HO_MAX_LEVELS 32
#define HO_MAX_DIM 256

typedef struct { uint32_t levels, feats, log2_table; uint32_t res[HO_MAX_LEVELS]; } ho_grid;
typedef struct { uint32_t in_dim, hidden, n_hidden, out_dim; } ho_mlp;
typedef struct { float R[9], t[3], fx, fy, cx, cy; } ho_camera;

typedef struct {
    uint32_t n;
    const float *pos;            /* [3][n] SoA */
    const float *rgb_logit;      /* [3][n] */
    const float *scale_logit;    /* [n] */
    const float *opacity_logit;  /* [n] */
    float aabb_min[3], aabb_max[3];
    ho_grid geo_grid, app_grid, bg_grid;
    ho_mlp geo_mlp, app_mlp, bg_mlp;
    const void *geo_table, *app_table, *bg_table;   /* [entries][2], f32 or f16 */
    const void *geo_w, *app_w, *bg_w;               /* layers concatenated, row-major [out][in] */
    int32_t fp16;
    uint32_t pe_octaves;
    float cull_tol, z_near, bg_radius, tau_T;
    /* compressed model (item 3): tables stored as 8-bit codes with per-level, per-feature
     * (min, step); q[(level * feats + f) * 2 + {0, 1}]. table_u8 != 0 implies fp16 weights / activations. */
    int32_t table_u8;
    const float *geo_q, *app_q, *bg_q;
} ho_scene;

/* ------------------------------------------------------------------------------------------------ */
/* fp16 <-> fp32, bit level (IEEE binary16, round-to-nearest-even). DESIGN.md §2 D3/D5 rounding points */

float ho_half_to_float(uint16_t h) {
    uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    uint32_t exp = (h >> 10) & 0x1Fu;
    uint32_t man = h & 0x3FFu;
    uint32_t bits;
    if (exp == 0) {
        if (man == 0) {
            bits = sign;
        } else {                       /* subnormal: value = man * 2^-24 */
            float v = (float)man * 5.9604644775390625e-08f;
            memcpy(&bits, &v, 4);
            bits |= sign;
        }
    } else if (exp == 31) {
        bits = sign | 0x7F800000u | (man << 13);
    } else {
        bits = sign | ((exp + 112u) << 23) | (man << 13);
    }
    float f;
    memcpy(&f, &bits, 4);
    return f;
}

uint16_t ho_float_to_half(float f) {
    uint32_t x;
    memcpy(&x, &f, 4);
    uint32_t sign = (x >> 16) & 0x8000u;
    uint32_t absx = x & 0x7FFFFFFFu;
    if (absx >= 0x7F800000u) {                               /* inf / nan */
        return (uint16_t)(sign | 0x7C00u | ((absx > 0x7F800000u) ? 0x200u : 0u));
    }
    if (absx >= 0x477FF000u) {                               /* rounds to >= 65520 -> inf */
        return (uint16_t)(sign | 0x7C00u);
    }
    if (absx < 0x38800000u) {                                /* result is subnormal or zero: |f| < 2^-14 */
        /* value / 2^-24 rounded to nearest even integer */
        float a;
        memcpy(&a, &absx, 4);
        float scaled = a * 16777216.0f;                      /* exact (power of two) */
        float r = rintf(scaled);                             /* RN-even in the default rounding mode */
        return (uint16_t)(sign | (uint32_t)r);               /* r <= 1024 -> may carry into exponent 1: correct */
    }
    uint32_t exp = (absx >> 23) - 112u;                      /* half exponent field */
    uint32_t man = absx & 0x7FFFFFu;
    uint32_t half = (exp << 10) | (man >> 13);
    uint32_t rem = man & 0x1FFFu;
    if (rem > 0x1000u || (rem == 0x1000u && (half & 1u))) half++;   /* carries propagate correctly */
    return (uint16_t)(sign | half);
}

static inline float round_h(float f) { return ho_half_to_float(ho_float_to_half(f)); }

/* ------------------------------------------------------------------------------------------------ */
/* D6 soft exponential and sigmoid */

float ho_softexp(float x) {
    x = fminf(fmaxf(x, -87.0f), 88.0f);
    float n = rintf(x * 1.44269504f);
    float r = fmaf(n, -0.693145752f, x);
    r = fmaf(n, -1.42860677e-6f, r);
    float p = 1.98412701e-4f;
    p = fmaf(p, r, 1.38888892e-3f);
    p = fmaf(p, r, 8.33333377e-3f);
    p = fmaf(p, r, 4.16666679e-2f);
    p = fmaf(p, r, 1.66666672e-1f);
    p = fmaf(p, r, 0.5f);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    int32_t ni = (int32_t)n;
    uint32_t bits = (uint32_t)(ni + 127) << 23;
    float s;
    memcpy(&s, &bits, 4);
    return p * s;
}

float ho_sigmoid(float v) { return 1.0f / (1.0f + ho_softexp(-v)); }

/* ------------------------------------------------------------------------------------------------ */
/* Camera helpers (DESIGN.md §2 "Camera", D1) */

void ho_camera_center(const ho_camera *cam, float o[3]) {
    const float *R = cam->R, *t = cam->t;
    for (int k = 0; k < 3; ++k)
        o[k] = -(fmaf(R[6 + k], t[2], fmaf(R[3 + k], t[1], R[k] * t[0])));
}

void ho_to_camera(const ho_camera *cam, const float p[3], float pc[3]) {
    const float *R = cam->R;
    for (int k = 0; k < 3; ++k)
        pc[k] = fmaf(R[3 * k + 2], p[2], fmaf(R[3 * k + 1], p[1], fmaf(R[3 * k], p[0], cam->t[k])));
}

/* D1 cull: Eq. 8-9 (readings A4-A6). Returns V; mask[n], idx[V] ascending. */
uint32_t ho_stage_cull(const ho_scene *s, const ho_camera *cam, int32_t W, int32_t H, uint8_t *mask,
                       uint32_t *idx) {
    float limx = (1.0f + s->cull_tol) * ((float)W / (2.0f * cam->fx));
    float limy = (1.0f + s->cull_tol) * ((float)H / (2.0f * cam->fy));
    uint32_t n = s->n;
#pragma omp parallel for schedule(static)
    for (uint32_t i = 0; i < n; ++i) {
        float p[3] = {s->pos[i], s->pos[n + i], s->pos[2u * n + i]}, pc[3];
        ho_to_camera(cam, p, pc);
        int keep = (pc[2] > s->z_near) && (fabsf(pc[0]) <= limx * pc[2]) && (fabsf(pc[1]) <= limy * pc[2]);
        mask[i] = (uint8_t)keep;
    }
    uint32_t v = 0;
    for (uint32_t i = 0; i < n; ++i)
        if (mask[i]) idx[v++] = i;
    return v;
}

/* D2 contraction: PAPER.md:65-70 Eq. 2, :347-358 Eq. 13-14 (readings A1-A3). */
void ho_contract(const float p[3], const float amin[3], const float amax[3], float x[3]) {
    float q[3];
    for (int a = 0; a < 3; ++a) {
        float c = 0.5f * (amin[a] + amax[a]);
        float h = 0.5f * (amax[a] - amin[a]);
        q[a] = (p[a] - c) / h;
    }
    float n2 = fmaf(q[2], q[2], fmaf(q[1], q[1], q[0] * q[0]));
    float n = sqrtf(n2);
    if (!(n <= 1.0f)) {
        float inv = 1.0f / n;
        float sc = (2.0f - inv) * inv;
        for (int a = 0; a < 3; ++a) q[a] = sc * q[a];
    }
    for (int a = 0; a < 3; ++a) x[a] = fminf(fmaxf(fmaf(0.25f, q[a], 0.5f), 0.0f), 1.0f);
}

/* D3 grid layout: sizes / offsets per level. Returns total entries. */
uint64_t ho_grid_layout(const ho_grid *g, uint32_t *sizes, uint32_t *offsets, uint8_t *dense) {
    uint64_t T = 1ull << g->log2_table, off = 0;
    for (uint32_t l = 0; l < g->levels; ++l) {
        uint64_t n1 = (uint64_t)g->res[l] + 1ull;
        uint64_t d = n1 * n1 * n1;
        int is_dense = d <= T;
        uint64_t sz = is_dense ? ((d + 7ull) / 8ull) * 8ull : T;
        if (sizes) sizes[l] = (uint32_t)sz;
        if (offsets) offsets[l] = (uint32_t)off;
        if (dense) dense[l] = (uint8_t)is_dense;
        off += sz;
    }
    return off;
}

/* D3 vertex -> entry index inside its level. */
uint32_t ho_grid_index(const ho_grid *g, uint32_t level, uint32_t vx, uint32_t vy, uint32_t vz) {
    uint64_t T = 1ull << g->log2_table;
    uint64_t n1 = (uint64_t)g->res[level] + 1ull;
    if (n1 * n1 * n1 <= T) return (uint32_t)(vx + n1 * (vy + n1 * vz));
    uint32_t h = (vx * 1u) ^ (vy * 2654435761u) ^ (vz * 805459861u);
    return h & (uint32_t)(T - 1ull);
}

/* mode 0: fp32 entries; 1: fp16 entries (exact in fp32); 2: 8-bit min-max codes, value = fma(code, step, min)
 * with the (min, step) of this level and feature (DESIGN.md §2 D3', "8-bit min-max quantization"). */
static inline float table_value(const void *table, int mode, const float *q, uint32_t level, uint64_t entry, uint32_t f,
                                uint32_t feats) {
    if (mode == 2) {
        const float *qp = q + ((size_t)level * feats + f) * 2;
        return fmaf((float)((const uint8_t *)table)[entry * feats + f], qp[1], qp[0]);
    }
    if (mode == 1) return ho_half_to_float(((const uint16_t *)table)[entry * feats + f]);
    return ((const float *)table)[entry * feats + f];
}

/* D3 encode: PAPER.md:61, :74 Eq. 3, :152. x in [0,1]^3 -> feat[levels*feats], level-major. */
void ho_grid_encode_q(const ho_grid *g, const void *table, int32_t mode, const float *q, const float x[3], float *feat) {
    const int fp16 = mode != 0;   /* fp16 and 8-bit tables both feed fp16 decoders: the feature is rounded to fp16 */
    uint32_t offsets[HO_MAX_LEVELS];
    ho_grid_layout(g, NULL, offsets, NULL);
    for (uint32_t l = 0; l < g->levels; ++l) {
        uint32_t N = g->res[l];
        uint32_t ci[3];
        float w[3];
        for (int a = 0; a < 3; ++a) {
            float u = x[a] * (float)N;
            int32_t i = (int32_t)floorf(u);
            if (i > (int32_t)N - 1) i = (int32_t)N - 1;
            ci[a] = (uint32_t)i;
            w[a] = u - (float)i;
        }
        for (uint32_t f = 0; f < g->feats; ++f) {
            float acc = 0.0f;
            for (uint32_t k = 0; k < 8; ++k) {
                uint32_t bx = k & 1u, by = (k >> 1) & 1u, bz = (k >> 2) & 1u;
                float ax = bx ? w[0] : 1.0f - w[0];
                float ay = by ? w[1] : 1.0f - w[1];
                float az = bz ? w[2] : 1.0f - w[2];
                float wt = (ax * ay) * az;
                uint32_t e = ho_grid_index(g, l, ci[0] + bx, ci[1] + by, ci[2] + bz);
                float val = table_value(table, mode, q, l, (uint64_t)offsets[l] + e, f, g->feats);
                acc = fmaf(wt, val, acc);
            }
            feat[l * g->feats + f] = fp16 ? round_h(acc) : acc;
        }
    }
}

void ho_grid_encode(const ho_grid *g, const void *table, int32_t fp16, const float x[3], float *feat) {
    ho_grid_encode_q(g, table, fp16 ? 1 : 0, NULL, x, feat);
}

/* D4: unit view direction from camera centre o to p (Eq. 5). */
void ho_view_dir(const float p[3], const float o[3], float d[3]) {
    float dx = p[0] - o[0], dy = p[1] - o[1], dz = p[2] - o[2];
    float n = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
    d[0] = dx / n; d[1] = dy / n; d[2] = dz / n;
}

/* D4 encoding of a unit direction: out[6k+a] = sin(pi 2^k d_a), out[6k+3+a] = cos(pi 2^k d_a). */
void ho_dir_pe(const float d[3], uint32_t octaves, int32_t fp16, float *out) {
    for (uint32_t k = 0; k < octaves; ++k) {
        float sc = (float)(1u << k);
        for (int a = 0; a < 3; ++a) {
            double arg = M_PI * (double)(sc * d[a]);
            float sv = (float)sin(arg), cv = (float)cos(arg);
            out[6 * k + a] = fp16 ? round_h(sv) : sv;
            out[6 * k + 3 + a] = fp16 ? round_h(cv) : cv;
        }
    }
}

/* D5 MLP: PAPER.md:83-95 Eq. 4/6, :152 (reading A11). in[in_dim] -> out[out_dim]. */
void ho_mlp_forward(const ho_mlp *m, const void *w, int32_t fp16, const float *in, float *out) {
    float a[HO_MAX_DIM], b[HO_MAX_DIM];
    uint32_t cur = m->in_dim;
    for (uint32_t k = 0; k < cur; ++k) a[k] = in[k];
    uint64_t woff = 0;
    for (uint32_t layer = 0; layer <= m->n_hidden; ++layer) {
        int last = (layer == m->n_hidden);
        uint32_t nout = last ? m->out_dim : m->hidden;
        for (uint32_t j = 0; j < nout; ++j) {
            float acc = 0.0f;
            for (uint32_t k = 0; k < cur; ++k) {
                uint64_t wi = woff + (uint64_t)j * cur + k;
                float wv = fp16 ? ho_half_to_float(((const uint16_t *)w)[wi]) : ((const float *)w)[wi];
                acc = fmaf(wv, a[k], acc);
            }
            if (!last) {
                acc = fmaxf(acc, 0.0f);
                if (fp16) acc = round_h(acc);
            }
            b[j] = acc;
        }
        woff += (uint64_t)nout * cur;
        cur = nout;
        for (uint32_t k = 0; k < cur; ++k) a[k] = b[k];
    }
    for (uint32_t k = 0; k < m->out_dim; ++k) out[k] = a[k];
}

/* S2 for one point: contraction, both encodes, PE, both decoders. raw = (alpha_n, s_n[3], r_n[4], c_n[3]). */
void ho_query_point(const ho_scene *s, const float p[3], const float o[3], float raw[11]) {
    float x[3], in[HO_MAX_DIM], d[3];
    ho_contract(p, s->aabb_min, s->aabb_max, x);
    /* geometry field: Eq. 3, 4 */
    memset(in, 0, sizeof(in));
    ho_grid_encode_q(&s->geo_grid, s->geo_table, s->table_u8 ? 2 : s->fp16, s->geo_q, x, in);
    ho_mlp_forward(&s->geo_mlp, s->geo_w, s->fp16, in, raw);
    /* appearance field: Eq. 3, 5, 6 */
    memset(in, 0, sizeof(in));
    ho_grid_encode_q(&s->app_grid, s->app_table, s->table_u8 ? 2 : s->fp16, s->app_q, x, in);
    ho_view_dir(p, o, d);
    ho_dir_pe(d, s->pe_octaves, s->fp16, in + s->app_grid.levels * s->app_grid.feats);
    ho_mlp_forward(&s->app_mlp, s->app_w, s->fp16, in, raw + 8);
}

void ho_stage_query(const ho_scene *s, const ho_camera *cam, uint32_t V, const uint32_t *idx, float *raw) {
    float o[3];
    ho_camera_center(cam, o);
    uint32_t n = s->n;
#pragma omp parallel for schedule(static)
    for (uint32_t j = 0; j < V; ++j) {
        uint32_t i = idx[j];
        float p[3] = {s->pos[i], s->pos[n + i], s->pos[2u * n + i]};
        ho_query_point(s, p, o, raw + 11ull * j);
    }
}

/* D7 aggregation: Eq. 7. attrs = (s[3], r[4] (w,x,y,z), alpha, c[3]). */
void ho_aggregate(const float raw[11], float s_e, float a_e, const float c_e[3], float attrs[11]) {
    for (int j = 0; j < 3; ++j) attrs[j] = ho_sigmoid(raw[1 + j] + s_e);
    float r0 = raw[4], r1 = raw[5], r2 = raw[6], r3 = raw[7];
    float m = sqrtf(fmaf(r3, r3, fmaf(r2, r2, fmaf(r1, r1, r0 * r0))));
    float den = fmaxf(m, 1e-12f);
    attrs[3] = r0 / den; attrs[4] = r1 / den; attrs[5] = r2 / den; attrs[6] = r3 / den;
    attrs[7] = ho_sigmoid(raw[0] + a_e);
    for (int j = 0; j < 3; ++j) attrs[8 + j] = ho_sigmoid(raw[8 + j] + c_e[j]);
}

void ho_stage_aggregate(const ho_scene *s, uint32_t V, const uint32_t *idx, const float *raw, float *attrs) {
    uint32_t n = s->n;
#pragma omp parallel for schedule(static)
    for (uint32_t j = 0; j < V; ++j) {
        uint32_t i = idx[j];
        float c_e[3] = {s->rgb_logit[i], s->rgb_logit[n + i], s->rgb_logit[2u * n + i]};
        ho_aggregate(raw + 11ull * j, s->scale_logit[i], s->opacity_logit[i], c_e, attrs + 11ull * j);
    }
}

/* D8 projection. pc = camera-space mean. Outputs proj[10] = (u, v, depth, A, B, C, opacity, r, g, b),
 * cov[3] = (a, b, c) of the filtered 2D covariance, radius, rect = (x0, x1, y0, y1). Returns tiles touched. */
uint32_t ho_project(const float attrs[11], const float pc[3], const ho_camera *cam, int32_t W, int32_t H,
                    float proj[10], float cov[3], float *radius_out, uint32_t rect[4]) {
    const float *R = cam->R;
    float s0 = attrs[0], s1 = attrs[1], s2 = attrs[2];
    float w = attrs[3], x = attrs[4], y = attrs[5], z = attrs[6];
    float M[9];
    M[0] = 1.0f - 2.0f * fmaf(y, y, z * z);
    M[1] = 2.0f * fmaf(x, y, -(w * z));
    M[2] = 2.0f * fmaf(x, z, w * y);
    M[3] = 2.0f * fmaf(x, y, w * z);
    M[4] = 1.0f - 2.0f * fmaf(x, x, z * z);
    M[5] = 2.0f * fmaf(y, z, -(w * x));
    M[6] = 2.0f * fmaf(x, z, -(w * y));
    M[7] = 2.0f * fmaf(y, z, w * x);
    M[8] = 1.0f - 2.0f * fmaf(x, x, y * y);
    float L[9];
    for (int i = 0; i < 3; ++i) {
        L[3 * i + 0] = M[3 * i + 0] * s0;
        L[3 * i + 1] = M[3 * i + 1] * s1;
        L[3 * i + 2] = M[3 * i + 2] * s2;
    }
    float S[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            S[3 * i + j] = fmaf(L[3 * i + 2], L[3 * j + 2], fmaf(L[3 * i + 1], L[3 * j + 1], L[3 * i] * L[3 * j]));
    float X = pc[0], Y = pc[1], Z = pc[2];
    float iz = 1.0f / Z, xn = X * iz, yn = Y * iz;
    float J00 = cam->fx * iz, J02 = -(cam->fx * xn) * iz;
    float J11 = cam->fy * iz, J12 = -(cam->fy * yn) * iz;
    float T0[3], T1[3];
    for (int j = 0; j < 3; ++j) {
        T0[j] = fmaf(J02, R[6 + j], J00 * R[j]);
        T1[j] = fmaf(J12, R[6 + j], J11 * R[3 + j]);
    }
    float U0[3], U1[3];
    for (int j = 0; j < 3; ++j) {
        U0[j] = fmaf(T0[2], S[6 + j], fmaf(T0[1], S[3 + j], T0[0] * S[j]));
        U1[j] = fmaf(T1[2], S[6 + j], fmaf(T1[1], S[3 + j], T1[0] * S[j]));
    }
    float a = fmaf(U0[2], T0[2], fmaf(U0[1], T0[1], U0[0] * T0[0])) + 0.3f;
    float b = fmaf(U0[2], T1[2], fmaf(U0[1], T1[1], U0[0] * T1[0]));
    float c = fmaf(U1[2], T1[2], fmaf(U1[1], T1[1], U1[0] * T1[0])) + 0.3f;
    cov[0] = a; cov[1] = b; cov[2] = c;
    float det = fmaf(a, c, -(b * b));
    float u = fmaf(cam->fx, xn, cam->cx), v = fmaf(cam->fy, yn, cam->cy);
    proj[0] = u; proj[1] = v; proj[2] = Z;
    proj[6] = attrs[7]; proj[7] = attrs[8]; proj[8] = attrs[9]; proj[9] = attrs[10];
    rect[0] = rect[1] = rect[2] = rect[3] = 0;
    *radius_out = 0.0f;
    proj[3] = proj[4] = proj[5] = 0.0f;
    if (det == 0.0f || !isfinite(det)) return 0;
    float di = 1.0f / det;
    proj[3] = c * di; proj[4] = -b * di; proj[5] = a * di;
    float mid = 0.5f * (a + c);
    float lam = mid + sqrtf(fmaxf(0.1f, fmaf(mid, mid, -det)));
    float radius = ceilf(3.0f * sqrtf(lam));
    *radius_out = radius;
    float gx = (float)((W + 15) / 16), gy = (float)((H + 15) / 16);
    float fx0 = fminf(fmaxf(floorf((u - radius) * 0.0625f), 0.0f), gx);
    float fx1 = fminf(fmaxf(floorf((u + radius + 15.0f) * 0.0625f), 0.0f), gx);
    float fy0 = fminf(fmaxf(floorf((v - radius) * 0.0625f), 0.0f), gy);
    float fy1 = fminf(fmaxf(floorf((v + radius + 15.0f) * 0.0625f), 0.0f), gy);
    if (!(fx0 == fx0) || !(fx1 == fx1) || !(fy0 == fy0) || !(fy1 == fy1)) return 0;   /* NaN */
    rect[0] = (uint32_t)fx0; rect[1] = (uint32_t)fx1; rect[2] = (uint32_t)fy0; rect[3] = (uint32_t)fy1;
    if (rect[1] <= rect[0] || rect[3] <= rect[2]) return 0;
    return (rect[1] - rect[0]) * (rect[3] - rect[2]);
}

/* S4a over all visible. Returns D = sum of tiles touched. */
uint64_t ho_stage_project(const ho_scene *s, const ho_camera *cam, int32_t W, int32_t H, uint32_t V,
                          const uint32_t *idx, const float *attrs, float *proj, float *cov, float *radius,
                          uint32_t *rect, uint32_t *tiles) {
    uint32_t n = s->n;
#pragma omp parallel for schedule(static)
    for (uint32_t j = 0; j < V; ++j) {
        uint32_t i = idx[j];
        float p[3] = {s->pos[i], s->pos[n + i], s->pos[2u * n + i]}, pc[3];
        ho_to_camera(cam, p, pc);
        tiles[j] = ho_project(attrs + 11ull * j, pc, cam, W, H, proj + 10ull * j, cov + 3ull * j, radius + j,
                              rect + 4ull * j);
    }
    uint64_t D = 0;
    for (uint32_t j = 0; j < V; ++j) D += tiles[j];
    return D;
}

/* D9 binning + order: entries (tile, depth bits, id); sort ascending by that triple. */
typedef struct { uint32_t tile, depth, id, rank; } ho_entry;

static int entry_cmp(const void *pa, const void *pb) {
    const ho_entry *a = (const ho_entry *)pa, *b = (const ho_entry *)pb;
    if (a->tile != b->tile) return a->tile < b->tile ? -1 : 1;
    if (a->depth != b->depth) return a->depth < b->depth ? -1 : 1;
    if (a->id != b->id) return a->id < b->id ? -1 : 1;
    return 0;
}

/* list_id[D] = Gaussian ids, list_rank[D] = index into the visible arrays, ranges[tiles][2] = [start,end). */
int32_t ho_stage_bin(int32_t W, int32_t H, uint32_t V, const uint32_t *idx, const float *proj,
                     const uint32_t *rect, const uint32_t *tiles, uint64_t D, uint32_t *list_id,
                     uint32_t *list_rank, uint32_t *ranges) {
    uint32_t gx = (uint32_t)((W + 15) / 16), gy = (uint32_t)((H + 15) / 16);
    ho_entry *e = (ho_entry *)malloc((D ? D : 1) * sizeof(ho_entry));
    if (!e) return -1;
    uint64_t k = 0;
    for (uint32_t j = 0; j < V; ++j) {
        if (!tiles[j]) continue;
        uint32_t depth;
        memcpy(&depth, &proj[10ull * j + 2], 4);
        const uint32_t *r = rect + 4ull * j;
        for (uint32_t ty = r[2]; ty < r[3]; ++ty)
            for (uint32_t tx = r[0]; tx < r[1]; ++tx) {
                e[k].tile = ty * gx + tx; e[k].depth = depth; e[k].id = idx[j]; e[k].rank = j;
                ++k;
            }
    }
    if (k != D) { free(e); return -2; }
    qsort(e, D, sizeof(ho_entry), entry_cmp);
    for (uint32_t t = 0; t < gx * gy; ++t) ranges[2 * t] = ranges[2 * t + 1] = 0;
    for (uint64_t q = 0; q < D; ++q) {
        list_id[q] = e[q].id;
        list_rank[q] = e[q].rank;
        if (q == 0 || e[q].tile != e[q - 1].tile) ranges[2 * e[q].tile] = (uint32_t)q;
        if (q + 1 == D || e[q].tile != e[q + 1].tile) ranges[2 * e[q].tile + 1] = (uint32_t)(q + 1);
    }
    free(e);
    return 0;
}

/* D10 per pair: alpha of projected Gaussian `proj` at pixel (i, j). Returns 0 if skipped by power > 0. */
float ho_pair_alpha(const float proj[10], float i, float j, int32_t *skipped_power) {
    float dx = proj[0] - i, dy = proj[1] - j;
    float A = proj[3], B = proj[4], C = proj[5];
    float power = fmaf(-0.5f, fmaf(A * dx, dx, (C * dy) * dy), -((B * dx) * dy));
    if (power > 0.0f) { if (skipped_power) *skipped_power = 1; return 0.0f; }
    if (skipped_power) *skipped_power = 0;
    return fminf(0.99f, proj[6] * ho_softexp(power));
}

/* D10 rasterise: Eq. 1. Per pixel outputs: cfg[3], T, and diagnostics:
 *   wsum = sum of blending weights alpha*T (for the invariant wsum + T_final = 1),
 *   m_alpha = min |alpha - 1/255| over evaluated pairs, m_stop = min |T' - 1e-4| / 1e-4 over blend decisions,
 *   n_eval = pairs evaluated (exp computed), n_blend = pairs blended. */
void ho_stage_raster(int32_t W, int32_t H, const float *proj, const uint32_t *list_rank, const uint32_t *ranges,
                     float *cfg, float *Tout, float *wsum, float *m_alpha, float *m_stop, uint32_t *n_eval,
                     uint32_t *n_blend) {
    uint32_t gx = (uint32_t)((W + 15) / 16);
#pragma omp parallel for schedule(dynamic, 16)
    for (int32_t py = 0; py < H; ++py) {
        for (int32_t px = 0; px < W; ++px) {
            uint32_t tile = (uint32_t)(py / 16) * gx + (uint32_t)(px / 16);
            uint32_t q0 = ranges[2 * tile], q1 = ranges[2 * tile + 1];
            float T = 1.0f, C0 = 0.0f, C1 = 0.0f, C2 = 0.0f, ws = 0.0f;
            float ma = INFINITY, ms = INFINITY;
            uint32_t ne = 0, nb = 0;
            for (uint32_t q = q0; q < q1; ++q) {
                const float *g = proj + 10ull * list_rank[q];
                int32_t skipped;
                float alpha = ho_pair_alpha(g, (float)px, (float)py, &skipped);
                if (skipped) continue;
                ++ne;
                ma = fminf(ma, fabsf(alpha - 1.0f / 255.0f));
                if (alpha < 1.0f / 255.0f) continue;
                float Tn = T * (1.0f - alpha);
                ms = fminf(ms, fabsf(Tn - 1e-4f) / 1e-4f);
                if (Tn < 1e-4f) break;
                float wgt = alpha * T;
                C0 = fmaf(g[7], wgt, C0); C1 = fmaf(g[8], wgt, C1); C2 = fmaf(g[9], wgt, C2);
                ws += wgt;
                T = Tn;
                ++nb;
            }
            uint64_t o = (uint64_t)py * (uint64_t)W + (uint64_t)px;
            cfg[3 * o] = C0; cfg[3 * o + 1] = C1; cfg[3 * o + 2] = C2;
            Tout[o] = T;
            if (wsum) wsum[o] = ws;
            if (m_alpha) m_alpha[o] = ma;
            if (m_stop) m_stop[o] = ms;
            if (n_eval) n_eval[o] = ne;
            if (n_blend) n_blend[o] = nb;
        }
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* D12 backward of D10 (first piece; the training of PAPER.md:136-142 back-propagates through the
 * 3DGS rasterizer the paper defers to, :108). The decisions of the forward pass are frozen: for every pixel, the
 * set of blended pairs is the one D10 takes in binary32. On that set C_fg = sum_k c_k a_k T_k and
 * T_final = prod_k (1 - a_k), with T_k = prod_{m<k} (1 - a_m), a_k = min(0.99, o_k exp(power_k)),
 * power = -0.5 (A dx^2 + C dy^2) - B dx dy, dx = u - i, dy = v - j. Given g_cfg = dL/dC_fg and g_T = dL/dT_final:
 *   dL/dc_k    += a_k T_k g_cfg
 *   dL/da_k     = sum_c g_cfg_c (c_kc T_k - S_kc / (1 - a_k)) - g_T T_final / (1 - a_k),  S_k = sum_{m>k} c_m a_m T_m
 *   a_k clamped at 0.99: nothing flows to o, power. Else dL/do += exp(power) dL/da, dL/dpower = a dL/da, and
 *   dA += -0.5 dx^2 dP, dC += -0.5 dy^2 dP, dB += -dx dy dP, du += -(A dx + B dy) dP, dv += -(C dy + B dx) dP.
 * The forward replay is D10's binary32; everything after it is binary64. grad: [V][9] = (u, v, A, B, C, o, r, g, b). */
void ho_stage_raster_backward(int32_t W, int32_t H, uint32_t V, const float *proj, const uint32_t *list_rank,
                              const uint32_t *ranges, const float *g_cfg, const float *g_T, double *grad) {
    uint32_t gx = (uint32_t)((W + 15) / 16), gy = (uint32_t)((H + 15) / 16);
    uint32_t maxlen = 1;
    for (uint32_t t = 0; t < gx * gy; ++t)
        if (ranges[2 * t + 1] - ranges[2 * t] > maxlen) maxlen = ranges[2 * t + 1] - ranges[2 * t];
    memset(grad, 0, (size_t)V * 9 * sizeof(double));
#pragma omp parallel
    {
        uint32_t *bq = (uint32_t *)malloc((size_t)maxlen * sizeof(uint32_t));
        float *ba = (float *)malloc((size_t)maxlen * sizeof(float));
        float *bT = (float *)malloc((size_t)maxlen * sizeof(float));
        float *be = (float *)malloc((size_t)maxlen * sizeof(float));
#pragma omp for schedule(dynamic, 4)
        for (int32_t py = 0; py < H; ++py) {
            for (int32_t px = 0; px < W; ++px) {
                uint32_t tile = (uint32_t)(py / 16) * gx + (uint32_t)(px / 16);
                uint32_t q0 = ranges[2 * tile], q1 = ranges[2 * tile + 1], nb = 0;
                float T = 1.0f;
                for (uint32_t q = q0; q < q1; ++q) {          /* D10, decisions in binary32 */
                    const float *g = proj + 10ull * list_rank[q];
                    float dx = g[0] - (float)px, dy = g[1] - (float)py;
                    float power = fmaf(-0.5f, fmaf(g[3] * dx, dx, (g[5] * dy) * dy), -((g[4] * dx) * dy));
                    if (power > 0.0f) continue;
                    float e = ho_softexp(power);
                    float alpha = fminf(0.99f, g[6] * e);
                    if (alpha < 1.0f / 255.0f) continue;
                    float Tn = T * (1.0f - alpha);
                    if (Tn < 1e-4f) break;
                    bq[nb] = q; ba[nb] = alpha; bT[nb] = T; be[nb] = (g[6] * e > 0.99f) ? -1.0f : e;
                    ++nb;
                    T = Tn;
                }
                uint64_t o = (uint64_t)py * (uint64_t)W + (uint64_t)px;
                const double gc[3] = {g_cfg[3 * o], g_cfg[3 * o + 1], g_cfg[3 * o + 2]};
                const double gT = g_T[o], Tfin = T;
                double S[3] = {0.0, 0.0, 0.0};
                for (uint32_t n = nb; n-- > 0;) {
                    uint32_t r = list_rank[bq[n]];
                    const float *g = proj + 10ull * r;
                    double a = ba[n], Tk = bT[n], w = a * Tk, da = 0.0;
                    double *G = grad + 9ull * r;
                    for (int c = 0; c < 3; ++c) {
                        da += gc[c] * ((double)g[7 + c] * Tk - S[c] / (1.0 - a));
#pragma omp atomic
                        G[6 + c] += w * gc[c];
                    }
                    da -= gT * Tfin / (1.0 - a);
                    for (int c = 0; c < 3; ++c) S[c] += (double)g[7 + c] * w;
                    if (be[n] < 0.0f) continue;               /* clamped at 0.99 */
                    double dx = (double)g[0] - (double)px, dy = (double)g[1] - (double)py, dP = a * da;
                    double A = g[3], B = g[4], C = g[5];
                    double add[6] = {-(A * dx + B * dy) * dP, -(C * dy + B * dx) * dP, -0.5 * dx * dx * dP,
                                     -dx * dy * dP, -0.5 * dy * dy * dP, (double)be[n] * da};
                    for (int k = 0; k < 6; ++k) {
#pragma omp atomic
                        G[k] += add[k];
                    }
                }
            }
        }
        free(bq); free(ba); free(bT); free(be);
    }
}

/* D11: ray direction of pixel (i, j) and its hit point on the background sphere. */
void ho_ray_sphere(const ho_camera *cam, float i, float j, float radius, float d[3], float ps[3]) {
    const float *R = cam->R;
    float o[3];
    ho_camera_center(cam, o);
    float dc[3] = {(i - cam->cx) / cam->fx, (j - cam->cy) / cam->fy, 1.0f};
    float dw[3];
    for (int k = 0; k < 3; ++k) dw[k] = fmaf(R[6 + k], dc[2], fmaf(R[3 + k], dc[1], R[k] * dc[0]));
    float n = sqrtf(fmaf(dw[2], dw[2], fmaf(dw[1], dw[1], dw[0] * dw[0])));
    for (int k = 0; k < 3; ++k) d[k] = dw[k] / n;
    float Bq = 2.0f * fmaf(o[2], d[2], fmaf(o[1], d[1], o[0] * d[0]));
    float Cq = fmaf(o[2], o[2], fmaf(o[1], o[1], o[0] * o[0])) - radius * radius;
    float disc = fmaf(Bq, Bq, -4.0f * Cq);
    float t = 0.5f * (-Bq + sqrtf(disc));
    for (int k = 0; k < 3; ++k) ps[k] = fmaf(t, d[k], o[k]);
}

/* D11 background colour for one pixel: c_s = sigmoid(dec(enc(p_s) (+) PE(d))). */
void ho_background_color(const ho_scene *s, const ho_camera *cam, float i, float j, float cs[3]) {
    float d[3], ps[3], x[3], in[HO_MAX_DIM], raw[3];
    ho_ray_sphere(cam, i, j, s->bg_radius, d, ps);
    ho_contract(ps, s->aabb_min, s->aabb_max, x);
    memset(in, 0, sizeof(in));
    ho_grid_encode_q(&s->bg_grid, s->bg_table, s->table_u8 ? 2 : s->fp16, s->bg_q, x, in);
    ho_dir_pe(d, s->pe_octaves, s->fp16, in + s->bg_grid.levels * s->bg_grid.feats);
    ho_mlp_forward(&s->bg_mlp, s->bg_w, s->fp16, in, raw);
    for (int k = 0; k < 3; ++k) cs[k] = ho_sigmoid(raw[k]);
}

/* S6: composite (Eq. 10-11) where T > tau_T (reading A17). bg_mask marks composited pixels. */
void ho_stage_background(const ho_scene *s, const ho_camera *cam, int32_t W, int32_t H, const float *cfg,
                         const float *T, float *out, uint8_t *bg_mask) {
#pragma omp parallel for schedule(dynamic, 8)
    for (int32_t py = 0; py < H; ++py) {
        for (int32_t px = 0; px < W; ++px) {
            uint64_t o = (uint64_t)py * (uint64_t)W + (uint64_t)px;
            float t = T[o];
            if (t > s->tau_T) {
                float cs[3];
                ho_background_color(s, cam, (float)px, (float)py, cs);
                for (int k = 0; k < 3; ++k) out[3 * o + k] = fmaf(t, cs[k], cfg[3 * o + k]);
                if (bg_mask) bg_mask[o] = 1;
            } else {
                for (int k = 0; k < 3; ++k) out[3 * o + k] = cfg[3 * o + k];
                if (bg_mask) bg_mask[o] = 0;
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* Compressed explicit Gaussians (PAPER.md:227-229 items 1-2; DESIGN.md §2 D1'): positions stored as IEEE binary16,
 * the five explicit properties (s_e, alpha_e, c_e[0..2]) as residual vector quantisation codes. The paper names
 * R-VQ and gives no formula; this is the textbook decode: the reconstruction is the sum over stages of one
 * codebook row per stage, x = C_0[k_0] + C_1[k_1] + ... + C_{S-1}[k_{S-1}], added in binary32 in stage order
 * (left to right, starting from the stage-0 row itself).
 *   pos_h      [3][n] binary16 bit patterns (SoA like the fp32 positions)
 *   codes      [S][n] uint16, codes[s][i] < K
 *   codebooks  [S][K][5] binary32, columns (s_e, alpha_e, c_e[0], c_e[1], c_e[2])
 * outputs in the layout of ho_scene: pos [3][n], scale_logit [n], opacity_logit [n], rgb_logit [3][n].
 * Returns 0, or 1 + the index of the first Gaussian with a code >= K (nothing is written for it). */
uint32_t ho_decode_explicit(uint32_t n, const uint16_t *pos_h, uint32_t S, uint32_t K, const uint16_t *codes,
                            const float *codebooks, float *pos, float *scale_logit, float *opacity_logit,
                            float *rgb_logit) {
    for (uint32_t i = 0; i < n; ++i) {
        float x[5];
        for (uint32_t s = 0; s < S; ++s) {
            const uint32_t k = codes[(size_t)s * n + i];
            if (k >= K) return 1u + i;
            const float *row = codebooks + ((size_t)s * K + k) * 5;
            for (int d = 0; d < 5; ++d) x[d] = (s == 0) ? row[d] : x[d] + row[d];
        }
        for (int a = 0; a < 3; ++a) pos[(size_t)a * n + i] = ho_half_to_float(pos_h[(size_t)a * n + i]);
        scale_logit[i] = x[0];
        opacity_logit[i] = x[1];
        for (int c = 0; c < 3; ++c) rgb_logit[(size_t)c * n + i] = x[2 + c];
    }
    return 0;
}

int32_t ho_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void ho_set_num_threads(int32_t n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
