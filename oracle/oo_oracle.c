/*
 * oo_oracle.c — CPU ORACLE (plain C, double precision) for the OctaOctree per-query radiance evaluation.
 *
 * TEST INFRASTRUCTURE ONLY: used by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs. It shares no code, header, table or constant with the CUDA path and is a
 * second, independent restatement of oracle/oo_oracle.py (the two are cross-checked to 1e-12).
 *
 * One query at a time, in the paper's order (/root/reference/PAPER.md cited as P:line; readings A1-A24
 * in DESIGN.md):
 *   O1 quantise  O2 descend the sparse octree  O3 octahedral projection, Eq. 4-5
 *   O4 remap to [0,1]^2 and to texel coordinates  O5 wrap taps across octahedron edges
 *   O6 bilinear, 4 taps, nearest cell  O7 concatenate levels and attributes (Eq. 11-13)
 *   O8 decoder MLP: H x (linear, ReLU), linear, exp.
 * Double everywhere, except the base-texel decision, which is taken in fp32 by the fixed operation
 * sequence of DESIGN.md "Index contract" (this file must be compiled with -ffp-contract=off).
 *
 * No blocking, no vectorisation tricks, no reordering: OpenMP `parallel for` over queries is the only
 * concession, so that the full-size configs finish in seconds.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC -o liboo_oracle.so oo_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_API __attribute__((visibility("default")))

enum { ORACLE_F16 = 0, ORACLE_F32 = 1 };
enum { ORACLE_ACT_NONE = 0, ORACLE_ACT_EXP = 1 };
enum { MAX_LEVELS = 16, MAX_LAYERS = 16, MAX_DIM = 512 };

typedef struct {
    uint32_t n_nodes, max_depth;
    const int32_t* child;      /* [n_nodes][8] */
    const int32_t* map_slot;   /* [n_nodes] */
    uint32_t n_levels;
    uint32_t level_depth[MAX_LEVELS];
    uint32_t level_res[MAX_LEVELS];
    uint32_t n_features;
    int32_t dtype;             /* ORACLE_F16 / ORACLE_F32 */
    const void* atlas[MAX_LEVELS];   /* [slots][R][R][F] */
} oracle_tree;

typedef struct {
    uint32_t in_dim, width, n_hidden, out_dim;
    const uint16_t* weights[MAX_LAYERS];  /* fp16 bits, row-major [out][in] */
    int32_t out_act;
} oracle_mlp;

/* exact widening of IEEE binary16 to double */
static double half_to_double(uint16_t h) {
    int s = h >> 15, e = (h >> 10) & 31, m = h & 1023;
    double v;
    if (e == 0) v = ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp((double)(1024 + m), e - 25);
    return s ? -v : v;
}

static double texel(const oracle_tree* t, int l, int64_t slot, int j, int i, int c) {
    int64_t R = t->level_res[l], F = t->n_features;
    int64_t idx = ((slot * R + j) * R + i) * F + c;
    if (t->dtype == ORACLE_F16) return half_to_double(((const uint16_t*)t->atlas[l])[idx]);
    return (double)((const float*)t->atlas[l])[idx];
}

/* O5: continuation across the crossed edge = point reflection about that edge's midpoint. */
static void wrap_tap(int* i, int* j, int R) {
    if (*i < 0) { *i = 0; *j = R - 1 - *j; }
    else if (*i >= R) { *i = R - 1; *j = R - 1 - *j; }
    if (*j < 0) { *j = 0; *i = R - 1 - *i; }
    else if (*j >= R) { *j = R - 1; *i = R - 1 - *i; }
}

/* The index contract: fp32, one rounding per operation (compile with -ffp-contract=off). */
static void base_texel_f32(const float w[3], int R, int* i0, int* j0) {
    float S = (fabsf(w[0]) + fabsf(w[1])) + fabsf(w[2]);
    float ux = w[0] / S, uy = w[1] / S;
    if (w[2] < 0.0f) {
        float tx = 1.0f - fabsf(uy), ty = 1.0f - fabsf(ux);
        float nx = (ux >= 0.0f) ? tx : -tx, ny = (uy >= 0.0f) ? ty : -ty;
        ux = nx; uy = ny;
    }
    float hr = (float)R * 0.5f, off = (float)R * 0.5f - 0.5f;
    volatile float px = ux * hr, py = uy * hr;      /* exact products (hr is a power of two) */
    float sx = px + off, sy = py + off;
    *i0 = (int)floorf(sx); *j0 = (int)floorf(sy);
}

/* O1-O6 for one query. feat[L*F] double, slot[L], tex[L][2]. */
static void encode_one(const oracle_tree* t, const float x[3], const float wo[3], double* feat, int32_t* slot,
                       int16_t* tex) {
    int D = (int)t->max_depth, L = (int)t->n_levels, F = (int)t->n_features;
    /* O1 */
    int64_t q[3], ncell = (int64_t)1 << D;
    for (int a = 0; a < 3; ++a) {
        double v = floor((double)x[a] * (double)ncell);
        if (v < 0) v = 0;
        if (v > (double)(ncell - 1)) v = (double)(ncell - 1);
        q[a] = (int64_t)v;
    }
    /* O2 */
    int64_t path[40];
    for (int d = 0; d <= D; ++d) path[d] = -1;
    int64_t node = 0; path[0] = 0;
    for (int d = 1; d <= D; ++d) {
        int s = D - d;
        int o = (int)(((q[0] >> s) & 1) | (((q[1] >> s) & 1) << 1) | (((q[2] >> s) & 1) << 2));
        node = t->child[8 * node + o];
        if (node < 0) break;
        path[d] = node;
    }
    /* O3 */
    double w[3] = {(double)wo[0], (double)wo[1], (double)wo[2]};
    double S = fabs(w[0]) + fabs(w[1]) + fabs(w[2]);
    double ux = w[0] / S, uy = w[1] / S;
    if (w[2] < 0.0) {
        double fx = (1.0 - fabs(uy)) * (ux >= 0.0 ? 1.0 : -1.0);
        double fy = (1.0 - fabs(ux)) * (uy >= 0.0 ? 1.0 : -1.0);
        ux = fx; uy = fy;
    }
    for (int l = 0; l < L; ++l) {
        int R = (int)t->level_res[l];
        int64_t nd = path[t->level_depth[l]];
        int64_t sl = nd >= 0 ? t->map_slot[nd] : -1;
        /* O4 */
        double sx = (ux + 1.0) / 2.0 * R - 0.5, sy = (uy + 1.0) / 2.0 * R - 0.5;
        int i0, j0;
        base_texel_f32(wo, R, &i0, &j0);
        double fx = sx - i0, fy = sy - j0;
        if (slot) slot[l] = (int32_t)sl;
        if (tex) { tex[2 * l] = (int16_t)i0; tex[2 * l + 1] = (int16_t)j0; }
        for (int c = 0; c < F; ++c) feat[l * F + c] = 0.0;
        if (sl < 0) continue;
        /* O5, O6 */
        for (int b = 0; b < 2; ++b)
            for (int a = 0; a < 2; ++a) {
                double wgt = (a ? fx : 1.0 - fx) * (b ? fy : 1.0 - fy);
                int i = i0 + a, j = j0 + b;
                wrap_tap(&i, &j, R);
                for (int c = 0; c < F; ++c) feat[l * F + c] += wgt * texel(t, l, sl, j, i, c);
            }
    }
}

/* O8.  W[layer] = the fp16 weights widened exactly to double (done once per call, see oracle_query). */
static void mlp_one(const oracle_mlp* m, double* const* W, const double* in, double* rgb) {
    double a[MAX_DIM], b[MAX_DIM];
    int n_in = (int)m->in_dim;
    for (int k = 0; k < n_in; ++k) a[k] = in[k];
    for (uint32_t layer = 0; layer <= m->n_hidden; ++layer) {
        int n_out = layer == m->n_hidden ? (int)m->out_dim : (int)m->width;
        for (int o = 0; o < n_out; ++o) {
            double acc = 0.0;
            for (int k = 0; k < n_in; ++k) acc += W[layer][(size_t)o * n_in + k] * a[k];
            if (layer < m->n_hidden) acc = acc > 0.0 ? acc : 0.0;
            b[o] = acc;
        }
        for (int o = 0; o < n_out; ++o) a[o] = b[o];
        n_in = n_out;
    }
    for (uint32_t o = 0; o < m->out_dim; ++o) rgb[o] = m->out_act == ORACLE_ACT_EXP ? exp(a[o]) : a[o];
}

ORACLE_API int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* features [n][L*F] double; slot [n][L] and tex [n][L][2] optional. n_threads <= 0: all cores. Returns threads used. */
ORACLE_API int oracle_encode(const oracle_tree* t, uint64_t n, const float* x, const float* wo, double* feat,
                             int32_t* slot, int16_t* tex, int n_threads) {
    int L = (int)t->n_levels, F = (int)t->n_features, used = 1;
    if (L > MAX_LEVELS || L * F > MAX_DIM) return -1;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
    used = n_threads;
#pragma omp parallel for schedule(static) num_threads(n_threads)
#endif
    for (int64_t k = 0; k < (int64_t)n; ++k)
        encode_one(t, x + 3 * k, wo + 3 * k, feat + (size_t)k * L * F, slot ? slot + (size_t)k * L : NULL,
                   tex ? tex + (size_t)k * L * 2 : NULL);
    return used;
}

/* rgb [n][out_dim] double. extra [n][n_extra] or NULL. Returns threads used, <0 on bad arguments. */
ORACLE_API int oracle_query(const oracle_tree* t, const oracle_mlp* m, uint64_t n, const float* x, const float* nrm,
                            const float* wo, const float* extra, uint32_t n_extra, double* rgb, int n_threads) {
    int L = (int)t->n_levels, F = (int)t->n_features, used = 1;
    if (L > MAX_LEVELS || m->n_hidden + 1 > MAX_LAYERS || m->in_dim > MAX_DIM || m->width > MAX_DIM) return -1;
    if ((uint32_t)(L * F) + 6 + n_extra != m->in_dim) return -2;
    double* W[MAX_LAYERS];
    for (uint32_t layer = 0; layer <= m->n_hidden; ++layer) {
        size_t n_in = layer == 0 ? m->in_dim : m->width, n_out = layer == m->n_hidden ? m->out_dim : m->width;
        W[layer] = (double*)malloc(n_in * n_out * sizeof(double));
        if (!W[layer]) return -3;
        for (size_t k = 0; k < n_in * n_out; ++k) W[layer][k] = half_to_double(m->weights[layer][k]);
    }
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
    used = n_threads;
#pragma omp parallel for schedule(static) num_threads(n_threads)
#endif
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        double in[MAX_DIM];
        encode_one(t, x + 3 * k, wo + 3 * k, in, NULL, NULL);
        /* O7 */
        int p = L * F;
        for (int a = 0; a < 3; ++a) in[p++] = (double)nrm[3 * k + a];
        for (int a = 0; a < 3; ++a) in[p++] = (double)wo[3 * k + a];
        for (uint32_t e = 0; e < n_extra; ++e) in[p++] = (double)extra[(size_t)k * n_extra + e];
        mlp_one(m, W, in, rgb + (size_t)k * m->out_dim);
    }
    for (uint32_t layer = 0; layer <= m->n_hidden; ++layer) free(W[layer]);
    return used;
}
