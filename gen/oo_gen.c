/*
 * oo_gen.c — seeded synthetic INPUT generators for the OctaOctree query path.
 *
 * This file produces inputs only (random numbers, scenes, octrees, camera rays). It holds none of
 * the method's arithmetic (no octree descent, no octahedral map, no interpolation, no MLP): both
 * the CPU oracle (oracle/) and the CUDA path (paper_2606_08469_b200/) consume the bytes written
 * here and share nothing else.  Recipe: DESIGN.md "Input recipe" (restating BASELINE.json configs
 * 0-4 and SURVEY.md §8(d)).
 *
 * Counter-based RNG: value(seed, stream, idx) = SplitMix64 finaliser applied twice to a mix of the
 * three counters; uniform double in [0,1) from the top 53 bits.  Any element can be generated
 * independently of any other, so atlases can be generated in parallel and re-generated lazily.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liboo_gen.so oo_gen.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OO_GEN_API __attribute__((visibility("default")))

/* ------------------------------------------------------------------------------------------ RNG */

static inline uint64_t mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

static inline uint64_t ctr_bits(uint64_t seed, uint64_t stream, uint64_t idx) {
    uint64_t k = mix64(seed * 0x9E3779B97F4A7C15ULL + stream * 0xD1B54A32D192ED03ULL + 0x632BE59BD9B4E019ULL);
    return mix64(k + (idx + 1) * 0x9E3779B97F4A7C15ULL);
}

static inline double ctr_u01(uint64_t seed, uint64_t stream, uint64_t idx) {
    return (double)(ctr_bits(seed, stream, idx) >> 11) * (1.0 / 9007199254740992.0);
}

/* Box-Muller in double; element idx consumes counters 2*idx and 2*idx+1. */
static inline double ctr_normal(uint64_t seed, uint64_t stream, uint64_t idx) {
    double u1 = 1.0 - ctr_u01(seed, stream, 2 * idx);       /* (0,1] */
    double u2 = ctr_u01(seed, stream, 2 * idx + 1);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* double -> IEEE binary16, round-to-nearest-even, one rounding (no float intermediate). */
static inline uint16_t f64_to_f16_rne(double d) {
    uint64_t b; memcpy(&b, &d, 8);
    uint16_t sign = (uint16_t)((b >> 48) & 0x8000u);
    int ebits = (int)((b >> 52) & 0x7ff);
    uint64_t m = b & 0xFFFFFFFFFFFFFULL;
    if (ebits == 0x7ff) return (uint16_t)(sign | 0x7c00u | (m ? 0x200u : 0u));
    int e = ebits - 1023;
    if (ebits == 0) return sign;                 /* double zero / subnormal -> 0 */
    if (e > 15) return (uint16_t)(sign | 0x7c00u);
    if (e >= -14) {
        uint32_t h = ((uint32_t)(e + 15) << 10) | (uint32_t)(m >> 42);
        uint64_t rem = m & ((1ULL << 42) - 1), half = 1ULL << 41;
        if (rem > half || (rem == half && (h & 1u))) h++;
        return (uint16_t)(sign | h);             /* a carry into 0x7c00 is +-inf, as it should be */
    }
    if (e >= -25) {
        uint64_t full = (1ULL << 52) | m;
        int shift = 42 + (-14 - e);              /* result in units of 2^-24 */
        uint32_t h = (uint32_t)(full >> shift);
        uint64_t rem = full & ((1ULL << shift) - 1), half = 1ULL << (shift - 1);
        if (rem > half || (rem == half && (h & 1u))) h++;
        return (uint16_t)(sign | h);
    }
    return sign;
}

OO_GEN_API void oo_gen_u01(uint64_t seed, uint64_t stream, uint64_t first, uint64_t n, double* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) out[i] = ctr_u01(seed, stream, first + (uint64_t)i);
}

OO_GEN_API void oo_gen_normal(uint64_t seed, uint64_t stream, uint64_t first, uint64_t n, double* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) out[i] = ctr_normal(seed, stream, first + (uint64_t)i);
}

/* out[i] = fp16( std * N(0,1) ), element index first+i */
OO_GEN_API void oo_gen_normal_f16(uint64_t seed, uint64_t stream, uint64_t first, uint64_t n, double std,
                                  uint16_t* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i)
        out[i] = f64_to_f16_rne(std * ctr_normal(seed, stream, first + (uint64_t)i));
}

/* out[i] = fp32( lo + (hi-lo) * U[0,1) ) */
OO_GEN_API void oo_gen_uniform_f32(uint64_t seed, uint64_t stream, uint64_t first, uint64_t n, double lo,
                                   double hi, float* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i)
        out[i] = (float)(lo + (hi - lo) * ctr_u01(seed, stream, first + (uint64_t)i));
}

OO_GEN_API void oo_gen_f64_to_f16(const double* in, uint64_t n, uint16_t* out) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) out[i] = f64_to_f16_rne(in[i]);
}

/* Uniform direction on the unit sphere: z = 1-2 xi1, phi = 2 pi xi2 (counters 2*idx, 2*idx+1). */
static inline void ctr_sphere(uint64_t seed, uint64_t stream, uint64_t idx, double w[3]) {
    double z = 1.0 - 2.0 * ctr_u01(seed, stream, 2 * idx);
    double phi = 6.283185307179586476925286766559 * ctr_u01(seed, stream, 2 * idx + 1);
    double r = sqrt(fmax(0.0, 1.0 - z * z));
    w[0] = r * cos(phi); w[1] = r * sin(phi); w[2] = z;
}

/* n ~ uniform sphere (stream_n); wo ~ uniform sphere (stream_w), negated if wo.n < 0 (hemisphere about n). */
OO_GEN_API void oo_gen_normals_and_dirs(uint64_t seed, uint64_t stream_n, uint64_t stream_w, uint64_t first,
                                        uint64_t n, float* nrm, float* wo) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        double a[3], w[3];
        ctr_sphere(seed, stream_n, first + (uint64_t)i, a);
        ctr_sphere(seed, stream_w, first + (uint64_t)i, w);
        if (a[0] * w[0] + a[1] * w[1] + a[2] * w[2] < 0.0) { w[0] = -w[0]; w[1] = -w[1]; w[2] = -w[2]; }
        for (int k = 0; k < 3; ++k) { nrm[3 * i + k] = (float)a[k]; wo[3 * i + k] = (float)w[k]; }
    }
}

/* ---------------------------------------------------------------------------------------- scene */
/* A scene = n_spheres spheres (cx,cy,cz,r) + a 5-plane box: x=lo, x=hi, y=lo, y=hi, z=lo, each a
 * rectangle spanning [lo,hi] on the other two axes; open towards +z. */

typedef struct {
    int32_t n_spheres;
    const double* spheres;  /* [n_spheres][4] */
    double lo, hi;          /* box planes */
    double eps;             /* cell dilation for the tree builder */
} oo_scene;

enum { N_PLANES = 5 };
static const int plane_axis[N_PLANES] = {0, 0, 1, 1, 2};
static const int plane_side[N_PLANES] = {0, 1, 0, 1, 0};   /* 0: at lo, 1: at hi */

/* does surface s (0..n_spheres-1 spheres, then planes) intersect the cube [c0,c1]^3 dilated by eps? */
static inline int surf_hits_cube(const oo_scene* sc, int s, const double c0[3], const double c1[3]) {
    double e = sc->eps;
    if (s < sc->n_spheres) {
        const double* sp = sc->spheres + 4 * s;
        double dmin2 = 0.0, dmax2 = 0.0;
        for (int a = 0; a < 3; ++a) {
            double lo = c0[a] - e, hi = c1[a] + e, c = sp[a];
            double dlo = c < lo ? lo - c : (c > hi ? c - hi : 0.0);
            double dhi = fmax(fabs(c - lo), fabs(c - hi));
            dmin2 += dlo * dlo; dmax2 += dhi * dhi;
        }
        double r2 = sp[3] * sp[3];
        return dmin2 <= r2 && r2 <= dmax2;
    }
    int p = s - sc->n_spheres, ax = plane_axis[p];
    double pos = plane_side[p] ? sc->hi : sc->lo;
    if (pos < c0[ax] - e || pos > c1[ax] + e) return 0;
    for (int a = 0; a < 3; ++a) {
        if (a == ax) continue;
        if (c1[a] + e < sc->lo || c0[a] - e > sc->hi) return 0;
    }
    return 1;
}

/* ------------------------------------------------------------------------------------ tree build */
/* BFS from the root; children created in octant order o = bx | by<<1 | bz<<2, so every depth is in
 * Morton order; node id = BFS index.  A child exists iff its (dilated) cube intersects a surface, or
 * always when `uniform` is set.  Outputs are malloc'ed here; free with oo_gen_free. */

typedef struct {
    uint32_t n_nodes;
    int32_t* child;        /* [n_nodes][8] */
    uint8_t* depth;        /* [n_nodes] */
    uint32_t* coords;      /* [n_nodes][3] integer cell coords at the node's depth */
    uint32_t depth_first[34]; /* first node id of each depth; depth_first[max_depth+1] = n_nodes */
} oo_tree_out;

OO_GEN_API void oo_gen_free(void* p) { free(p); }

OO_GEN_API int oo_gen_build_tree(const oo_scene* sc, uint32_t max_depth, int uniform, oo_tree_out* out) {
    if (max_depth > 16) return 1;
    int n_surf = sc ? sc->n_spheres + N_PLANES : 0;
    size_t cap = 1024;
    int32_t* child = malloc(cap * 8 * sizeof(int32_t));
    uint8_t* depth = malloc(cap);
    uint32_t* coords = malloc(cap * 3 * sizeof(uint32_t));
    /* candidate surface lists per node of the current and next BFS level */
    size_t ccap_cur = 1 << 16, ccap = 1 << 16;     /* ccap = capacity of cand_nxt */
    int32_t* cand_cur = malloc(ccap_cur * sizeof(int32_t));
    int32_t* cand_nxt = malloc(ccap * sizeof(int32_t));
    size_t lcap = 1024;
    uint64_t* off_cur = malloc((lcap + 1) * sizeof(uint64_t));
    uint64_t* off_nxt = malloc((lcap + 1) * sizeof(uint64_t));
    if (!child || !depth || !coords || !cand_cur || !cand_nxt || !off_cur || !off_nxt) return 2;

    uint32_t n = 1;
    for (int o = 0; o < 8; ++o) child[o] = -1;
    depth[0] = 0; coords[0] = coords[1] = coords[2] = 0;
    off_cur[0] = 0;
    for (int s = 0; s < n_surf; ++s) cand_cur[s] = s;
    off_cur[1] = (uint64_t)n_surf;
    out->depth_first[0] = 0;
    uint32_t level_first = 0, level_count = 1;

    for (uint32_t d = 0; d < max_depth; ++d) {
        out->depth_first[d + 1] = n;
        double cw = ldexp(1.0, -(int)(d + 1));   /* child cell width */
        uint32_t nxt_count = 0;
        uint64_t nxt_used = 0;
        for (uint32_t k = 0; k < level_count; ++k) {
            uint32_t id = level_first + k;
            const int32_t* cl = cand_cur + off_cur[k];
            int ncl = (int)(off_cur[k + 1] - off_cur[k]);
            for (int o = 0; o < 8; ++o) {
                uint32_t cx = coords[3 * id] * 2 + (o & 1), cy = coords[3 * id + 1] * 2 + ((o >> 1) & 1),
                         cz = coords[3 * id + 2] * 2 + ((o >> 2) & 1);
                double c0[3] = {cx * cw, cy * cw, cz * cw};
                double c1[3] = {(cx + 1) * cw, (cy + 1) * cw, (cz + 1) * cw};
                if (nxt_used + (uint64_t)n_surf + 1 > ccap) {
                    while (nxt_used + (uint64_t)n_surf + 1 > ccap) ccap *= 2;
                    cand_nxt = realloc(cand_nxt, ccap * sizeof(int32_t));
                    if (!cand_nxt) return 2;
                }
                int kept = 0;
                for (int t = 0; t < ncl; ++t)
                    if (surf_hits_cube(sc, cl[t], c0, c1)) cand_nxt[nxt_used + kept++] = cl[t];
                if (!uniform && kept == 0) continue;
                if (n + 1 > cap) {
                    cap *= 2;
                    child = realloc(child, cap * 8 * sizeof(int32_t));
                    depth = realloc(depth, cap);
                    coords = realloc(coords, cap * 3 * sizeof(uint32_t));
                    if (!child || !depth || !coords) return 2;
                }
                if ((size_t)nxt_count + 2 > lcap) {
                    lcap *= 2;
                    off_nxt = realloc(off_nxt, (lcap + 1) * sizeof(uint64_t));
                    off_cur = realloc(off_cur, (lcap + 1) * sizeof(uint64_t));
                    if (!off_nxt || !off_cur) return 2;
                }
                child[8 * (size_t)id + o] = (int32_t)n;
                for (int q = 0; q < 8; ++q) child[8 * (size_t)n + q] = -1;
                depth[n] = (uint8_t)(d + 1);
                coords[3 * (size_t)n] = cx; coords[3 * (size_t)n + 1] = cy; coords[3 * (size_t)n + 2] = cz;
                off_nxt[nxt_count] = nxt_used;
                nxt_used += (uint64_t)kept;
                off_nxt[nxt_count + 1] = nxt_used;
                ++nxt_count; ++n;
            }
        }
        /* swap levels */
        int32_t* tc = cand_cur; cand_cur = cand_nxt; cand_nxt = tc;
        size_t tcap = ccap_cur; ccap_cur = ccap; ccap = tcap;
        uint64_t* to = off_cur; off_cur = off_nxt; off_nxt = to;
        level_first += level_count;
        level_count = nxt_count;
        if (level_count == 0) {           /* nothing deeper: fill the remaining depth_first entries */
            for (uint32_t dd = d + 1; dd <= max_depth; ++dd) out->depth_first[dd + 1] = n;
            break;
        }
    }
    out->depth_first[max_depth + 1] = n;
    free(cand_cur); free(cand_nxt); free(off_cur); free(off_nxt);
    out->n_nodes = n; out->child = child; out->depth = depth; out->coords = coords;
    return 0;
}

/* --------------------------------------------------------------------------------------- camera */

typedef struct {
    double eye[3], look[3], up[3];
    double vfov_deg;
    uint32_t width, height;
} oo_camera;

static inline void norm3(double v[3]) {
    double l = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    v[0] /= l; v[1] /= l; v[2] /= l;
}
static inline void cross3(const double a[3], const double b[3], double c[3]) {
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}

/* nearest hit of ray o + t d (t > tmin) with the scene; returns surface id or -1, fills t and normal
 * (sphere: outward; plane: pointing into the box). */
static int scene_hit(const oo_scene* sc, const double o[3], const double d[3], double* t_out, double nrm[3]) {
    double best = INFINITY; int bs = -1;
    const double tmin = 1e-9;
    for (int s = 0; s < sc->n_spheres; ++s) {
        const double* sp = sc->spheres + 4 * s;
        double oc[3] = {o[0] - sp[0], o[1] - sp[1], o[2] - sp[2]};
        double b = oc[0] * d[0] + oc[1] * d[1] + oc[2] * d[2];
        double c = oc[0] * oc[0] + oc[1] * oc[1] + oc[2] * oc[2] - sp[3] * sp[3];
        double disc = b * b - c;
        if (disc < 0.0) continue;
        double sq = sqrt(disc), t = -b - sq;
        if (t <= tmin) t = -b + sq;
        if (t > tmin && t < best) { best = t; bs = s; }
    }
    for (int p = 0; p < N_PLANES; ++p) {
        int ax = plane_axis[p];
        double pos = plane_side[p] ? sc->hi : sc->lo;
        if (d[ax] == 0.0) continue;
        double t = (pos - o[ax]) / d[ax];
        if (t <= tmin || t >= best) continue;
        int ok = 1;
        for (int a = 0; a < 3; ++a) {
            if (a == ax) continue;
            double q = o[a] + t * d[a];
            if (q < sc->lo || q > sc->hi) ok = 0;
        }
        if (ok) { best = t; bs = sc->n_spheres + p; }
    }
    if (bs < 0) return -1;
    *t_out = best;
    if (bs < sc->n_spheres) {
        const double* sp = sc->spheres + 4 * bs;
        for (int a = 0; a < 3; ++a) nrm[a] = (o[a] + best * d[a] - sp[a]) / sp[3];
    } else {
        int p = bs - sc->n_spheres;
        nrm[0] = nrm[1] = nrm[2] = 0.0;
        nrm[plane_axis[p]] = plane_side[p] ? -1.0 : 1.0;
    }
    return bs;
}

/* Primary hits for rows [row0, row0+nrows) of the frame, scanline order. Returns number of misses
 * (a miss writes x = n = wo = 0 and surf = -1). x is clamped into [lo,hi]^3 on plane hits' own axis
 * only through rounding; no other post-processing. */
OO_GEN_API uint64_t oo_gen_raycast(const oo_scene* sc, const oo_camera* cam, uint32_t row0, uint32_t nrows,
                                   float* x, float* nrm, float* wo, int32_t* surf) {
    double f[3] = {cam->look[0] - cam->eye[0], cam->look[1] - cam->eye[1], cam->look[2] - cam->eye[2]};
    norm3(f);
    double r[3], u[3];
    cross3(f, cam->up, r); norm3(r);
    cross3(r, f, u);
    double th = tan(0.5 * cam->vfov_deg * 3.14159265358979323846 / 180.0);
    double aspect = (double)cam->width / (double)cam->height;
    uint64_t misses = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : misses)
    for (int64_t jj = 0; jj < (int64_t)nrows; ++jj) {
        uint32_t j = row0 + (uint32_t)jj;
        for (uint32_t i = 0; i < cam->width; ++i) {
            double px = (2.0 * ((double)i + 0.5) / cam->width - 1.0) * th * aspect;
            double py = (1.0 - 2.0 * ((double)j + 0.5) / cam->height) * th;
            double d[3] = {f[0] + px * r[0] + py * u[0], f[1] + px * r[1] + py * u[1], f[2] + px * r[2] + py * u[2]};
            norm3(d);
            double t, nn[3];
            int s = scene_hit(sc, cam->eye, d, &t, nn);
            size_t q = (size_t)jj * cam->width + i;
            if (s < 0) {
                ++misses;
                for (int a = 0; a < 3; ++a) x[3 * q + a] = nrm[3 * q + a] = wo[3 * q + a] = 0.0f;
                if (surf) surf[q] = -1;
                continue;
            }
            for (int a = 0; a < 3; ++a) {
                x[3 * q + a] = (float)(cam->eye[a] + t * d[a]);
                nrm[3 * q + a] = (float)nn[a];
                wo[3 * q + a] = (float)(-d[a]);
            }
            if (surf) surf[q] = s;
        }
    }
    return misses;
}

/* --------------------------------------------------------------------------- incoherent sampler */
/* Sample k: surface chosen with probability proportional to its area, point uniform on it; rejected
 * (and retried with the next attempt counter) if a plane point lies inside a sphere or a sphere
 * point lies outside the box or inside another sphere.  Normal analytic (sphere outward, plane
 * inward); wo uniform on the hemisphere about the normal.  Order as generated. */
OO_GEN_API void oo_gen_incoherent(const oo_scene* sc, uint64_t seed, uint64_t stream, uint64_t first, uint64_t n,
                                  float* x, float* nrm, float* wo) {
    int ns = sc->n_spheres, n_surf = ns + N_PLANES;
    double* cdf = malloc((size_t)n_surf * sizeof(double));
    double side = sc->hi - sc->lo, acc = 0.0;
    for (int s = 0; s < n_surf; ++s) {
        double a = s < ns ? 4.0 * 3.14159265358979323846 * sc->spheres[4 * s + 3] * sc->spheres[4 * s + 3] : side * side;
        acc += a; cdf[s] = acc;
    }
    enum { MAX_TRY = 64, PER_TRY = 8 };
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < (int64_t)n; ++i) {
        uint64_t k = first + (uint64_t)i;
        double p[3] = {0, 0, 0}, nn[3] = {0, 0, 1};
        for (int a = 0; a < MAX_TRY; ++a) {
            uint64_t base = (k * MAX_TRY + (uint64_t)a) * PER_TRY;
            double us = ctr_u01(seed, stream, base) * acc;
            int s = 0;
            while (s < n_surf - 1 && us >= cdf[s]) ++s;
            int ok = 1;
            if (s < ns) {
                const double* sp = sc->spheres + 4 * s;
                double z = 1.0 - 2.0 * ctr_u01(seed, stream, base + 1);
                double phi = 6.283185307179586476925286766559 * ctr_u01(seed, stream, base + 2);
                double rr = sqrt(fmax(0.0, 1.0 - z * z));
                nn[0] = rr * cos(phi); nn[1] = rr * sin(phi); nn[2] = z;
                for (int c = 0; c < 3; ++c) p[c] = sp[c] + sp[3] * nn[c];
                for (int c = 0; c < 3; ++c) if (p[c] < sc->lo || p[c] > sc->hi) ok = 0;
            } else {
                int pl = s - ns, ax = plane_axis[pl];
                double u1 = ctr_u01(seed, stream, base + 1), u2 = ctr_u01(seed, stream, base + 2);
                int c2 = 0;
                for (int c = 0; c < 3; ++c) {
                    if (c == ax) { p[c] = plane_side[pl] ? sc->hi : sc->lo; nn[c] = plane_side[pl] ? -1.0 : 1.0; }
                    else { p[c] = sc->lo + side * (c2++ == 0 ? u1 : u2); nn[c] = 0.0; }
                }
            }
            for (int t = 0; ok && t < ns; ++t) {
                if (t == s) continue;
                const double* sp = sc->spheres + 4 * t;
                double dx = p[0] - sp[0], dy = p[1] - sp[1], dz = p[2] - sp[2];
                if (dx * dx + dy * dy + dz * dz < sp[3] * sp[3]) ok = 0;
            }
            if (ok) break;
        }
        uint64_t wb = (k * MAX_TRY + MAX_TRY - 1) * PER_TRY + 4;
        double z = 1.0 - 2.0 * ctr_u01(seed, stream, wb);
        double phi = 6.283185307179586476925286766559 * ctr_u01(seed, stream, wb + 1);
        double rr = sqrt(fmax(0.0, 1.0 - z * z));
        double w[3] = {rr * cos(phi), rr * sin(phi), z};
        if (w[0] * nn[0] + w[1] * nn[1] + w[2] * nn[2] < 0.0) { w[0] = -w[0]; w[1] = -w[1]; w[2] = -w[2]; }
        for (int c = 0; c < 3; ++c) {
            x[3 * i + c] = (float)p[c]; nrm[3 * i + c] = (float)nn[c]; wo[3 * i + c] = (float)w[c];
        }
    }
    free(cdf);
}
