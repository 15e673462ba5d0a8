/*
 * gadep_oracle.c -- CPU ORACLE for the Gadep photon-transport hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision, one history at a time, brute-force ray-triangle tests over all
 * facets.  It shares no code with the CUDA path (paper_2605_25963_b200/csrc) and must only be used by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arxiv 2605.25963; SURVEY.md 8(c) = the
 * step list O1..O14 written from the paper + BASELINE.json; readings listed in DESIGN.md):
 *   - Triangle record with inside / outside material per facet            PAPER.md:111  (sec 2.2.3)
 *   - facet normal n = (v1-v0) x (v2-v0), its sign decides enter / leave  PAPER.md:103-107 (Eq. 5)
 *   - nearest facet along the flight direction + side material ids        PAPER.md:191  (sec 2.4.2, "original algorithm")
 *   - parity (Jordan) localisation, used here as a cross-check only
 *   - photoelectric, Compton, pair production (+ coherent per BASELINE.json configs[1])
 *   - scoring of deposited energy in the sensitive Ge volume -> FEPE
 *   - optional (orc_set_electron_mode): the electrons of PAPER.md:179's coupled photon-electron physics as straight
 *     segments of the Katz-Penfold range instead of a local deposit (reading R16)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors; ray-triangle vs a second
 * formulation and hand-computed rays; slab transmission exp(-mu x); on-axis solid angle of the N-gon
 * cylinder; Klein-Nishina / Thomson moments vs quadrature; energy accounting per history; parity rule ==
 * side-id rule; pair escape peaks; electron mode: range values, kept fraction below a plane face (closed form),
 * photon trajectories untouched.  FEPE values themselves: parity unpinned by the paper (it prints no
 * numeric FEPE, Fig. 11 is an image); they are pinned only through the closed forms above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MEC2 0.51099895
#define ORC_ECUT 0.010
#define ORC_TBACK 1e-9
#define ORC_MAT_KILL (-1)
#define ORC_TWO_PI 6.283185307179586476925286766559

#define ORC_F_ESCAPED 1u
#define ORC_F_PEAK 2u
#define ORC_F_LEAK 4u
#define ORC_F_NONSCORING 8u

typedef struct {
    /* materials (O1/O2) */
    int n_mat, n_grid;
    double ln_e0, dln_e, e_min, e_max;
    double *mu;              /* [n_mat][4][n_grid] 1/mm, exact double images of the caller's float32 table */
    unsigned char *is_scoring;
    /* mesh */
    int n_vert, n_tri, n_surf, world_material;
    double *v0, *e1, *e2;    /* per triangle: vertex 0 and the two edge vectors (doubles of the f32 input) */
    int *tri_surface, *surf_in, *surf_out;
    int *surf_first, *surf_count; /* triangles of a surface are not assumed contiguous: index lists */
    int *surf_tris;
    double *surf_box;        /* [n_surf][6] AABB, for the optional pre-reject of PAPER.md:191 */
    /* source (O4) */
    int src_kind;
    double src_pos[3], src_dir[3], cyl_r, cyl_z0, cyl_z1, ex_r, ex_z0, ex_z1;
    int n_lines;
    double *line_mev, *line_int, line_int_sum;
    /* NEXT-3: the source replicated at n_copies translations, one per detector of a
     * batched scene; history h is emitted from copy h mod n_copies and counted under line copy * n_lines + l */
    int n_copies;
    double copy_off[8][3];
    /* NEXT-4 ("coupled photon-electron"): straight CSDA electron segments, see deposit() */
    int electron_mode;
    double rho[16];          /* g/cm^3 per material */
} orc_scene;

typedef struct {
    uint64_t n_queries, n_crossings, n_pe, n_compton, n_coherent, n_pair, n_escaped, n_leak, n_cutoff,
        n_filter_reject;
} orc_counters;

/* ------------------------------------------------------------------ O3: Philox4x32-10 (Salmon et al. 2011) */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }

typedef struct { uint64_t seed, history; uint32_t stream, draw; } orc_rng;

/* draw k of a stream = word (k mod 4) of block k/4; u = ((w >> 9) + 0.5) * 2^-23 in (0,1).
 * 23 bits, not the 24 of SURVEY.md O3: (k + 0.5) with k < 2^23 has 24 significant bits and is exact in
 * float32 as well as in double, so the float32 CUDA path sees identical uniforms (reading R3). */
static double rng_next(orc_rng *g) {
    uint32_t ctr[4] = {(uint32_t)g->history, (uint32_t)(g->history >> 32), g->draw >> 2, g->stream};
    uint32_t key[2] = {(uint32_t)g->seed, (uint32_t)(g->seed >> 32)};
    uint32_t w[4];
    philox4x32_10(ctr, key, w);
    double u = ((double)(w[g->draw & 3u] >> 9) + 0.5) * (1.0 / 8388608.0);
    g->draw++;
    return u;
}

double orc_u01(uint64_t seed, uint64_t history, uint32_t stream, uint32_t draw) {
    orc_rng g = {seed, history, stream, draw};
    return rng_next(&g);
}

/* ------------------------------------------------------------------ scene set-up */
orc_scene *orc_create(void) { return (orc_scene *)calloc(1, sizeof(orc_scene)); }

static void free_mesh(orc_scene *s) {
    free(s->v0); free(s->e1); free(s->e2); free(s->tri_surface); free(s->surf_in); free(s->surf_out);
    free(s->surf_first); free(s->surf_count); free(s->surf_tris); free(s->surf_box);
    s->v0 = s->e1 = s->e2 = s->surf_box = NULL;
    s->tri_surface = s->surf_in = s->surf_out = s->surf_first = s->surf_count = s->surf_tris = NULL;
}

void orc_destroy(orc_scene *s) {
    if (!s) return;
    free_mesh(s);
    free(s->mu); free(s->is_scoring); free(s->line_mev); free(s->line_int);
    free(s);
}

int orc_set_materials(orc_scene *s, int n_mat, int n_grid, double e_min, double e_max, const float *mu,
                      const unsigned char *is_scoring) {
    if (!s || n_mat <= 0 || n_grid < 2 || !(e_min > 0) || !(e_max > e_min)) return -1;
    free(s->mu); free(s->is_scoring);
    s->n_mat = n_mat; s->n_grid = n_grid; s->e_min = e_min; s->e_max = e_max;
    s->ln_e0 = log(e_min);
    s->dln_e = (log(e_max) - log(e_min)) / (double)(n_grid - 1);
    size_t n = (size_t)n_mat * 4 * n_grid;
    s->mu = (double *)malloc(n * sizeof(double));
    for (size_t i = 0; i < n; ++i) s->mu[i] = (double)mu[i];
    s->is_scoring = (unsigned char *)malloc(n_mat);
    memcpy(s->is_scoring, is_scoring, n_mat);
    return 0;
}

int orc_load_mesh(orc_scene *s, const float *vertices, int n_vert, const int *triangles, const int *tri_surface,
                  int n_tri, const int *surf_inside, const int *surf_outside, int n_surf, int world_material) {
    if (!s || n_vert <= 0 || n_tri <= 0 || n_surf <= 0) return -1;
    free_mesh(s);
    s->n_vert = n_vert; s->n_tri = n_tri; s->n_surf = n_surf; s->world_material = world_material;
    s->v0 = (double *)malloc(sizeof(double) * 3 * n_tri);
    s->e1 = (double *)malloc(sizeof(double) * 3 * n_tri);
    s->e2 = (double *)malloc(sizeof(double) * 3 * n_tri);
    s->tri_surface = (int *)malloc(sizeof(int) * n_tri);
    s->surf_in = (int *)malloc(sizeof(int) * n_surf);
    s->surf_out = (int *)malloc(sizeof(int) * n_surf);
    s->surf_first = (int *)calloc(n_surf + 1, sizeof(int));
    s->surf_count = (int *)calloc(n_surf, sizeof(int));
    s->surf_tris = (int *)malloc(sizeof(int) * n_tri);
    s->surf_box = (double *)malloc(sizeof(double) * 6 * n_surf);
    memcpy(s->surf_in, surf_inside, sizeof(int) * n_surf);
    memcpy(s->surf_out, surf_outside, sizeof(int) * n_surf);
    for (int k = 0; k < n_surf; ++k) {
        for (int a = 0; a < 3; ++a) { s->surf_box[6 * k + a] = INFINITY; s->surf_box[6 * k + 3 + a] = -INFINITY; }
    }
    for (int i = 0; i < n_tri; ++i) {
        int sf = tri_surface[i];
        if (sf < 0 || sf >= n_surf) return -2;
        s->tri_surface[i] = sf;
        s->surf_count[sf]++;
        const float *p[3];
        for (int c = 0; c < 3; ++c) {
            int vi = triangles[3 * i + c];
            if (vi < 0 || vi >= n_vert) return -3;
            p[c] = vertices + 3 * (size_t)vi;
        }
        for (int a = 0; a < 3; ++a) {
            double a0 = (double)p[0][a], a1 = (double)p[1][a], a2 = (double)p[2][a];
            s->v0[3 * i + a] = a0;
            s->e1[3 * i + a] = a1 - a0;   /* exact in double: differences of float32 values */
            s->e2[3 * i + a] = a2 - a0;
            double lo = fmin(a0, fmin(a1, a2)), hi = fmax(a0, fmax(a1, a2));
            if (lo < s->surf_box[6 * sf + a]) s->surf_box[6 * sf + a] = lo;
            if (hi > s->surf_box[6 * sf + 3 + a]) s->surf_box[6 * sf + 3 + a] = hi;
        }
    }
    for (int k = 0; k < n_surf; ++k) s->surf_first[k + 1] = s->surf_first[k] + s->surf_count[k];
    int *fill = (int *)calloc(n_surf, sizeof(int));
    for (int i = 0; i < n_tri; ++i) {
        int sf = s->tri_surface[i];
        s->surf_tris[s->surf_first[sf] + fill[sf]++] = i;   /* ascending triangle index inside a surface */
    }
    free(fill);
    return 0;
}

int orc_set_source(orc_scene *s, int kind, const double *pos, const double *dir, double cyl_r, double cyl_z0,
                   double cyl_z1, double ex_r, double ex_z0, double ex_z1, int n_lines, const float *line_mev,
                   const float *line_intensity) {
    if (!s || n_lines <= 0 || kind < 0 || kind > 2) return -1;
    s->src_kind = kind;
    if (s->n_copies < 1) s->n_copies = 1;
    memcpy(s->src_pos, pos, sizeof(double) * 3);
    memcpy(s->src_dir, dir, sizeof(double) * 3);
    s->cyl_r = cyl_r; s->cyl_z0 = cyl_z0; s->cyl_z1 = cyl_z1;
    s->ex_r = ex_r; s->ex_z0 = ex_z0; s->ex_z1 = ex_z1;
    free(s->line_mev); free(s->line_int);
    s->n_lines = n_lines;
    s->line_mev = (double *)malloc(sizeof(double) * n_lines);
    s->line_int = (double *)malloc(sizeof(double) * n_lines);
    s->line_int_sum = 0;
    for (int i = 0; i < n_lines; ++i) {
        s->line_mev[i] = (double)line_mev[i];
        s->line_int[i] = (double)line_intensity[i];
        if (!(s->line_int[i] >= 0)) return -2;
        s->line_int_sum += s->line_int[i];
    }
    return 0;
}

/* ------------------------------------------------------------------ O2: table interpolation */
/* channels 0..2 log-log, channel 3 (pair) lin in f; identically-zero entries give 0 */
static double mu_channel(const orc_scene *s, int m, int ch, double e) {
    double x = (log(e) - s->ln_e0) / s->dln_e;
    int j = (int)floor(x);
    if (j < 0) j = 0;
    if (j > s->n_grid - 2) j = s->n_grid - 2;
    double f = (log(e) - (s->ln_e0 + j * s->dln_e)) / s->dln_e;
    const double *t = s->mu + ((size_t)m * 4 + ch) * s->n_grid;
    double a = t[j], b = t[j + 1];
    if (ch == 3) {
        /* pair production needs E > 2 m_e c^2 (PAPER.md:179 names the process; BASELINE.json configs[0]: "pair
         * production 0 below 1.022 MeV").  The grid cell 1.00949-1.03885 MeV straddles the threshold, so the linear
         * interpolation alone would leave mu_pair > 0 just below it (reading R17). */
        if (e <= 2.0 * ORC_MEC2) return 0.0;
        return (1.0 - f) * a + f * b;
    }
    if (a <= 0.0 || b <= 0.0) return 0.0;
    return exp((1.0 - f) * log(a) + f * log(b));
}

double orc_mu(const orc_scene *s, int m, int ch, double e) { return mu_channel(s, m, ch, e); }

/* ------------------------------------------------------------------ O6: ray-triangle, brute force */
/* Moeller-Trumbore, two-sided, edge-inclusive.  Returns 1 and *t (signed), *dn = sign carrier of d.n
 * (n = e1 x e2, Eq. 5 un-normalised) when the line through (o, d) meets the facet. */
static int ray_tri(const orc_scene *s, int i, const double o[3], const double d[3], double *t, double *dn) {
    const double *e1 = s->e1 + 3 * i, *e2 = s->e2 + 3 * i, *v0 = s->v0 + 3 * i;
    double p[3] = {d[1] * e2[2] - d[2] * e2[1], d[2] * e2[0] - d[0] * e2[2], d[0] * e2[1] - d[1] * e2[0]};
    double det = e1[0] * p[0] + e1[1] * p[1] + e1[2] * p[2];
    if (fabs(det) < 1e-300) return 0;
    double inv = 1.0 / det;
    double tv[3] = {o[0] - v0[0], o[1] - v0[1], o[2] - v0[2]};
    double u = (tv[0] * p[0] + tv[1] * p[1] + tv[2] * p[2]) * inv;
    if (u < 0.0 || u > 1.0) return 0;
    double q[3] = {tv[1] * e1[2] - tv[2] * e1[1], tv[2] * e1[0] - tv[0] * e1[2], tv[0] * e1[1] - tv[1] * e1[0]};
    double v = (d[0] * q[0] + d[1] * q[1] + d[2] * q[2]) * inv;
    if (v < 0.0 || u + v > 1.0) return 0;
    *t = (e2[0] * q[0] + e2[1] * q[1] + e2[2] * q[2]) * inv;
    /* d . (e1 x e2) = -det  (det = e1 . (d x e2)) */
    *dn = -det;
    return 1;
}

int orc_ray_triangle(const orc_scene *s, int tri, const double *o, const double *d, double *t, double *dn) {
    if (tri < 0 || tri >= s->n_tri) return 0;
    return ray_tri(s, tri, o, d, t, dn);
}

static int ray_box(const double *b, const double o[3], const double d[3], double t_lo) {
    double t0 = t_lo, t1 = INFINITY;
    for (int a = 0; a < 3; ++a) {
        double lo = b[a] - 1e-6, hi = b[3 + a] + 1e-6;
        if (d[a] == 0.0) {
            if (o[a] < lo || o[a] > hi) return 0;
        } else {
            double ta = (lo - o[a]) / d[a], tb = (hi - o[a]) / d[a];
            if (ta > tb) { double x = ta; ta = tb; tb = x; }
            if (ta > t0) t0 = ta;
            if (tb < t1) t1 = tb;
            if (t0 > t1) return 0;
        }
    }
    return 1;
}

/* nearest facet with t > t_min; if filter_mat != -2 only facets whose from-side material == filter_mat
 * (from-side = inside id if d.n > 0 else outside id, O7.3).  Ties -> lowest triangle index. */
static int nearest_hit(const orc_scene *s, const double o[3], const double d[3], int filter_mat, double t_min,
                       double *t_out, int *leaving_out, orc_counters *cnt) {
    int best = -1;
    double best_t = INFINITY, rej_t = INFINITY;
    int best_leaving = 0;
    for (int k = 0; k < s->n_surf; ++k) {
        if (!ray_box(s->surf_box + 6 * k, o, d, t_min)) continue;
        for (int q = s->surf_first[k]; q < s->surf_first[k + 1]; ++q) {
            int i = s->surf_tris[q];
            double t, dn;
            if (!ray_tri(s, i, o, d, &t, &dn)) continue;
            if (!(t > t_min)) continue;
            int leaving = dn > 0.0;
            if (filter_mat != -2) {
                int from = leaving ? s->surf_in[k] : s->surf_out[k];
                if (from != filter_mat) {
                    if (t > 1e-6 && t < rej_t) rej_t = t;   /* diagnostic: expected never nearest (O7.3) */
                    continue;
                }
            }
            if (t < best_t || (t == best_t && i < best)) { best_t = t; best = i; best_leaving = leaving; }
        }
    }
    if (cnt && rej_t < best_t) cnt->n_filter_reject++;
    if (best >= 0) { *t_out = best_t; *leaving_out = best_leaving; }
    return best;
}

int orc_nearest_hit(const orc_scene *s, const double *o, const double *d, int filter_mat, double t_min, double *t,
                    int *leaving) {
    double tt = INFINITY; int lv = 0;
    int r = nearest_hit(s, o, d, filter_mat, t_min, &tt, &lv, NULL);
    if (t) *t = tt;
    if (leaving) *leaving = lv;
    return r;
}

void orc_trace_rays(const orc_scene *s, const float *org, const float *dir, long long n, int filter_mat, double t_min,
                    int *tri_out, double *t_out) {
#pragma omp parallel for schedule(dynamic, 64)
    for (long long r = 0; r < n; ++r) {
        double o[3] = {org[3 * r], org[3 * r + 1], org[3 * r + 2]};
        double d[3] = {dir[3 * r], dir[3 * r + 1], dir[3 * r + 2]};
        double t = INFINITY; int lv;
        int h = nearest_hit(s, o, d, filter_mat, t_min, &t, &lv, NULL);
        tri_out[r] = h;
        t_out[r] = h >= 0 ? t : INFINITY;
    }
}

/* O5: material at a point from the nearest facet ahead (no filter): leaving -> inside id, entering -> outside id */
static int locate_sideid(const orc_scene *s, const double o[3], const double d[3], orc_counters *cnt) {
    double t; int leaving;
    if (cnt) cnt->n_queries++;
    int h = nearest_hit(s, o, d, -2, 0.0, &t, &leaving, NULL);
    if (h < 0) return s->world_material;
    int k = s->tri_surface[h];
    return leaving ? s->surf_in[k] : s->surf_out[k];
}

int orc_locate_sideid(const orc_scene *s, const double *o, const double *d) { return locate_sideid(s, o, d, NULL); }

/* Jordan parity rule: count intersections per closed geometry along the ray; among the
 * geometries with an odd count, the one whose first intersection is nearest contains the point. */
int orc_locate_parity(const orc_scene *s, const double *o, const double *d) {
    int best_surf = -1;
    double best_first = INFINITY;
    for (int k = 0; k < s->n_surf; ++k) {
        int count = 0;
        double first = INFINITY;
        for (int q = s->surf_first[k]; q < s->surf_first[k + 1]; ++q) {
            double t, dn;
            if (ray_tri(s, s->surf_tris[q], o, d, &t, &dn) && t > 0.0) {
                count++;
                if (t < first) first = t;
            }
        }
        if ((count & 1) && first < best_first) { best_first = first; best_surf = k; }
    }
    return best_surf < 0 ? s->world_material : s->surf_in[best_surf];
}

/* ------------------------------------------------------------------ sampling laws */
/* O4 / O12: isotropic direction from 2 draws */
static void sample_isotropic(orc_rng *g, double d[3]) {
    double u1 = rng_next(g), u2 = rng_next(g);
    double w = 1.0 - 2.0 * u1, phi = ORC_TWO_PI * u2;
    double st = sqrt(fmax(0.0, 1.0 - w * w));
    d[0] = st * cos(phi); d[1] = st * sin(phi); d[2] = w;
}

/* O13: rotate d by polar cosine c and azimuth phi */
static void rotate_dir(double d[3], double c, double phi) {
    double u = d[0], v = d[1], w = d[2];
    double s = sqrt(fmax(0.0, 1.0 - c * c));
    double cp = cos(phi), sp = sin(phi);
    double r[3];
    double q = 1.0 - w * w;
    if (q > 1e-12) {
        double rho = sqrt(q);
        r[0] = u * c + s * (u * w * cp - v * sp) / rho;
        r[1] = v * c + s * (v * w * cp + u * sp) / rho;
        r[2] = w * c - s * rho * cp;
    } else {
        double sg = w >= 0.0 ? 1.0 : -1.0;
        r[0] = s * cp; r[1] = s * sp; r[2] = c * sg;
    }
    double n = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
    d[0] = r[0] / n; d[1] = r[1] / n; d[2] = r[2] / n;
}

/* O10: Klein-Nishina composition-rejection (Butcher-Messel as restated in SURVEY.md 8(c)); returns eps = E'/E */
static double sample_compton(orc_rng *g, double e, double *cos_theta) {
    double k = e / ORC_MEC2;
    double eps0 = 1.0 / (1.0 + 2.0 * k);
    double a1 = log(1.0 / eps0);
    double a2 = 0.5 * (1.0 - eps0 * eps0);
    double eps, t;
    for (;;) {
        double u1 = rng_next(g), u2 = rng_next(g), u3 = rng_next(g);
        if (a1 / (a1 + a2) > u1) eps = exp(-a1 * u2);
        else eps = sqrt(eps0 * eps0 + (1.0 - eps0 * eps0) * u2);
        t = (1.0 - eps) / (k * eps);
        double sin2 = t * (2.0 - t);
        if (1.0 - eps * sin2 / (1.0 + eps * eps) >= u3) break;
    }
    *cos_theta = 1.0 - t;
    return eps;
}

/* O11: Thomson 1 + cos^2 law, exact CDF inversion */
static double sample_thomson(orc_rng *g) {
    double u = rng_next(g);
    double c = 8.0 * u - 4.0;
    double r = sqrt(0.25 * c * c + 1.0);
    return cbrt(0.5 * c + r) + cbrt(0.5 * c - r);
}

void orc_test_compton(double e, uint64_t seed, long long n, double *eps_out, double *cos_out) {
    for (long long i = 0; i < n; ++i) {
        orc_rng g = {seed, (uint64_t)i, 0, 0};
        eps_out[i] = sample_compton(&g, e, &cos_out[i]);
    }
}
void orc_test_thomson(uint64_t seed, long long n, double *cos_out) {
    for (long long i = 0; i < n; ++i) { orc_rng g = {seed, (uint64_t)i, 0, 0}; cos_out[i] = sample_thomson(&g); }
}
void orc_test_isotropic(uint64_t seed, long long n, double *d_out) {
    for (long long i = 0; i < n; ++i) { orc_rng g = {seed, (uint64_t)i, 0, 0}; sample_isotropic(&g, d_out + 3 * i); }
}
void orc_test_rotate(const double *d_in, double c, double phi, double *d_out) {
    d_out[0] = d_in[0]; d_out[1] = d_in[1]; d_out[2] = d_in[2];
    rotate_dir(d_out, c, phi);
}

/* ------------------------------------------------------------------ one history (O4 .. O14) */
typedef struct {
    double dep_scoring, dep_other, e_escaped;
    uint32_t flags, n_events, n_electrons;
} orc_hist;

typedef struct { double pos[3], dir[3], e; int m; uint32_t stream; } orc_photon;

/* Electron range, Katz & Penfold (1952): R [mg/cm^2] = 412 T^n, n = 1.265 - 0.0954 ln T, T in MeV; in mm for the
 * material's density.  DESIGN.md reading R16. */
double orc_electron_range_mm(double t_mev, double rho_g_cm3) {
    if (!(t_mev > 0.0) || !(rho_g_cm3 > 0.0)) return 0.0;
    double n = 1.265 - 0.0954 * log(t_mev);
    return 412.0 * pow(t_mev, n) / (100.0 * rho_g_cm3);
}

/* Energy `t_kin` set free as one electron at `pos` in material m.  Local deposit (O9/O10/O12) unless the electron mode
 * is on: then the energy is laid down uniformly along a straight segment of the CSDA range in a direction drawn
 * isotropically from stream 3 of the history (draws 2k, 2k+1 for the k-th electron); the segment is cut at the first
 * facet that has m on its from-side, what is left goes to the material behind that facet, on the spot (lost if KILL). */
static void deposit(const orc_scene *s, orc_hist *h, const double pos[3], int m, double t_kin, uint64_t seed,
                    uint64_t history, uint32_t *n_electrons, orc_counters *cnt) {
    double in_m = t_kin, beyond = 0.0;
    int m2 = m;
    if (s->electron_mode) {
        double range = orc_electron_range_mm(t_kin, s->rho[m]);
        orc_rng g = {seed, history, 3, 2u * (*n_electrons)};
        (*n_electrons)++;
        double u[3];
        sample_isotropic(&g, u);
        if (range > 0.0) {
            double t = INFINITY; int leaving = 0;
            cnt->n_queries++;
            int hit = nearest_hit(s, pos, u, m, 0.0, &t, &leaving, cnt);
            if (hit >= 0 && t < range) {
                in_m = t_kin * (t / range); beyond = t_kin - in_m;
                int k = s->tri_surface[hit];
                m2 = leaving ? s->surf_out[k] : s->surf_in[k];
            }
        }
    }
    if (s->is_scoring[m]) h->dep_scoring += in_m; else { h->dep_other += in_m; h->flags |= ORC_F_NONSCORING; }
    if (beyond > 0.0) {
        if (m2 != ORC_MAT_KILL && s->is_scoring[m2]) h->dep_scoring += beyond;
        else { h->dep_other += beyond; h->flags |= ORC_F_NONSCORING; }
    }
}

/* O7-O12 for one photon; secondaries (pair) are appended to `stack` */
static void transport_photon(const orc_scene *s, orc_photon ph, uint64_t seed, uint64_t history, uint32_t draw0,
                             orc_hist *h, orc_photon *stack, int *n_stack, orc_counters *cnt) {
    orc_rng g = {seed, history, ph.stream, draw0};
    double tau = -log(rng_next(&g));                                   /* O7.1 */
    for (;;) {
        double mu[4], mu_tot = 0.0;
        for (int c = 0; c < 4; ++c) { mu[c] = mu_channel(s, ph.m, c, ph.e); mu_tot += mu[c]; }   /* O2 */
        double sdist = mu_tot > 0.0 ? tau / mu_tot : INFINITY;         /* O7.2 */
        double t = INFINITY; int leaving = 0;
        cnt->n_queries++;
        int hit = nearest_hit(s, ph.pos, ph.dir, ph.m, -ORC_TBACK, &t, &leaving, cnt);   /* O7.3 */
        if (hit >= 0 && t < 0.0) t = 0.0;
        if (hit < 0 && !(sdist < INFINITY)) {                          /* O7.5 */
            h->flags |= ORC_F_ESCAPED; h->e_escaped += ph.e; cnt->n_escaped++;
            if (ph.m != s->world_material) { h->flags |= ORC_F_LEAK; cnt->n_leak++; }
            return;
        }
        if (hit >= 0 && !(sdist < t)) {                                /* O7.6 boundary first */
            for (int a = 0; a < 3; ++a) ph.pos[a] += t * ph.dir[a];
            tau -= mu_tot * t;
            int k = s->tri_surface[hit];
            ph.m = leaving ? s->surf_out[k] : s->surf_in[k];
            cnt->n_crossings++;
            if (ph.m == ORC_MAT_KILL) { h->flags |= ORC_F_ESCAPED; h->e_escaped += ph.e; cnt->n_escaped++; return; }
            continue;
        }
        /* O7.4 interaction at pos + s d */
        for (int a = 0; a < 3; ++a) ph.pos[a] += sdist * ph.dir[a];
        h->n_events++;
        if (ph.e < ORC_ECUT) {                                          /* O8 cut-off */
            deposit(s, h, ph.pos, ph.m, ph.e, seed, history, &h->n_electrons, cnt);
            cnt->n_cutoff++;
            return;
        }
        double u = rng_next(&g) * mu_tot;                               /* O8 channel selection */
        int ch = -1; double acc = 0.0;
        for (int c = 0; c < 4; ++c) { acc += mu[c]; if (u < acc) { ch = c; break; } }
        if (ch < 0) { for (int c = 3; c >= 0; --c) if (mu[c] > 0.0) { ch = c; break; } }
        if (ch == 0) {                                                  /* O9 photoelectric */
            deposit(s, h, ph.pos, ph.m, ph.e, seed, history, &h->n_electrons, cnt);
            cnt->n_pe++;
            return;
        } else if (ch == 1) {                                           /* O10 Compton */
            double cost;
            double eps = sample_compton(&g, ph.e, &cost);
            double phi = ORC_TWO_PI * rng_next(&g);
            double e_new = eps * ph.e, dep = ph.e - e_new;
            deposit(s, h, ph.pos, ph.m, dep, seed, history, &h->n_electrons, cnt);
            rotate_dir(ph.dir, cost, phi);
            ph.e = e_new;
            cnt->n_compton++;
            if (ph.e < ORC_ECUT) {
                deposit(s, h, ph.pos, ph.m, ph.e, seed, history, &h->n_electrons, cnt);
                cnt->n_cutoff++;
                return;
            }
        } else if (ch == 2) {                                           /* O11 coherent */
            double cost = sample_thomson(&g);
            double phi = ORC_TWO_PI * rng_next(&g);
            rotate_dir(ph.dir, cost, phi);
            cnt->n_coherent++;
        } else {                                                        /* O12 pair */
            double dep = ph.e - 2.0 * ORC_MEC2;
            deposit(s, h, ph.pos, ph.m, dep, seed, history, &h->n_electrons, cnt);
            double ax[3];
            sample_isotropic(&g, ax);
            cnt->n_pair++;
            orc_photon b = ph; b.e = ORC_MEC2; b.stream = 2;
            b.dir[0] = -ax[0]; b.dir[1] = -ax[1]; b.dir[2] = -ax[2];
            orc_photon a = ph; a.e = ORC_MEC2; a.stream = 1;
            a.dir[0] = ax[0]; a.dir[1] = ax[1]; a.dir[2] = ax[2];
            stack[(*n_stack)++] = b;   /* popped last */
            stack[(*n_stack)++] = a;   /* popped first: deposit order primary, A, B */
            return;
        }
        tau = -log(rng_next(&g));                                       /* O7.1 after every interaction */
    }
}

/* Batched scenes: n_copies translations of the source (NULL / 1 = the plain source).  n_copies * n_lines <= 64. */
int orc_set_source_copies(orc_scene *s, int n_copies, const double *offsets) {
    if (!s || n_copies < 1 || n_copies > 8 || (n_copies > 1 && !offsets)) return -1;
    s->n_copies = n_copies;
    memset(s->copy_off, 0, sizeof(s->copy_off));
    for (int c = 0; c < n_copies && offsets; ++c)
        for (int a = 0; a < 3; ++a) s->copy_off[c][a] = offsets[3 * c + a];
    return 0;
}

/* O4: line by cumulative intensity (draw 0, always consumed), emission point, direction.  Returns the line
 * (copy * n_lines + l for a replicated source). */
static int sample_source(const orc_scene *s, orc_rng *g, orc_photon *ph) {
    double ul = rng_next(g) * s->line_int_sum;
    int line = s->n_lines - 1; double acc = 0.0;
    for (int l = 0; l < s->n_lines; ++l) { acc += s->line_int[l]; if (ul < acc) { line = l; break; } }
    ph->e = s->line_mev[line]; ph->stream = 0;
    if (s->src_kind == 1) {
        for (;;) {
            double u1 = rng_next(g), u2 = rng_next(g), u3 = rng_next(g);
            double r = s->cyl_r * sqrt(u1), phi = ORC_TWO_PI * u2;
            double z = s->cyl_z0 + (s->cyl_z1 - s->cyl_z0) * u3;
            if (s->ex_r > 0.0 && r < s->ex_r && z >= s->ex_z0 && z <= s->ex_z1) continue;
            ph->pos[0] = r * cos(phi); ph->pos[1] = r * sin(phi); ph->pos[2] = z;
            break;
        }
    } else {
        memcpy(ph->pos, s->src_pos, sizeof(ph->pos));
    }
    if (s->src_kind == 2) memcpy(ph->dir, s->src_dir, sizeof(ph->dir));
    else sample_isotropic(g, ph->dir);
    if (s->n_copies > 1) {
        const int copy = (int)(g->history % (uint64_t)s->n_copies);
        for (int a = 0; a < 3; ++a) ph->pos[a] += s->copy_off[copy][a];
        line += copy * s->n_lines;
    }
    return line;
}

/* test hook (pins of O4): line, emission point, direction and the index of the first draw after the source
 * sampling (= draw of the first optical depth) for histories first .. first+n-1.  Any output may be NULL. */
void orc_test_source(const orc_scene *s, uint64_t seed, uint64_t first, long long n, int *line_out, double *pos_out,
                     double *dir_out, uint32_t *draw_out) {
    for (long long i = 0; i < n; ++i) {
        orc_rng g = {seed, first + (uint64_t)i, 0, 0};
        orc_photon ph;
        int line = sample_source(s, &g, &ph);
        if (line_out) line_out[i] = line;
        if (pos_out) memcpy(pos_out + 3 * i, ph.pos, sizeof(ph.pos));
        if (dir_out) memcpy(dir_out + 3 * i, ph.dir, sizeof(ph.dir));
        if (draw_out) draw_out[i] = g.draw;
    }
}

static int run_history(const orc_scene *s, uint64_t seed, uint64_t history, orc_hist *h, orc_counters *cnt) {
    memset(h, 0, sizeof(*h));
    orc_rng g = {seed, history, 0, 0};
    orc_photon ph;
    int line = sample_source(s, &g, &ph);                               /* O4 */
    ph.m = locate_sideid(s, ph.pos, ph.dir, cnt);                       /* O5 */
    orc_photon stack[4]; int n_stack = 0;
    transport_photon(s, ph, seed, history, g.draw, h, stack, &n_stack, cnt);
    while (n_stack > 0) {
        orc_photon q = stack[--n_stack];
        transport_photon(s, q, seed, history, 0, h, stack, &n_stack, cnt);
    }
    /* O14 */
    if (!(h->flags & (ORC_F_ESCAPED | ORC_F_NONSCORING))) h->flags |= ORC_F_PEAK;
    h->flags |= ((uint32_t)line & 0xFFu) << 8;
    h->flags |= (h->n_events > 0xFFFFu ? 0xFFFFu : h->n_events) << 16;
    return line;
}

static void add_counters(orc_counters *a, const orc_counters *b) {
    uint64_t *x = (uint64_t *)a; const uint64_t *y = (const uint64_t *)b;
    for (size_t i = 0; i < sizeof(orc_counters) / sizeof(uint64_t); ++i) x[i] += y[i];
}

/* NEXT-4: switch the straight-segment electron model on (densities in g/cm^3 per material) or off (rho == NULL) */
int orc_set_electron_mode(orc_scene *s, const double *rho, int n_mat) {
    if (!s || n_mat > 16) return -1;
    s->electron_mode = rho != NULL;
    for (int m = 0; m < n_mat && rho; ++m) s->rho[m] = rho[m];
    return 0;
}

/* test hook: fraction of t_kin that stays in material m for electrons number 0 of histories first .. first+n-1 */
void orc_test_electron_split(const orc_scene *s, const double *pos, int m, double t_kin, uint64_t seed, uint64_t first,
                             long long n, double *frac_in_m) {
    orc_counters cnt; memset(&cnt, 0, sizeof(cnt));
    for (long long i = 0; i < n; ++i) {
        orc_hist h; memset(&h, 0, sizeof(h));
        deposit(s, &h, pos, m, t_kin, seed, first + (uint64_t)i, &h.n_electrons, &cnt);
        /* in_m is whichever of the two tallies material m feeds; the rest went beyond the facet */
        frac_in_m[i] = (s->is_scoring[m] ? h.dep_scoring : h.dep_other) / t_kin;
    }
}

/* per-history dump (parity T4).  Any output pointer may be NULL. */
int orc_run_histories(const orc_scene *s, uint64_t first, long long n, uint64_t seed, double *edep_out,
                      uint32_t *flags_out, double *dep_other_out, double *escaped_out, orc_counters *cnt_out) {
    if (!s || !s->mu || !s->v0 || !s->line_mev) return -1;
    orc_counters total; memset(&total, 0, sizeof(total));
#pragma omp parallel
    {
        orc_counters local; memset(&local, 0, sizeof(local));
#pragma omp for schedule(dynamic, 256)
        for (long long i = 0; i < n; ++i) {
            orc_hist h;
            int line = run_history(s, seed, first + (uint64_t)i, &h, &local);
            double e = (h.flags & ORC_F_PEAK) ? s->line_mev[line % s->n_lines] : h.dep_scoring;
            if (edep_out) edep_out[i] = e;
            if (flags_out) flags_out[i] = h.flags;
            if (dep_other_out) dep_other_out[i] = h.dep_other;
            if (escaped_out) escaped_out[i] = h.e_escaped;
        }
#pragma omp critical
        add_counters(&total, &local);
    }
    if (cnt_out) *cnt_out = total;
    return 0;
}

/* O14: spectrum[n_bins+1] (last = overflow), emitted[n_lines], peak[n_lines] */
int orc_run(const orc_scene *s, uint64_t first, long long n, uint64_t seed, int n_bins, double e_max_mev,
            uint64_t *spectrum, uint64_t *emitted, uint64_t *peak, orc_counters *cnt_out) {
    if (!s || !s->mu || !s->v0 || !s->line_mev || n_bins <= 0) return -1;
    memset(spectrum, 0, sizeof(uint64_t) * (n_bins + 1));
    const int n_ctr = s->n_lines * (s->n_copies > 1 ? s->n_copies : 1);
    memset(emitted, 0, sizeof(uint64_t) * n_ctr);
    memset(peak, 0, sizeof(uint64_t) * n_ctr);
    double de = e_max_mev / (double)n_bins;
    orc_counters total; memset(&total, 0, sizeof(total));
#pragma omp parallel
    {
        uint64_t *sp = (uint64_t *)calloc(n_bins + 1, sizeof(uint64_t));
        uint64_t *em = (uint64_t *)calloc(n_ctr, sizeof(uint64_t));
        uint64_t *pk = (uint64_t *)calloc(n_ctr, sizeof(uint64_t));
        orc_counters local; memset(&local, 0, sizeof(local));
#pragma omp for schedule(dynamic, 256)
        for (long long i = 0; i < n; ++i) {
            orc_hist h;
            int line = run_history(s, seed, first + (uint64_t)i, &h, &local);
            em[line]++;
            double e = h.dep_scoring;
            if (h.flags & ORC_F_PEAK) { pk[line]++; e = s->line_mev[line % s->n_lines]; }
            if (e > 0.0) {
                double b = floor(e / de);
                int bin = b >= (double)n_bins ? n_bins : (int)b;
                sp[bin]++;
            }
        }
#pragma omp critical
        {
            for (int b = 0; b <= n_bins; ++b) spectrum[b] += sp[b];
            for (int l = 0; l < n_ctr; ++l) { emitted[l] += em[l]; peak[l] += pk[l]; }
            add_counters(&total, &local);
        }
        free(sp); free(em); free(pk);
    }
    if (cnt_out) *cnt_out = total;
    return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
