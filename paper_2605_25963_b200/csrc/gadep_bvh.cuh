// gadep_bvh.cuh -- LBVH construction helpers and nearest-hit traversal ("BVH ... to store
// triangular-facet data"; PAPER.md:191 nearest intersection along the flight direction).
// Morton-code LBVH after Karras 2012 (restated), watertight ray-triangle test after Woop, Benthin & Wald 2013
// (restated), while-while traversal with the children's boxes stored in the parent (Aila & Laine 2009 layout).
#pragma once
#include "gadep_common.cuh"

// ---------------------------------------------------------------- Morton keys (21 bits per axis -> 63 bits)
GD_HD unsigned long long gd_expand21(unsigned long long v) {
    v &= 0x1FFFFFull;
    v = (v | (v << 32)) & 0x001F00000000FFFFull;
    v = (v | (v << 16)) & 0x001F0000FF0000FFull;
    v = (v | (v << 8)) & 0x100F00F00F00F00Full;
    v = (v | (v << 4)) & 0x10C30C30C30C30C3ull;
    v = (v | (v << 2)) & 0x1249249249249249ull;
    return v;
}
GD_HD unsigned long long gd_morton63(float x, float y, float z) {   // x,y,z in [0,1]
    const float s = 2097151.0f;
    unsigned long long ix = (unsigned long long)fminf(fmaxf(x * s, 0.0f), s);
    unsigned long long iy = (unsigned long long)fminf(fmaxf(y * s, 0.0f), s);
    unsigned long long iz = (unsigned long long)fminf(fmaxf(z * s, 0.0f), s);
    return (gd_expand21(ix) << 2) | (gd_expand21(iy) << 1) | gd_expand21(iz);
}

GD_HD int gd_clz64(unsigned long long x) {
#ifdef __CUDA_ARCH__
    return __clzll((long long)x);
#else
    return x ? __builtin_clzll(x) : 64;
#endif
}
// common-prefix length of sorted keys i and j, index as tie-break (Karras 2012, sec. 4); -1 out of range
GD_HD int gd_delta(const unsigned long long *keys, int n, int i, int j) {
    if (j < 0 || j >= n) return -1;
    unsigned long long a = keys[i], b = keys[j];
    if (a == b) return 64 + gd_clz64((unsigned long long)(unsigned)(i ^ j)) - 32;
    return gd_clz64(a ^ b);
}
// Internal node i of the radix tree over n sorted keys: covers [first,last], split after `split`.
GD_HD void gd_karras_node(const unsigned long long *keys, int n, int i, int &first, int &last, int &split) {
    int d = (gd_delta(keys, n, i, i + 1) - gd_delta(keys, n, i, i - 1)) >= 0 ? 1 : -1;
    int dmin = gd_delta(keys, n, i, i - d);
    int lmax = 2;
    while (gd_delta(keys, n, i, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t = lmax >> 1; t >= 1; t >>= 1)
        if (gd_delta(keys, n, i, i + (l + t) * d) > dmin) l += t;
    int j = i + l * d;
    int dnode = gd_delta(keys, n, i, j);
    int s = 0;
    int t = l;
    do {
        t = (t + 1) >> 1;
        if (gd_delta(keys, n, i, i + (s + t) * d) > dnode) s += t;
    } while (t > 1);
    split = i + s * d + (d < 0 ? -1 : 0);
    first = d > 0 ? i : j;
    last = d > 0 ? j : i;
}

// ---------------------------------------------------------------- rays
struct GdRay {
    GdVec3 o, d, inv;     // origin, direction, safe reciprocal direction
    int kx, ky, kz;       // Woop axis permutation: kz = dominant axis
    float sx, sy, sz;     // shear / scale constants
};

GD_HD float gd_safe_rcp(float v) {
    const float tiny = 1.0e-30f;
    if (fabsf(v) < tiny) v = (v < 0.0f || (v == 0.0f && signbit(v))) ? -tiny : tiny;
    return 1.0f / v;
}

GD_HD void gd_ray_setup(GdRay &r, GdVec3 o, GdVec3 d) {
    r.o = o; r.d = d;
    r.inv = gd_make(gd_safe_rcp(d.x), gd_safe_rcp(d.y), gd_safe_rcp(d.z));
    float ax = fabsf(d.x), ay = fabsf(d.y), az = fabsf(d.z);
    int kz = (ax > ay) ? (ax > az ? 0 : 2) : (ay > az ? 1 : 2);
    int kx = kz + 1; if (kx == 3) kx = 0;
    int ky = kx + 1; if (ky == 3) ky = 0;
    float dz = gd_get(d, kz);
    if (dz < 0.0f) { int t = kx; kx = ky; ky = t; }     // keep the winding
    float dx = gd_get(d, kx), dy = gd_get(d, ky);
    r.kx = kx; r.ky = ky; r.kz = kz;
    r.sz = 1.0f / dz;
    r.sx = dx * r.sz;
    r.sy = dy * r.sz;
}

#ifdef __CUDA_ARCH__
#define GD_MUL(a, b) __fmul_rn((a), (b))
#define GD_SUB(a, b) __fsub_rn((a), (b))
#define GD_DMUL(a, b) __dmul_rn((a), (b))
#define GD_DSUB(a, b) __dsub_rn((a), (b))
#else
#define GD_MUL(a, b) ((a) * (b))
#define GD_SUB(a, b) ((a) - (b))
#define GD_DMUL(a, b) ((a) * (b))
#define GD_DSUB(a, b) ((a) - (b))
#endif

// Watertight test: returns true and (t, det) when the ray's line meets the facet (edges inclusive).
// det > 0  <=>  d . ((v1-v0) x (v2-v0)) < 0  (front face: entering);  det < 0: leaving.
// No FMA contraction in the edge functions: shared edges must evaluate to exact negatives.
GD_HD bool gd_ray_tri(const GdRay &r, const float4 &p0, const float4 &p1, const float4 &p2, float &t, float &det) {
    GdVec3 a = gd_make(p0.x - r.o.x, p0.y - r.o.y, p0.z - r.o.z);
    GdVec3 b = gd_make(p1.x - r.o.x, p1.y - r.o.y, p1.z - r.o.z);
    GdVec3 c = gd_make(p2.x - r.o.x, p2.y - r.o.y, p2.z - r.o.z);
    float akz = gd_get(a, r.kz), bkz = gd_get(b, r.kz), ckz = gd_get(c, r.kz);
    float ax = GD_SUB(gd_get(a, r.kx), GD_MUL(r.sx, akz)), ay = GD_SUB(gd_get(a, r.ky), GD_MUL(r.sy, akz));
    float bx = GD_SUB(gd_get(b, r.kx), GD_MUL(r.sx, bkz)), by = GD_SUB(gd_get(b, r.ky), GD_MUL(r.sy, bkz));
    float cx = GD_SUB(gd_get(c, r.kx), GD_MUL(r.sx, ckz)), cy = GD_SUB(gd_get(c, r.ky), GD_MUL(r.sy, ckz));
    float u = GD_SUB(GD_MUL(cx, by), GD_MUL(cy, bx));
    float v = GD_SUB(GD_MUL(ax, cy), GD_MUL(ay, cx));
    float w = GD_SUB(GD_MUL(bx, ay), GD_MUL(by, ax));
    if (u == 0.0f || v == 0.0f || w == 0.0f) {          // on an edge in float: decide in double
        double du = GD_DSUB(GD_DMUL((double)cx, (double)by), GD_DMUL((double)cy, (double)bx));
        double dv = GD_DSUB(GD_DMUL((double)ax, (double)cy), GD_DMUL((double)ay, (double)cx));
        double dw = GD_DSUB(GD_DMUL((double)bx, (double)ay), GD_DMUL((double)by, (double)ax));
        u = (float)du; v = (float)dv; w = (float)dw;
        if ((du < 0.0 || dv < 0.0 || dw < 0.0) && (du > 0.0 || dv > 0.0 || dw > 0.0)) return false;
    } else if ((u < 0.0f || v < 0.0f || w < 0.0f) && (u > 0.0f || v > 0.0f || w > 0.0f)) {
        return false;
    }
    det = u + v + w;
    if (det == 0.0f) return false;
    float az = r.sz * akz, bz = r.sz * bkz, cz = r.sz * ckz;
    float tt = u * az + v * bz + w * cz;
    t = tt / det;
    return true;
}

struct GdHit {
    float t;
    int leaf;        // index into the leaf-ordered triangle array, -1 = none
    int orig;        // caller's triangle index
    int leaving;     // 1: d.n > 0
    int mats;        // packed side materials of the facet
};

GD_HD int gd_mat_inside(int packed) { return (int)(short)(packed & 0xFFFF); }
GD_HD int gd_mat_outside(int packed) { return (int)(short)((unsigned)packed >> 16); }
GD_HD int gd_as_int(float f) {
#ifdef __CUDA_ARCH__
    return __float_as_int(f);
#else
    union { float f; int i; } c; c.f = f; return c.i;
#endif
}
GD_HD float gd_as_float(int i) {
#ifdef __CUDA_ARCH__
    return __int_as_float(i);
#else
    union { float f; int i; } c; c.i = i; return c.f;
#endif
}

// Facets already crossed on the current straight flight segment and still inside the negative-t window: a line meets
// a planar facet at most once, so they can never be the next boundary (without this, two facets of a corner cut
// thinner than the window would be re-accepted behind the photon for ever).
struct GdExclude {
    int a, b, c;
};
GD_HD GdExclude gd_no_exclude() { GdExclude x = {-1, -1, -1}; return x; }

GD_HD void gd_test_leaf(const GdBvh &bvh, const GdRay &ray, int leaf, int filter_mat, float t_min, const GdExclude &ex,
                        GdHit &hit, unsigned &n_tri_tests) {
    const GdTri &tr = bvh.tris[leaf];
    float4 p0 = tr.v0, p1 = tr.v1, p2 = tr.v2;
    const int facet = gd_as_int(p0.w);                       // caller's facet index (a facet may own several leaves)
    if (facet == ex.a || facet == ex.b || facet == ex.c) return;
    float t, det;
    n_tri_tests++;
    if (!gd_ray_tri(ray, p0, p1, p2, t, det)) return;
    if (!(t > t_min) || t > hit.t) return;
    int leaving = det < 0.0f;
    int mats = gd_as_int(p1.w);
    if (filter_mat != -2) {
        int from = leaving ? gd_mat_inside(mats) : gd_mat_outside(mats);
        if (from != filter_mat) return;
    }
    int orig = facet;
    if (t < hit.t || hit.leaf < 0 || orig < hit.orig) {
        hit.t = t; hit.leaf = leaf; hit.orig = orig; hit.leaving = leaving; hit.mats = mats;
    }
}

#ifdef __CUDA_ARCH__
#define GD_WARP_ALL(p) __all_sync(0xFFFFFFFFu, (p))
#else
#define GD_WARP_ALL(p) (p)
#endif

// Nearest facet with t in (t_min, t_max].  On return hit.leaf < 0 if none.
// WARP-SYNCHRONOUS: all 32 lanes of a warp must call it together (lanes without a ray pass active = false).  The
// vote at the end of every outer iteration re-converges the warp once per leaf visit; without it the lanes of a
// warp drift apart inside the two nested loops and the kernel runs at ~3.6 of 32 lanes (profiles/r01_*).
// SYNC = false: plain per-lane loop (history-per-thread kernel, host emulation).
template <bool SYNC>
GD_HD void gd_nearest_hit(const GdBvh &bvh, const GdRay &ray, float t_min, float t_max, int filter_mat,
                          const GdExclude &ex, bool active, GdHit &hit, unsigned &n_box_tests, unsigned &n_tri_tests) {
    hit.t = t_max; hit.leaf = -1; hit.orig = 0x7FFFFFFF; hit.leaving = 0; hit.mats = 0;
    if (bvh.root_is_leaf) {
        if (active) gd_test_leaf(bvh, ray, 0, filter_mat, t_min, ex, hit, n_tri_tests);
        return;
    }
    int stack[GD_STACK];
    int sp = 0;
    int node = 0;
    bool done = !active;
    const float pad = 4.0e-7f;     // far side padded by ~3 ulp (robust slab test)
    for (;;) {
        while (!done && node >= 0) {
            const GdNode &nd = bvh.nodes[node];
            float4 a = nd.n0xy, b = nd.n1xy, z = nd.nz;
            int4 lk = nd.link;
            n_box_tests += 2;
            float x0 = (a.x - ray.o.x) * ray.inv.x, x1 = (a.y - ray.o.x) * ray.inv.x;
            float y0 = (a.z - ray.o.y) * ray.inv.y, y1 = (a.w - ray.o.y) * ray.inv.y;
            float z0 = (z.x - ray.o.z) * ray.inv.z, z1 = (z.y - ray.o.z) * ray.inv.z;
            float n0 = fmaxf(fmaxf(fminf(x0, x1), fminf(y0, y1)), fmaxf(fminf(z0, z1), t_min));
            float f0 = fminf(fminf(fmaxf(x0, x1), fmaxf(y0, y1)), fminf(fmaxf(z0, z1), hit.t));
            f0 = f0 + fabsf(f0) * pad;
            x0 = (b.x - ray.o.x) * ray.inv.x; x1 = (b.y - ray.o.x) * ray.inv.x;
            y0 = (b.z - ray.o.y) * ray.inv.y; y1 = (b.w - ray.o.y) * ray.inv.y;
            z0 = (z.z - ray.o.z) * ray.inv.z; z1 = (z.w - ray.o.z) * ray.inv.z;
            float n1 = fmaxf(fmaxf(fminf(x0, x1), fminf(y0, y1)), fmaxf(fminf(z0, z1), t_min));
            float f1 = fminf(fminf(fmaxf(x0, x1), fmaxf(y0, y1)), fminf(fmaxf(z0, z1), hit.t));
            f1 = f1 + fabsf(f1) * pad;
            bool h0 = n0 <= f0, h1 = n1 <= f1;
            if (h0 && h1) {
                int near_c = lk.x, far_c = lk.y;
                if (n1 < n0) { near_c = lk.y; far_c = lk.x; }
                stack[sp++] = far_c;
                node = near_c;
            } else if (h0) {
                node = lk.x;
            } else if (h1) {
                node = lk.y;
            } else if (sp == 0) {
                done = true;
            } else {
                node = stack[--sp];
            }
        }
        if (!done) {     // leaf
            gd_test_leaf(bvh, ray, ~node, filter_mat, t_min, ex, hit, n_tri_tests);
            if (sp == 0) done = true;
            else node = stack[--sp];
        }
        if (SYNC ? GD_WARP_ALL(done) : done) break;
    }
}

// ---------------------------------------------------------------- reference splitting for long thin facets
// A cap of a revolved surface is a fan of N_theta slivers (PAPER.md:82-90 angularly equidistant sampling); the AABB
// of a sliver covers up to a quarter of the cap, so a ray through the cap would have to test dozens of them.  The
// builder therefore cuts a long facet into k references along its longest axis; each reference keeps the facet
// index and gets the AABB of the facet clipped to its slab.  (Early split clipping, Ernst & Greiner 2007, restated.)
// k = how loose the facet's AABB is: half its surface area over the facet area (2 for a tight axis-aligned fit)
GD_HD int gd_split_count(const float p[3][3], const float lo[3], const float hi[3], int max_splits, int &axis) {
    float e[3] = {hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]};
    axis = e[0] > e[1] ? (e[0] > e[2] ? 0 : 2) : (e[1] > e[2] ? 1 : 2);
    float ux = p[1][0] - p[0][0], uy = p[1][1] - p[0][1], uz = p[1][2] - p[0][2];
    float vx = p[2][0] - p[0][0], vy = p[2][1] - p[0][1], vz = p[2][2] - p[0][2];
    float cx = uy * vz - uz * vy, cy = uz * vx - ux * vz, cz = ux * vy - uy * vx;
    float area = 0.5f * sqrtf(cx * cx + cy * cy + cz * cz);
    float half_sa = e[0] * e[1] + e[1] * e[2] + e[2] * e[0];
    if (!(area > 0.0f) || !(e[axis] > 0.0f)) return 1;
    int k = (int)ceilf(half_sa / area * 0.25f);
    if (k < 1) k = 1;
    if (k > max_splits) k = max_splits;
    return k;
}

// AABB of triangle (p0,p1,p2) clipped to the slab [a,b] on `axis`; conservative (padded by 1 ulp-ish of the slab)
GD_HD void gd_clip_tri_box(const float p[3][3], int axis, float a, float b, float lo[3], float hi[3]) {
    for (int k = 0; k < 3; ++k) { lo[k] = 3.0e38f; hi[k] = -3.0e38f; }
    for (int i = 0; i < 3; ++i) {
        const float *u = p[i], *v = p[(i + 1) % 3];
        float ua = u[axis], va = v[axis];
        if (ua >= a && ua <= b)
            for (int k = 0; k < 3; ++k) { lo[k] = fminf(lo[k], u[k]); hi[k] = fmaxf(hi[k], u[k]); }
        for (int s = 0; s < 2; ++s) {       // edge crossings with the two slab planes
            float pl = s == 0 ? a : b;
            if ((ua < pl && va > pl) || (ua > pl && va < pl)) {
                float f = (pl - ua) / (va - ua);
                for (int k = 0; k < 3; ++k) {
                    float x = k == axis ? pl : u[k] + f * (v[k] - u[k]);
                    float padk = 4.0e-7f * (fabsf(u[k]) + fabsf(v[k])) + 1.0e-30f;
                    lo[k] = fminf(lo[k], x - padk); hi[k] = fmaxf(hi[k], x + padk);
                }
            }
        }
    }
    lo[axis] = fmaxf(lo[axis], a); hi[axis] = fminf(hi[axis], b);
}
