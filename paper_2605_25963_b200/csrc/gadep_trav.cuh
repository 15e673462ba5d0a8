// gadep_trav.cuh -- resumable per-lane BVH traversal for the wavefront kernels (PAPER.md:219 BVH over the facets;
// PAPER.md:191 nearest facet along the flight direction).
//
// A lane owns one ray at a time; its whole traversal state sits in registers (+ a local-memory stack), so that a
// lane can (a) take a new ray the moment its ray ends while its neighbours keep going (dynamic fetch), and (b) hold
// an unfinished ray across a physics burst of its warp.  One call of gd_trav_step advances every busy lane of the
// warp by at most one inner-node visit and -- when enough lanes wait at a leaf -- one ray-triangle test.
#pragma once
#include "gadep_bvh.cuh"

#define GD_TRAV_DONE ((int)0x80000000)     // node value: traversal finished (leaf codes are ~index > GD_TRAV_DONE)
#define GD_NO_FACET 0x7FFFFFFF
#define GD_TINF __int_as_float(0x7F800000)
#ifndef GD_FULL_SORT
#define GD_FULL_SORT 1
#endif

struct GdTrav {
    float ox, oy, oz;        // origin (ray-triangle test)
    float ix, iy, iz;        // safe reciprocal direction
    float bx, by, bz;        // origin * reciprocal direction (slab test as one FMA per plane)
    float err;               // absolute error bound of the FMA slab distances
    float sx, sy, sz;        // Woop shear / scale
    int kxyz;                // kx | ky << 2 | kz << 4 | octant << 8 (bit a of the octant: direction component a < 0)
    float tmin, t;           // window (tmin, t]; t shrinks to the nearest accepted hit
    int orig;                // caller's facet index of that hit, GD_NO_FACET = none
    int fromto;              // (from-side material & 0xFFFF) | (to-side material << 16) of that hit
    int filter, exa, exb, exc;
    int node, sp;
    int slot;                // owner's handle (photon slot / ray index), < 0 = lane idle
};

GD_D void gd_trav_idle(GdTrav &T) { T.slot = -1; T.node = GD_TRAV_DONE; T.sp = 0; }

GD_D void gd_trav_begin(GdTrav &T, const GdBvh &bvh, int *stack, float px, float py, float pz, float dx, float dy, float dz,
                        float t_min, float t_max, int filter, int exa, int exb, int exc, int slot) {
    T.ox = px; T.oy = py; T.oz = pz;
    T.ix = gd_safe_rcp(dx); T.iy = gd_safe_rcp(dy); T.iz = gd_safe_rcp(dz);
    T.bx = px * T.ix; T.by = py * T.iy; T.bz = pz * T.iz;
    // |fma(lo, inv, -b) - exact| <= ulp(b) (rounding of b) + rounding of the result (covered by the far-side pad)
    T.err = fmaxf(fmaxf(fabsf(T.bx), fabsf(T.by)), fabsf(T.bz)) * 1.1920929e-7f;
    float ax = fabsf(dx), ay = fabsf(dy), az = fabsf(dz);
    int kz = (ax > ay) ? (ax > az ? 0 : 2) : (ay > az ? 1 : 2);
    int kx = kz + 1; if (kx == 3) kx = 0;
    int ky = kx + 1; if (ky == 3) ky = 0;
    float ddz = kz == 0 ? dx : (kz == 1 ? dy : dz);
    if (ddz < 0.0f) { int t = kx; kx = ky; ky = t; }
    float ddx = kx == 0 ? dx : (kx == 1 ? dy : dz), ddy = ky == 0 ? dx : (ky == 1 ? dy : dz);
    T.sz = 1.0f / ddz; T.sx = ddx * T.sz; T.sy = ddy * T.sz;
    T.kxyz = kx | (ky << 2) | (kz << 4) |
             (int)((((unsigned)__float_as_int(T.ix) >> 31) | (((unsigned)__float_as_int(T.iy) >> 31) << 1) |
                    (((unsigned)__float_as_int(T.iz) >> 31) << 2)) << 8);
    T.tmin = t_min; T.t = t_max; T.orig = GD_NO_FACET; T.fromto = 0;
    T.filter = filter; T.exa = exa; T.exb = exb; T.exc = exc;
    T.sp = 0; T.node = bvh.root_is_leaf ? ~0 : 0;
    T.slot = slot;
    if (bvh.mat_entry && filter >= 0) {
        // only facets with `filter` on their from-side can be accepted: start at the subtrees of the surfaces that have
        // this material on one side
        const int *e = bvh.mat_entry + filter * (1 + GD_ENTRY_MAX);
        const int ne = __ldg(e);
        if (ne > 0) {
            T.node = __ldg(e + 1);
            for (int k = 2; k <= ne; ++k) stack[T.sp++] = __ldg(e + k);
        }
    }
}

struct GdEdge3 { float u, v, w; int ok; };
__device__ __noinline__ GdEdge3 gd_edges_double(float ax, float ay, float bx, float by, float cx, float cy) {
    const double du = GD_DSUB(GD_DMUL((double)cx, (double)by), GD_DMUL((double)cy, (double)bx));
    const double dv = GD_DSUB(GD_DMUL((double)ax, (double)cy), GD_DMUL((double)ay, (double)cx));
    const double dw = GD_DSUB(GD_DMUL((double)bx, (double)ay), GD_DMUL((double)by, (double)ax));
    GdEdge3 e;
    e.u = (float)du; e.v = (float)dv; e.w = (float)dw;
    e.ok = !((du < 0.0 || dv < 0.0 || dw < 0.0) && (du > 0.0 || dv > 0.0 || dw > 0.0));
    return e;
}

GD_D float gd_sel3(float x, float y, float z, int k) { return k == 0 ? x : (k == 1 ? y : z); }

// same arithmetic as gd_ray_tri / gd_test_leaf (gadep_bvh.cuh), on the register-resident ray
GD_D void gd_trav_leaf(GdTrav &T, const GdBvh &bvh, int leaf, unsigned &n_tri_tests) {
    const GdTri &tr = bvh.tris[leaf];
    float4 p0 = tr.v0, p1 = tr.v1, p2 = tr.v2;
    const int facet = __float_as_int(p0.w);
    if (facet == T.exa || facet == T.exb || facet == T.exc) return;
    n_tri_tests++;
    const int kx = T.kxyz & 3, ky = (T.kxyz >> 2) & 3, kz = (T.kxyz >> 4) & 3;
    float a0 = p0.x - T.ox, a1 = p0.y - T.oy, a2 = p0.z - T.oz;
    float b0 = p1.x - T.ox, b1 = p1.y - T.oy, b2 = p1.z - T.oz;
    float c0 = p2.x - T.ox, c1 = p2.y - T.oy, c2 = p2.z - T.oz;
    float akz = gd_sel3(a0, a1, a2, kz), bkz = gd_sel3(b0, b1, b2, kz), ckz = gd_sel3(c0, c1, c2, kz);
    float ax = GD_SUB(gd_sel3(a0, a1, a2, kx), GD_MUL(T.sx, akz)), ay = GD_SUB(gd_sel3(a0, a1, a2, ky), GD_MUL(T.sy, akz));
    float bx = GD_SUB(gd_sel3(b0, b1, b2, kx), GD_MUL(T.sx, bkz)), by = GD_SUB(gd_sel3(b0, b1, b2, ky), GD_MUL(T.sy, bkz));
    float cx = GD_SUB(gd_sel3(c0, c1, c2, kx), GD_MUL(T.sx, ckz)), cy = GD_SUB(gd_sel3(c0, c1, c2, ky), GD_MUL(T.sy, ckz));
    float u = GD_SUB(GD_MUL(cx, by), GD_MUL(cy, bx));
    float v = GD_SUB(GD_MUL(ax, cy), GD_MUL(ay, cx));
    float w = GD_SUB(GD_MUL(bx, ay), GD_MUL(by, ax));
    if (u == 0.0f || v == 0.0f || w == 0.0f) {          // on an edge in float: decide in double (out of line: rare)
        const GdEdge3 e = gd_edges_double(ax, ay, bx, by, cx, cy);
        u = e.u; v = e.v; w = e.w;
        if (!e.ok) return;
    } else if ((u < 0.0f || v < 0.0f || w < 0.0f) && (u > 0.0f || v > 0.0f || w > 0.0f)) {
        return;
    }
    float det = u + v + w;
    if (det == 0.0f) return;
    float az = T.sz * akz, bz = T.sz * bkz, cz = T.sz * ckz;
    float tt = u * az + v * bz + w * cz;
    float t = tt / det;
    if (!(t > T.tmin) || t > T.t) return;
    const int leaving = det < 0.0f;
    const int mats = __float_as_int(p1.w);
    const int m_in = gd_mat_inside(mats), m_out = gd_mat_outside(mats);
    const int from = leaving ? m_in : m_out, to = leaving ? m_out : m_in;
    if (T.filter != -2 && from != T.filter) return;
    if (t < T.t || facet < T.orig) {
        T.t = t; T.orig = facet; T.fromto = (from & 0xFFFF) | (int)((unsigned)(to & 0xFFFF) << 16);
    }
}

GD_D int gd_trav_pop(GdTrav &T, const int *stack) { return T.sp == 0 ? GD_TRAV_DONE : stack[--T.sp]; }

#define GD_CSWAP(ka, ca, kb, cb) do { if (kb < ka) { float tk = ka; ka = kb; kb = tk; int tc = ca; ca = cb; cb = tc; } } while (0)

// order the four (key, child) pairs, push the valid ones farthest first, continue with the nearest
GD_D void gd_trav_descend4(GdTrav &T, int *stack, float k0, float k1, float k2, float k3, int c0, int c1, int c2, int c3) {
#if GD_FULL_SORT
    GD_CSWAP(k0, c0, k1, c1); GD_CSWAP(k2, c2, k3, c3); GD_CSWAP(k0, c0, k2, c2); GD_CSWAP(k1, c1, k3, c3);
    GD_CSWAP(k1, c1, k2, c2);
#else
    // nearest child first; the others (usually none or one) in stored order, farther of a pair pushed first
    GD_CSWAP(k0, c0, k1, c1); GD_CSWAP(k2, c2, k3, c3); GD_CSWAP(k0, c0, k2, c2);
#endif
    if (c3 != GD_NO_CHILD) stack[T.sp++] = c3;
    if (c2 != GD_NO_CHILD) stack[T.sp++] = c2;
    if (c1 != GD_NO_CHILD) stack[T.sp++] = c1;
    T.node = c0 != GD_NO_CHILD ? c0 : gd_trav_pop(T, stack);
}

// one 4-wide node visit of a ray: FMA slab tests, far sides padded by the FMA error bound and ~3 ulp.
// The near / far plane of every slab is picked by address from the sign of the direction component (lo and hi are
// 16 bytes apart in GdNode4), which equals min / max of the two plane distances (fma is monotonic in its first
// operand) and saves 24 min/max per visit.
GD_D void gd_trav_node4(GdTrav &T, const GdBvh &bvh, int *stack, unsigned &n_box_tests) {
    const char *nd = (const char *)(bvh.nodes4 + T.node);
    const int sx = (__float_as_int(T.ix) >> 31) & 16, sy = (__float_as_int(T.iy) >> 31) & 16, sz = (__float_as_int(T.iz) >> 31) & 16;
    const float4 nx = *(const float4 *)(nd + sx), fx = *(const float4 *)(nd + (16 - sx));
    const float4 ny = *(const float4 *)(nd + 32 + sy), fy = *(const float4 *)(nd + 32 + (16 - sy));
    const float4 nz = *(const float4 *)(nd + 64 + sz), fz = *(const float4 *)(nd + 64 + (16 - sz));
    const int4 ch = *(const int4 *)(nd + 96);
    n_box_tests += 4;
    const float pad = 4.0e-7f, tlo = T.tmin + T.err, e2 = 2.0f * T.err;
    float key[4];
    int cc[4] = {ch.x, ch.y, ch.z, ch.w};
    const float ax[4] = {nx.x, nx.y, nx.z, nx.w}, bx[4] = {fx.x, fx.y, fx.z, fx.w};
    const float ay[4] = {ny.x, ny.y, ny.z, ny.w}, by[4] = {fy.x, fy.y, fy.z, fy.w};
    const float az[4] = {nz.x, nz.y, nz.z, nz.w}, bz[4] = {fz.x, fz.y, fz.z, fz.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float x0 = fmaf(ax[k], T.ix, -T.bx), x1 = fmaf(bx[k], T.ix, -T.bx);
        const float y0 = fmaf(ay[k], T.iy, -T.by), y1 = fmaf(by[k], T.iy, -T.by);
        const float z0 = fmaf(az[k], T.iz, -T.bz), z1 = fmaf(bz[k], T.iz, -T.bz);
        const float n = fmaxf(fmaxf(x0, y0), fmaxf(z0, tlo));
        float f = fminf(fminf(x1, y1), fminf(z1, T.t));
        f = fmaf(fabsf(f), pad, f) + e2;
        const bool h = n <= f && cc[k] != GD_NO_CHILD;
        key[k] = h ? n : GD_TINF;
        cc[k] = h ? cc[k] : GD_NO_CHILD;
    }
    gd_trav_descend4(T, stack, key[0], key[1], key[2], key[3], cc[0], cc[1], cc[2], cc[3]);
}


// rays that ran out of traversal stack (8-wide nodes: up to 7 pushes per visit); read and reported by the host
__device__ unsigned gd_stack_overflow;

// one 8-wide compressed node visit (GdNode8): six 16-byte loads for eight boxes.  A quantised plane q of an axis lies at
// o + q 2^e; its slab distance is ((o - p) + q 2^e) / d = A + q B with B = 2^e / d and A from the same FMA as the
// 4-wide test.  The byte goes straight into the mantissa of the float 32768 + q (one PRMT, no integer-to-float
// conversion), so the distance is fma(32768 + q, B, A - 32768 B); the two extra roundings are bounded by |B| / 256
// per axis, which widens that axis' slab.  Hit children are visited in octant order (slot ^ direction signs).
#define GD_SELB(c, a, b) ((c) ? (a) : (b))
GD_D void gd_trav_node8(GdTrav &T, const GdBvh &bvh, int *stack, unsigned &n_box_tests) {
    const uint4 *nd = reinterpret_cast<const uint4 *>(bvh.nodes8 + T.node);
    const uint4 hd = nd[0], qx = nd[1], qy = nd[2], qz = nd[3];
    const uint4 ca = nd[4], cb = nd[5];
    const unsigned valid = hd.w >> 24;
    n_box_tests += __popc(valid);
    const float Bx = __uint_as_float((hd.w & 0xFFu) << 23) * T.ix;
    const float By = __uint_as_float(((hd.w >> 8) & 0xFFu) << 23) * T.iy;
    const float Bz = __uint_as_float(((hd.w >> 16) & 0xFFu) << 23) * T.iz;
    const float Ax = fmaf(-32768.0f, Bx, fmaf(__uint_as_float(hd.x), T.ix, -T.bx));
    const float Ay = fmaf(-32768.0f, By, fmaf(__uint_as_float(hd.y), T.iy, -T.by));
    const float Az = fmaf(-32768.0f, Bz, fmaf(__uint_as_float(hd.z), T.iz, -T.bz));
    // error bound of a slab distance, per axis (an axis the ray is almost parallel to has a huge B: its bound must not
    // loosen the other two): |B| / 256 for the two extra roundings + the bound of the 4-wide test; near planes move
    // down by it, far planes up
    const float ex = fmaf(fabsf(Bx), 1.0f / 256.0f, T.err), ey = fmaf(fabsf(By), 1.0f / 256.0f, T.err), ez = fmaf(fabsf(Bz), 1.0f / 256.0f, T.err);
    const float Anx = Ax - ex, Afx = Ax + ex, Any = Ay - ey, Afy = Ay + ey, Anz = Az - ez, Afz = Az + ez;
    const bool ngx = __float_as_int(T.ix) < 0, ngy = __float_as_int(T.iy) < 0, ngz = __float_as_int(T.iz) < 0;
    // near / far plane words of slots 0-3 and 4-7: the near plane is lo for a positive direction component, else hi
    const unsigned nx0 = GD_SELB(ngx, qx.z, qx.x), nx1 = GD_SELB(ngx, qx.w, qx.y), fx0 = GD_SELB(ngx, qx.x, qx.z), fx1 = GD_SELB(ngx, qx.y, qx.w);
    const unsigned ny0 = GD_SELB(ngy, qy.z, qy.x), ny1 = GD_SELB(ngy, qy.w, qy.y), fy0 = GD_SELB(ngy, qy.x, qy.z), fy1 = GD_SELB(ngy, qy.y, qy.w);
    const unsigned nz0 = GD_SELB(ngz, qz.z, qz.x), nz1 = GD_SELB(ngz, qz.w, qz.y), fz0 = GD_SELB(ngz, qz.x, qz.z), fz1 = GD_SELB(ngz, qz.y, qz.w);
    const float pad = 4.0e-7f;
    unsigned hm = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const unsigned sel = 0x7604u | ((unsigned)(k & 3) << 4);       // byte k & 3 of the word -> bits 8..15 of 0x47000000
        const float x0 = fmaf(__uint_as_float(__byte_perm(k < 4 ? nx0 : nx1, 0x47000000u, sel)), Bx, Anx);
        const float x1 = fmaf(__uint_as_float(__byte_perm(k < 4 ? fx0 : fx1, 0x47000000u, sel)), Bx, Afx);
        const float y0 = fmaf(__uint_as_float(__byte_perm(k < 4 ? ny0 : ny1, 0x47000000u, sel)), By, Any);
        const float y1 = fmaf(__uint_as_float(__byte_perm(k < 4 ? fy0 : fy1, 0x47000000u, sel)), By, Afy);
        const float z0 = fmaf(__uint_as_float(__byte_perm(k < 4 ? nz0 : nz1, 0x47000000u, sel)), Bz, Anz);
        const float z1 = fmaf(__uint_as_float(__byte_perm(k < 4 ? fz0 : fz1, 0x47000000u, sel)), Bz, Afz);
        const float n = fmaxf(fmaxf(x0, y0), fmaxf(z0, T.tmin));
        float f = fminf(fminf(x1, y1), fminf(z1, T.t));
        f = fmaf(fabsf(f), pad, f);
        hm |= n <= f ? (1u << k) : 0u;
    }
    hm &= valid;
    // octant order: position p = slot ^ r is visited before p + 1; permute links and hit bits into position order
    const unsigned r = ((unsigned)T.kxyz >> 8) & 7u;
    int c0 = (int)ca.x, c1 = (int)ca.y, c2 = (int)ca.z, c3 = (int)ca.w, c4 = (int)cb.x, c5 = (int)cb.y, c6 = (int)cb.z, c7 = (int)cb.w;
    {
        const bool s1 = r & 1u, s2 = r & 2u, s4 = r & 4u;
        int t;
        t = GD_SELB(s1, c1, c0); c1 = GD_SELB(s1, c0, c1); c0 = t;  t = GD_SELB(s1, c3, c2); c3 = GD_SELB(s1, c2, c3); c2 = t;
        t = GD_SELB(s1, c5, c4); c5 = GD_SELB(s1, c4, c5); c4 = t;  t = GD_SELB(s1, c7, c6); c7 = GD_SELB(s1, c6, c7); c6 = t;
        hm = GD_SELB(s1, ((hm & 0xAAu) >> 1) | ((hm & 0x55u) << 1), hm);
        t = GD_SELB(s2, c2, c0); c2 = GD_SELB(s2, c0, c2); c0 = t;  t = GD_SELB(s2, c3, c1); c3 = GD_SELB(s2, c1, c3); c1 = t;
        t = GD_SELB(s2, c6, c4); c6 = GD_SELB(s2, c4, c6); c4 = t;  t = GD_SELB(s2, c7, c5); c7 = GD_SELB(s2, c5, c7); c5 = t;
        hm = GD_SELB(s2, ((hm & 0xCCu) >> 2) | ((hm & 0x33u) << 2), hm);
        t = GD_SELB(s4, c4, c0); c4 = GD_SELB(s4, c0, c4); c0 = t;  t = GD_SELB(s4, c5, c1); c5 = GD_SELB(s4, c1, c5); c1 = t;
        t = GD_SELB(s4, c6, c2); c6 = GD_SELB(s4, c2, c6); c2 = t;  t = GD_SELB(s4, c7, c3); c7 = GD_SELB(s4, c3, c7); c3 = t;
        hm = GD_SELB(s4, ((hm & 0xF0u) >> 4) | ((hm & 0x0Fu) << 4), hm);
    }
    if (hm == 0u) { T.node = gd_trav_pop(T, stack); return; }
    if (T.sp > GD_STACK8 - 8) {                 // cannot happen on the meshes of the five workloads; reported, never silent
        atomicAdd(&gd_stack_overflow, 1u);
        T.node = GD_TRAV_DONE; T.sp = 0; T.orig = GD_NO_FACET;
        return;
    }
    const unsigned rest = hm & (hm - 1u);       // all hits but the first in order: pushed far to near
    if (rest & 0x80u) stack[T.sp++] = c7;
    if (rest & 0x40u) stack[T.sp++] = c6;
    if (rest & 0x20u) stack[T.sp++] = c5;
    if (rest & 0x10u) stack[T.sp++] = c4;
    if (rest & 0x08u) stack[T.sp++] = c3;
    if (rest & 0x04u) stack[T.sp++] = c2;
    if (rest & 0x02u) stack[T.sp++] = c1;
    const unsigned low = hm & (0u - hm);
    T.node = (low & 0x0Fu) ? ((low & 0x03u) ? ((low & 1u) ? c0 : c1) : ((low & 4u) ? c2 : c3))
                           : ((low & 0x30u) ? ((low & 0x10u) ? c4 : c5) : ((low & 0x40u) ? c6 : c7));
}

// one 4-wide compressed node visit (GdNode4q): four 16-byte loads for four boxes; dequantisation and error bounds as in
// gd_trav_node8, distance-sorted descent as in gd_trav_node4
GD_D void gd_trav_node4q(GdTrav &T, const GdBvh &bvh, int *stack, unsigned &n_box_tests) {
    const uint4 *nd = reinterpret_cast<const uint4 *>(bvh.nodes4q + T.node);
    const uint4 hd = nd[0], qa = nd[1], qb = nd[2];
    const int4 ch = *reinterpret_cast<const int4 *>(nd + 3);
    n_box_tests += 4;
    const float Bx = __uint_as_float((hd.w & 0xFFu) << 23) * T.ix;
    const float By = __uint_as_float(((hd.w >> 8) & 0xFFu) << 23) * T.iy;
    const float Bz = __uint_as_float(((hd.w >> 16) & 0xFFu) << 23) * T.iz;
    const float Ax = fmaf(-32768.0f, Bx, fmaf(__uint_as_float(hd.x), T.ix, -T.bx));
    const float Ay = fmaf(-32768.0f, By, fmaf(__uint_as_float(hd.y), T.iy, -T.by));
    const float Az = fmaf(-32768.0f, Bz, fmaf(__uint_as_float(hd.z), T.iz, -T.bz));
    const float ex = fmaf(fabsf(Bx), 1.0f / 256.0f, T.err), ey = fmaf(fabsf(By), 1.0f / 256.0f, T.err), ez = fmaf(fabsf(Bz), 1.0f / 256.0f, T.err);
    const float Anx = Ax - ex, Afx = Ax + ex, Any = Ay - ey, Afy = Ay + ey, Anz = Az - ez, Afz = Az + ez;
    const bool ngx = __float_as_int(T.ix) < 0, ngy = __float_as_int(T.iy) < 0, ngz = __float_as_int(T.iz) < 0;
    const unsigned nx = GD_SELB(ngx, qa.y, qa.x), fx = GD_SELB(ngx, qa.x, qa.y);
    const unsigned ny = GD_SELB(ngy, qa.w, qa.z), fy = GD_SELB(ngy, qa.z, qa.w);
    const unsigned nz = GD_SELB(ngz, qb.y, qb.x), fz = GD_SELB(ngz, qb.x, qb.y);
    const float pad = 4.0e-7f;
    float key[4];
    int cc[4] = {ch.x, ch.y, ch.z, ch.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const unsigned sel = 0x7604u | ((unsigned)k << 4);       // byte k of the word -> bits 8..15 of 0x47000000
        const float x0 = fmaf(__uint_as_float(__byte_perm(nx, 0x47000000u, sel)), Bx, Anx);
        const float x1 = fmaf(__uint_as_float(__byte_perm(fx, 0x47000000u, sel)), Bx, Afx);
        const float y0 = fmaf(__uint_as_float(__byte_perm(ny, 0x47000000u, sel)), By, Any);
        const float y1 = fmaf(__uint_as_float(__byte_perm(fy, 0x47000000u, sel)), By, Afy);
        const float z0 = fmaf(__uint_as_float(__byte_perm(nz, 0x47000000u, sel)), Bz, Anz);
        const float z1 = fmaf(__uint_as_float(__byte_perm(fz, 0x47000000u, sel)), Bz, Afz);
        const float n = fmaxf(fmaxf(x0, y0), fmaxf(z0, T.tmin));
        float f = fminf(fminf(x1, y1), fminf(z1, T.t));
        f = fmaf(fabsf(f), pad, f);
        const bool h = n <= f && cc[k] != GD_NO_CHILD;
        key[k] = h ? n : GD_TINF;
        cc[k] = h ? cc[k] : GD_NO_CHILD;
    }
    gd_trav_descend4(T, stack, key[0], key[1], key[2], key[3], cc[0], cc[1], cc[2], cc[3]);
}

// Advance the warp: every busy lane makes up to `n_steps` inner-node visits (no warp vote in between: a lane that
// reaches a leaf or the end of its ray idles for the rest of the round), then the lanes waiting at a leaf run
// their triangle test together.  One vote-free round amortises the scheduling work of the caller (fetch, retire)
// over several node visits and gathers several lanes for the rarer, more expensive leaf step.
template <int WIDTH>
GD_D void gd_trav_step(GdTrav &T, const GdBvh &bvh, int *stack, int n_steps, unsigned &n_box_tests,
                       unsigned &n_tri_tests) {
#pragma unroll 1
    for (int k = 0; k < n_steps; ++k) {
        if (T.node >= 0) {
            if (WIDTH == 8) gd_trav_node8(T, bvh, stack, n_box_tests);
            else if (WIDTH == GD_WIDTH_4Q) gd_trav_node4q(T, bvh, stack, n_box_tests);
            else gd_trav_node4(T, bvh, stack, n_box_tests);
        }
    }
    if (T.node < 0 && T.node != GD_TRAV_DONE) {
        gd_trav_leaf(T, bvh, ~T.node, n_tri_tests);
        T.node = gd_trav_pop(T, stack);
    }
}
