// gadep_common.cuh -- shared device-side types of the CUDA path (sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

#define GD_HD __host__ __device__ __forceinline__
#define GD_D __device__ __forceinline__

#define GD_MEC2 0.51099895f
#define GD_TWO_MEC2 1.0219979f
#define GD_TBACK 1.0e-4f            // negative-t acceptance window [mm] (reading Q5)
#define GD_MAT_KILL (-1)
#define GD_MAX_LINES 64
#define GD_MAX_MAT 16
#define GD_STACK 96                 // LBVH depth bound: 63 Morton bits + index tie-break bits
#define GD_STACK4 196                // 4-wide traversal: up to 3 pushes per binary level descended (depth <= 64)

#define GD_F_ESCAPED 1u
#define GD_F_PEAK 2u
#define GD_F_LEAK 4u
#define GD_F_NONSCORING 8u
#define GD_F_RELOC 0x80u             // internal: a re-localisation query is pending (never leaves the kernel)

// ---------------------------------------------------------------- BVH layout
// Binary BVH, children's boxes stored in the parent (one 64-byte node = 4 x 16 B loads):
//   n0xy = (c0.lo.x, c0.hi.x, c0.lo.y, c0.hi.y)   n1xy = same for child 1
//   nz   = (c0.lo.z, c0.hi.z, c1.lo.z, c1.hi.z)   link = (child0, child1, -, -)
// child >= 0: inner node index; child < 0: leaf, ~child = index into the leaf-ordered triangle array.
struct __align__(16) GdNode {
    float4 n0xy, n1xy, nz;
    int4 link;
};

// Leaf-ordered triangle: 48 bytes.  v0.w = caller's triangle index (bits), v1.w = side materials
// (inside & 0xFFFF) | (outside << 16), v2.w = surface index (bits).
struct __align__(16) GdTri {
    float4 v0, v1, v2;
};

// 4-wide node of the wavefront kernels (128 bytes = 8 x 16 B loads): the grandchildren of a binary node, boxes in SoA
// (component k of lox .. hiz belongs to child k).  child: >= 0 inner node index (same numbering as the binary
// nodes), < 0 leaf (~index into the leaf-ordered triangles), GD_NO_CHILD = unused entry.
#define GD_NO_CHILD ((int)0x80000000)
struct __align__(16) GdNode4 {
    float4 lox, hix, loy, hiy, loz, hiz;
    int4 child;
    int4 pad;
};

// 8-wide compressed node of the default traversal (96 bytes = 6 x 16 B): up to eight descendants of a binary node
// (greedy expansion of the child with the largest surface area), their boxes quantised to 8 bits per plane on a
// per-node grid: plane coordinate = o + q * 2^e per axis (e biased by 127, i.e. the exponent field of a float).
// Quantisation is outward (lo: floor, hi: ceil, plus 1/64 of a step), so a dequantised box contains the child's box
// and the set of facets a ray can reach is unchanged.  Children sit in the slot whose 3-bit number says on which
// side of the node's centre they lie (x: bit 0, y: bit 1, z: bit 2; greedy assignment), so that slot ^ (signs of
// the ray direction) is a front-to-back order without sorting distances (octant order of Ylitie, Karras & Laine,
// "Efficient incoherent ray traversal on GPUs through compressed wide BVHs", HPG 2017 -- idea restated, layout own).
// child[k]: as in GdNode4; unused slots have an inverted box (qlo 255, qhi 0) and no bit in the valid mask.
struct __align__(32) GdNode8 {
    float ox, oy, oz;
    unsigned exyz_valid;         // ex | ey << 8 | ez << 16 | valid mask << 24
    unsigned qx[4];              // qlo of slots 0-3, qlo of slots 4-7, qhi of slots 0-3, qhi of slots 4-7 (one byte per slot)
    unsigned qy[4], qz[4];
    int child[8];
};
// 4-wide compressed node (64 bytes = 4 x 16 B, half of GdNode4): the same four children as the GdNode4 of the same index,
// their boxes quantised to 8 bits per plane on the node's own grid exactly as in GdNode8 (plane = o + q * 2^e per axis,
// outward rounding).  For hierarchies far larger than the L2, where a node visit is a fetch from HBM: half the bytes per
// visit, twice the nodes per cache.  Unused children: link GD_NO_CHILD and an inverted box (qlo 255, qhi 0).
struct __align__(16) GdNode4q {
    float ox, oy, oz;
    unsigned exyz;               // ex | ey << 8 | ez << 16
    unsigned qx_lo, qx_hi, qy_lo, qy_hi;   // one byte per child
    unsigned qz_lo, qz_hi, pad0, pad1;
    int child[4];
};
#define GD_WIDTH_4Q 5               // template value of the traversal over GdNode4q (4 = GdNode4, 8 = GdNode8)
#define GD_STACK8 224               // 8-wide traversal: up to 7 pushes per node visited; overflow is detected and reported

#define GD_CELL_PLANES 8           // plane slots per listed cell
// Facet-clearance grid (built by gadep_build_bvh beside the hierarchy): uniform cells of edge h over the box of all
// surfaces but the world boundary.  One 32-bit word per cell:
//   bit 31 clear: bits 0-7 = lower bound of the distance from any point of the cell to any facet, in units of h / 4
//                 (0 = unknown / a facet may be near).  A flight that ends before that distance cannot meet a facet, so
//                 its nearest-hit query is answered ("none") without touching the BVH -- the answer the traversal gives.
//   bit 31 set:   the cell lies near facets and has a plane list: bits 0-2 = the scalar bound as above, bits 3-6 = number
//                 of planes (15 = no facet within reach), bits 7-30 = list index.  Every facet that comes within `reach`
//                 of the cell lies in one of the listed planes, so for a point p of the cell
//                 min(reach, min_k |n_k . (p - centre) + d_k|) is a lower bound of the distance to any facet (a triangle
//                 is never nearer than its plane) -- it resolves the tiny steps of a scattering chain inside a thin layer
//                 or beside a wall, where the scalar is zero.  planes[index * GD_CELL_PLANES + k] = (n_k, d_k), cell
//                 centre as origin.
struct GdGrid {
    const unsigned *info;           // [nz][ny][nx], nullptr = no grid
    const float4 *planes;
    float lox, loy, loz, inv_h, quarter_h, h, reach;
    int nx, ny, nz;
};
#define GD_CELL_LIST 0x80000000u

struct GdBvh {
    GdGrid grid;
    const GdNode *nodes;
    const GdNode4 *nodes4;
    const GdNode8 *nodes8;
    const GdNode4q *nodes4q;
    const GdTri *tris;
    int n_tri;
    int root_is_leaf;   // n_tri == 1
    // Surface-clustered hierarchy (gadep_build_bvh): the references sort by surface first, so every closed surface is one
    // subtree.  A flight in a known material can only meet the surfaces that have it on one side: mat_entry (device,
    // [material][1 + GD_ENTRY_MAX]: count, links) names their subtrees; count 0 = start at the root.  nullptr = off.
    const int *mat_entry;
};
#define GD_ENTRY_MAX 8

struct GdCounters {    // device-side totals, 64-bit
    unsigned long long n_histories, n_queries, n_box_tests, n_tri_tests, n_crossings, n_pe, n_compton, n_coherent,
        n_pair, n_escaped, n_leak, n_cutoff, n_safety, n_skipped, n_parity, n_parity_mismatch;
};

struct GdLocalCounters {  // per-thread, 32-bit
    unsigned n_queries, n_box_tests, n_tri_tests, n_crossings, n_pe, n_compton, n_coherent, n_pair, n_escaped, n_leak,
        n_cutoff;
};

struct GdSource {
    int kind;
    float pos[3], dir[3];
    float cyl_r, cyl_z0, cyl_z1, ex_r, ex_z0, ex_z1;
    int n_lines;
    float line_mev[GD_MAX_LINES];
    float line_cum[GD_MAX_LINES];   // running sums of the intensities, float32 left to right
    int line_bin[GD_MAX_LINES];     // spectrum bin of the line energy (host, double)
    // replicated source (gadep_set_source_copies): history h is emitted from copy h mod n_copies, translated by copy_off,
    // and counted under line copy * n_lines + l; line_mev / line_bin hold n_copies * n_lines entries
    int n_copies;
    float copy_off[8][3];
};

struct GdMaterials {
    int n_mat, n_grid;
    float ln_e0, inv_dln, e_cut;
    const float *table;             // device [n_mat][4][n_grid]: ln(mu) for channels 0..2 (-1e30 = zero), mu for 3
    unsigned scoring_mask;          // bit m set = material m scores
    int world_material;
    float rho[16];                  // g/cm^3 per material (electron-range mode only, R16)
};

struct GdVec3 {
    float x, y, z;
};
GD_HD GdVec3 gd_make(float x, float y, float z) { GdVec3 v = {x, y, z}; return v; }
GD_HD float gd_get(const GdVec3 &v, int k) { return k == 0 ? v.x : (k == 1 ? v.y : v.z); }

// ---------------------------------------------------------------- Philox4x32-10 (Salmon et al., SC'11)
struct GdU4 { uint32_t x, y, z, w; };
#define GD_HD_NI __host__ __device__ __noinline__   // one copy in the instruction cache instead of one per call site
GD_HD_NI GdU4 gd_philox4x32_10v(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
#ifdef __CUDA_ARCH__
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
#else
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t h0 = (uint32_t)(p0 >> 32), l0 = (uint32_t)p0, h1 = (uint32_t)(p1 >> 32), l1 = (uint32_t)p1;
#endif
        uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    GdU4 o = {c0, c1, c2, c3};
    return o;
}
GD_HD void gd_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                            uint32_t out[4]) {
    GdU4 o = gd_philox4x32_10v(c0, c1, c2, c3, k0, k1);
    out[0] = o.x; out[1] = o.y; out[2] = o.z; out[3] = o.w;
}

// Counter-based stream: key = seed, counter = (history_lo, history_hi, draw/4, stream); draw k = word k%4.
struct GdRng {
    uint32_t k0, k1, h0, h1, stream, draw;
    uint32_t w[4];
    uint32_t block;   // block index held in w, 0xFFFFFFFF = none
};
GD_HD void gd_rng_init(GdRng &g, unsigned long long seed, unsigned long long history, uint32_t stream, uint32_t draw) {
    g.k0 = (uint32_t)seed; g.k1 = (uint32_t)(seed >> 32);
    g.h0 = (uint32_t)history; g.h1 = (uint32_t)(history >> 32);
    g.stream = stream; g.draw = draw; g.block = 0xFFFFFFFFu;
}
// u = ((w >> 9) + 0.5) * 2^-23 in (0,1): k + 0.5 with k < 2^23 is exact in float32
#ifndef GD_RNG_CACHE
#define GD_RNG_CACHE 0      // 1: keep the last Philox block in registers (4 draws per block, ~30 instructions per call site)
#endif
GD_HD_NI float gd_rng_uniform_v(uint32_t k0, uint32_t k1, uint32_t h0, uint32_t h1, uint32_t stream, uint32_t draw) {
    const GdU4 o = gd_philox4x32_10v(h0, h1, draw >> 2, stream, k0, k1);
    const uint32_t k = draw & 3u;
    const uint32_t w = k == 0 ? o.x : (k == 1 ? o.y : (k == 2 ? o.z : o.w));
    return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f);
}
// the next four uniforms of the stream (draws d .. d+3) from one or two Philox blocks, without advancing the counter:
// an interaction that knows it will use several draws in a row peeks them with one call and then advances by what
// it used -- the stream is a pure function of the draw index, so the values are those gd_rng_next would return
struct GdF4u { float a, b, c, d; };
GD_HD_NI GdF4u gd_rng_peek4_v(uint32_t k0, uint32_t k1, uint32_t h0, uint32_t h1, uint32_t stream, uint32_t draw) {
    const uint32_t b = draw >> 2, o = draw & 3u;
    const GdU4 A = gd_philox4x32_10v(h0, h1, b, stream, k0, k1);
    uint32_t w0 = A.x, w1 = A.y, w2 = A.z, w3 = A.w;
    if (o) {
        const GdU4 B = gd_philox4x32_10v(h0, h1, b + 1u, stream, k0, k1);
        if (o == 1) { w0 = A.y; w1 = A.z; w2 = A.w; w3 = B.x; }
        else if (o == 2) { w0 = A.z; w1 = A.w; w2 = B.x; w3 = B.y; }
        else { w0 = A.w; w1 = B.x; w2 = B.y; w3 = B.z; }
    }
    const float s = 1.0f / 8388608.0f;
    GdF4u u = {((float)(w0 >> 9) + 0.5f) * s, ((float)(w1 >> 9) + 0.5f) * s, ((float)(w2 >> 9) + 0.5f) * s,
               ((float)(w3 >> 9) + 0.5f) * s};
    return u;
}
GD_HD GdF4u gd_rng_peek4(const GdRng &g) { return gd_rng_peek4_v(g.k0, g.k1, g.h0, g.h1, g.stream, g.draw); }

GD_HD float gd_rng_next(GdRng &g) {
#if GD_RNG_CACHE
    uint32_t b = g.draw >> 2;
    if (b != g.block) {
        gd_philox4x32_10(g.h0, g.h1, b, g.stream, g.k0, g.k1, g.w);
        g.block = b;
    }
    uint32_t k = g.draw & 3u;
    uint32_t w = k == 0 ? g.w[0] : (k == 1 ? g.w[1] : (k == 2 ? g.w[2] : g.w[3]));
    g.draw++;
    return ((float)(w >> 9) + 0.5f) * (1.0f / 8388608.0f);
#else
    // one out-of-line copy of the generator for all call sites (the transport kernels are instruction-fetch bound)
    return gd_rng_uniform_v(g.k0, g.k1, g.h0, g.h1, g.stream, g.draw++);
#endif
}
