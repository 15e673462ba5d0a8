// gadep_build_kernels.cuh -- GPU construction of the BVH over the facets:
// facet boxes + scene bounds -> 63-bit Morton keys -> LSD radix sort (own kernels) -> Karras radix tree ->
// bottom-up refit that emits the 64-byte traversal nodes -> leaf-ordered triangle records.
#pragma once
#include "gadep_bvh.cuh"

#define GD_SORT_THREADS 256
#define GD_SORT_ITEMS 8
#define GD_SORT_TILE (GD_SORT_THREADS * GD_SORT_ITEMS)

GD_D int gd_f2o(float f) { int b = __float_as_int(f); return b >= 0 ? b : b ^ 0x7FFFFFFF; }
GD_D float gd_o2f(int o) { return __int_as_float(o >= 0 ? o : o ^ 0x7FFFFFFF); }

// scene[0..2] = min centroid (ordered int), scene[3..5] = max centroid
__global__ void gd_k_init_scene(int *scene) {
    if (threadIdx.x < 3) scene[threadIdx.x] = 0x7FFFFFFF;
    else if (threadIdx.x < 6) scene[threadIdx.x] = (int)0x80000000;
    else if (threadIdx.x < 16) scene[threadIdx.x] = 0;
}

// ---------------------------------------------------------------- mesh validation (gadep_load_mesh)
// Everything gadep_load_mesh promises to reject is found on the device, in the copies the BVH build will read: vertex
// coordinates that are not finite, surface / vertex indices out of range, zero-area triangles, and surfaces that are
// not closed and consistently oriented (PAPER.md:193 needs closed geometry): every directed edge of a surface must
// occur once and its reverse once, in the same surface -- one open-addressing table over all directed edges.
// err[k] = smallest offending index of class k (0xFFFFFFFF = none).
#define GD_ERR_NONFINITE 0    // vertex index
#define GD_ERR_SURFACE 1      // triangle index: surface id out of range
#define GD_ERR_VERTEX 2       // triangle index: vertex id out of range
#define GD_ERR_DEGENERATE 3   // triangle index
#define GD_ERR_EDGE_TWICE 4   // triangle index: a directed edge used twice
#define GD_ERR_OPEN 5         // surface id: an edge without its reverse in the same surface
#define GD_ERR_N 8
#define GD_EDGE_EMPTY (~0ull)

GD_D size_t gd_edge_slot(unsigned long long key, int shift) { return (size_t)((key * 0x9E3779B97F4A7C15ull) >> shift); }

__global__ void gd_k_check_verts(const float *__restrict__ verts, size_t n3, unsigned *err) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n3 && !isfinite(verts[i])) atomicMin(&err[GD_ERR_NONFINITE], (unsigned)(i / 3));
}

__global__ void gd_k_check_tris(const float *__restrict__ verts, const int *__restrict__ tris, const int *__restrict__ tri_surf,
                                int n_tri, int n_vert, int n_surf, const int *__restrict__ surf_sides, int *__restrict__ mats,
                                unsigned long long *ekey, int *esurf, size_t cap_mask, int shift, unsigned *err) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tri) return;
    const int s = tri_surf[t];
    if (s < 0 || s >= n_surf) { atomicMin(&err[GD_ERR_SURFACE], (unsigned)t); return; }
    const int v[3] = {tris[3 * t], tris[3 * t + 1], tris[3 * t + 2]};
    for (int k = 0; k < 3; ++k)
        if (v[k] < 0 || v[k] >= n_vert) { atomicMin(&err[GD_ERR_VERTEX], (unsigned)t); return; }
    const float *a = verts + 3 * (size_t)v[0], *b = verts + 3 * (size_t)v[1], *q = verts + 3 * (size_t)v[2];
    const double e1[3] = {(double)b[0] - a[0], (double)b[1] - a[1], (double)b[2] - a[2]};
    const double e2[3] = {(double)q[0] - a[0], (double)q[1] - a[1], (double)q[2] - a[2]};
    const double nx = e1[1] * e2[2] - e1[2] * e2[1], ny = e1[2] * e2[0] - e1[0] * e2[2], nz = e1[0] * e2[1] - e1[1] * e2[0];
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2] || !(nx * nx + ny * ny + nz * nz > 0.0)) {
        atomicMin(&err[GD_ERR_DEGENERATE], (unsigned)t);
        return;
    }
    mats[t] = (surf_sides[2 * s] & 0xFFFF) | (int)((unsigned)(surf_sides[2 * s + 1] & 0xFFFF) << 16);
    for (int k = 0; k < 3; ++k) {
        const unsigned long long key = ((unsigned long long)(unsigned)v[k] << 32) | (unsigned)v[(k + 1) % 3];
        size_t i = gd_edge_slot(key, shift);
        for (;;) {
            const unsigned long long seen = atomicCAS(&ekey[i], GD_EDGE_EMPTY, key);
            if (seen == GD_EDGE_EMPTY) { esurf[i] = s; break; }
            if (seen == key) { atomicMin(&err[GD_ERR_EDGE_TWICE], (unsigned)t); break; }
            i = (i + 1) & cap_mask;
        }
    }
}

__global__ void gd_k_check_closed(const unsigned long long *__restrict__ ekey, const int *__restrict__ esurf, size_t cap,
                                  int shift, unsigned *err) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cap) return;
    const unsigned long long key = ekey[i];
    if (key == GD_EDGE_EMPTY) return;
    const unsigned long long rev = (key << 32) | (key >> 32);
    size_t j = gd_edge_slot(rev, shift);
    while (ekey[j] != GD_EDGE_EMPTY && ekey[j] != rev) j = (j + 1) & (cap - 1);
    if (ekey[j] == GD_EDGE_EMPTY || esurf[j] != esurf[i]) atomicMin(&err[GD_ERR_OPEN], (unsigned)esurf[i]);
}

#define GD_MAX_SPLITS 16

GD_D void gd_load_tri(const float *__restrict__ verts, const int *__restrict__ tris, int i, float p[3][3], float lo[3],
                      float hi[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        int v = tris[3 * i + c];
#pragma unroll
        for (int a = 0; a < 3; ++a) p[c][a] = verts[3 * v + a];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        lo[a] = fminf(p[0][a], fminf(p[1][a], p[2][a]));
        hi[a] = fmaxf(p[0][a], fmaxf(p[1][a], p[2][a]));
    }
}

// Reference splitting under a global budget (after Karras & Aila 2013, restated): a facet's priority is the cube root
// of the area its AABB wastes; the extra references (at most one per facet on average) are handed out in proportion,
// never more than the looseness rule gd_split_count asks for.  Without the budget the 2 M-facet mesh of config 4
// (slivers of 0.05 x 3 mm at every azimuth) grew to 12 M references and a 3 GB hierarchy.
GD_D float gd_wasted_area(const float p[3][3], const float lo[3], const float hi[3]) {
    const float e0 = hi[0] - lo[0], e1 = hi[1] - lo[1], e2 = hi[2] - lo[2];
    const float ux = p[1][0] - p[0][0], uy = p[1][1] - p[0][1], uz = p[1][2] - p[0][2];
    const float vx = p[2][0] - p[0][0], vy = p[2][1] - p[0][1], vz = p[2][2] - p[0][2];
    const float cx = uy * vz - uz * vy, cy = uz * vx - ux * vz, cz = ux * vy - uy * vx;
    return fmaxf(e0 * e1 + e1 * e2 + e2 * e0 - sqrtf(cx * cx + cy * cy + cz * cz), 0.0f);
}
// pass 1: priority in fixed point (1e-3 mm^(2/3)) into counts[], exact integer sum into *prio_sum
__global__ void gd_k_split_prio(const float *__restrict__ verts, const int *__restrict__ tris, int n_tri,
                                unsigned *__restrict__ counts, unsigned long long *prio_sum) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned q = 0;
    if (i < n_tri) {
        float p[3][3], lo[3], hi[3];
        gd_load_tri(verts, tris, i, p, lo, hi);
        int axis;
        if (gd_split_count(p, lo, hi, GD_MAX_SPLITS, axis) > 1)
            q = (unsigned)fminf(cbrtf(gd_wasted_area(p, lo, hi)) * 1000.0f, 4.0e9f);
        counts[i] = q;
    }
    unsigned long long x = q;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
    if ((threadIdx.x & 31) == 0 && x) atomicAdd(prio_sum, x);
}
// pass 2: number of references of each facet
__global__ void gd_k_ref_count(const float *__restrict__ verts, const int *__restrict__ tris, int n_tri,
                               unsigned *__restrict__ counts, const unsigned long long *__restrict__ prio_sum,
                               unsigned long long budget) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_tri) return;
    float p[3][3], lo[3], hi[3];
    gd_load_tri(verts, tris, i, p, lo, hi);
    int axis;
    const int k_loose = gd_split_count(p, lo, hi, GD_MAX_SPLITS, axis);
    const unsigned long long total = *prio_sum;
    unsigned long long extra = total ? (unsigned long long)counts[i] * budget / total : 0ull;
    if (extra > (unsigned long long)(k_loose - 1)) extra = (unsigned long long)(k_loose - 1);
    counts[i] = 1u + (unsigned)extra;
}

// per reference: AABB (lo.w = centroid x, hi.w = centroid y), facet index; scene bounds of the centroids
__global__ void gd_k_make_refs(const float *__restrict__ verts, const int *__restrict__ tris, int n_tri,
                               const unsigned *__restrict__ offsets, unsigned n_ref, float4 *__restrict__ ref_lo,
                               float4 *__restrict__ ref_hi, int *__restrict__ ref_tri, int *scene) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int slo[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF};
    int shi[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    if (i < n_tri) {
        float p[3][3], lo[3], hi[3];
        gd_load_tri(verts, tris, i, p, lo, hi);
        int axis;
        gd_split_count(p, lo, hi, GD_MAX_SPLITS, axis);
        unsigned base = offsets[i];
        const int k = (int)((i + 1 < n_tri ? offsets[i + 1] : n_ref) - base);      // exclusive scan of the counts
        float ext = hi[axis] - lo[axis];
        for (int j = 0; j < k; ++j) {
            float rl[3] = {lo[0], lo[1], lo[2]}, rh[3] = {hi[0], hi[1], hi[2]};
            if (k > 1) {
                float a0 = lo[axis] + ext * (float)j / (float)k;
                float b0 = (j == k - 1) ? hi[axis] : lo[axis] + ext * (float)(j + 1) / (float)k;
                float cl[3], ch[3];
                gd_clip_tri_box(p, axis, a0, b0, cl, ch);
                if (cl[0] <= ch[0] && cl[1] <= ch[1] && cl[2] <= ch[2]) {      // else keep the whole facet box (safe)
#pragma unroll
                    for (int a = 0; a < 3; ++a) { rl[a] = fmaxf(cl[a], lo[a]); rh[a] = fminf(ch[a], hi[a]); }
                }
            }
            float cx = 0.5f * (rl[0] + rh[0]), cy = 0.5f * (rl[1] + rh[1]), cz = 0.5f * (rl[2] + rh[2]);
            ref_lo[base + j] = make_float4(rl[0], rl[1], rl[2], cx);
            ref_hi[base + j] = make_float4(rh[0], rh[1], rh[2], cy);
            ref_tri[base + j] = i;
            int ox = gd_f2o(cx), oy = gd_f2o(cy), oz = gd_f2o(cz);
            slo[0] = min(slo[0], ox); slo[1] = min(slo[1], oy); slo[2] = min(slo[2], oz);
            shi[0] = max(shi[0], ox); shi[1] = max(shi[1], oy); shi[2] = max(shi[2], oz);
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        slo[k] = __reduce_min_sync(0xFFFFFFFFu, slo[k]);
        shi[k] = __reduce_max_sync(0xFFFFFFFFu, shi[k]);
    }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { atomicMin(&scene[k], slo[k]); atomicMax(&scene[3 + k], shi[k]); }
    }
}

__global__ void gd_k_morton(const float4 *__restrict__ tri_lo, const float4 *__restrict__ tri_hi, int n_tri,
                            const int *__restrict__ scene, unsigned long long *__restrict__ keys,
                            unsigned *__restrict__ vals, const int *__restrict__ ref_tri, const int *__restrict__ tri_surf,
                            int cls_bits) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_tri) return;
    float sx = gd_o2f(scene[0]), sy = gd_o2f(scene[1]), sz = gd_o2f(scene[2]);
    float ex = gd_o2f(scene[3]) - sx, ey = gd_o2f(scene[4]) - sy, ez = gd_o2f(scene[5]) - sz;
    float4 lo = tri_lo[i], hi = tri_hi[i];
    float cx = lo.w, cy = hi.w, cz = 0.5f * (lo.z + hi.z);
    float nx = ex > 0.0f ? (cx - sx) / ex : 0.0f;
    float ny = ey > 0.0f ? (cy - sy) / ey : 0.0f;
    float nz = ez > 0.0f ? (cz - sz) / ez : 0.0f;
    unsigned long long key = gd_morton63(nx, ny, nz);
    // surface id above the Morton code: every closed surface becomes one subtree of the radix tree
    if (cls_bits > 0) key = (key >> (cls_bits - 1)) | ((unsigned long long)tri_surf[ref_tri[i]] << (64 - cls_bits));
    keys[i] = key;
    vals[i] = (unsigned)i;
}

// ---------------------------------------------------------------- LSD radix sort, 8 bits per pass
// hist[d * n_blocks + b] = number of keys of tile b with digit d
__global__ void gd_k_sort_hist(const unsigned long long *__restrict__ keys, int n, int shift, unsigned *hist,
                               int n_blocks) {
    __shared__ unsigned s_h[256];
    s_h[threadIdx.x] = 0;
    __syncthreads();
    int base = blockIdx.x * GD_SORT_TILE;
#pragma unroll
    for (int k = 0; k < GD_SORT_ITEMS; ++k) {
        int i = base + k * GD_SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&s_h[(unsigned)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[threadIdx.x * n_blocks + blockIdx.x] = s_h[threadIdx.x];
}

// exclusive scan of `count` unsigneds in place, single block of 1024 threads
__global__ void gd_k_scan(unsigned *data, int count, unsigned *total) {
    __shared__ unsigned s_w[32];
    __shared__ unsigned s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < count; base += 1024) {
        int i = base + threadIdx.x;
        unsigned v = i < count ? data[i] : 0u;
        unsigned x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xFFFFFFFFu, x, o); if ((threadIdx.x & 31) >= o) x += y; }
        if ((threadIdx.x & 31) == 31) s_w[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x < 32) {
            unsigned w = s_w[threadIdx.x], t = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(0xFFFFFFFFu, t, o); if (threadIdx.x >= o) t += y; }
            s_w[threadIdx.x] = t - w;
        }
        __syncthreads();
        unsigned carry = s_carry;
        unsigned excl = carry + s_w[threadIdx.x >> 5] + x - v;
        if (i < count) data[i] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = excl + v;
        __syncthreads();
    }
    if (total && threadIdx.x == 0) *total = s_carry;
}

// stable scatter: tile order, chunk order, lane order preserved
__global__ void gd_k_sort_scatter(const unsigned long long *__restrict__ keys_in, const unsigned *__restrict__ vals_in,
                                  unsigned long long *__restrict__ keys_out, unsigned *__restrict__ vals_out, int n,
                                  int shift, const unsigned *__restrict__ offsets, int n_blocks) {
    __shared__ unsigned s_base[256];
    __shared__ unsigned s_cnt[GD_SORT_THREADS / 32][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    s_base[threadIdx.x] = offsets[threadIdx.x * n_blocks + blockIdx.x];
    int base = blockIdx.x * GD_SORT_TILE;
    for (int k = 0; k < GD_SORT_ITEMS; ++k) {
#pragma unroll
        for (int w = 0; w < GD_SORT_THREADS / 32; ++w) s_cnt[w][threadIdx.x] = 0;
        __syncthreads();
        int i = base + k * GD_SORT_THREADS + threadIdx.x;
        bool valid = i < n;
        unsigned long long key = valid ? keys_in[i] : 0ull;
        unsigned val = valid ? vals_in[i] : 0u;
        unsigned d = valid ? ((unsigned)(key >> shift) & 255u) : 256u + (unsigned)lane;   // invalid lanes match nobody
        unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
        unsigned rank = __popc(peers & ((1u << lane) - 1u));
        if (valid && rank == 0) s_cnt[warp][d] = __popc(peers);
        __syncthreads();
        {   // thread = digit: offsets of each warp's group, then advance the block's running base
            unsigned run = s_base[threadIdx.x];
#pragma unroll
            for (int w = 0; w < GD_SORT_THREADS / 32; ++w) { unsigned c = s_cnt[w][threadIdx.x]; s_cnt[w][threadIdx.x] = run; run += c; }
            s_base[threadIdx.x] = run;
        }
        __syncthreads();
        if (valid) {
            unsigned pos = s_cnt[warp][d] + rank;
            keys_out[pos] = key;
            vals_out[pos] = val;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- Karras radix tree
// internal node i in [0, n-1); children encoded >= 0 internal, < 0 leaf (~sorted index)
__global__ void gd_k_karras(const unsigned long long *__restrict__ keys, int n, int *__restrict__ child_l,
                            int *__restrict__ child_r, int *__restrict__ parent_int, int *__restrict__ parent_leaf,
                            int cls_bits, int *__restrict__ surf_entry) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n - 1) return;
    int first, last, split;
    gd_karras_node(keys, n, i, first, last, split);
    int l, r;
    if (first == split) { l = ~split; parent_leaf[split] = i; } else { l = split; parent_int[split] = i; }
    if (last == split + 1) { r = ~(split + 1); parent_leaf[split + 1] = i; } else { r = split + 1; parent_int[split + 1] = i; }
    child_l[i] = l;
    child_r[i] = r;
    if (i == 0) parent_int[0] = -1;
    if (cls_bits > 0) {        // the node that covers exactly the references of one surface is that surface's entry
        const int sh = 64 - cls_bits;
        const unsigned long long ca = keys[first] >> sh, cb = keys[last] >> sh;
        if (ca == cb && (first == 0 || (keys[first - 1] >> sh) != ca) && (last == n - 1 || (keys[last + 1] >> sh) != ca))
            surf_entry[ca] = i;
    }
}

// leaf-ordered triangle records
__global__ void gd_k_leaf_tris(const float *__restrict__ verts, const int *__restrict__ tris,
                               const int *__restrict__ tri_mats, const int *__restrict__ tri_surf,
                               const int *__restrict__ ref_tri, const unsigned *__restrict__ order, int n,
                               GdTri *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int o = ref_tri[order[i]];
    int a = tris[3 * o], b = tris[3 * o + 1], c = tris[3 * o + 2];
    GdTri t;
    t.v0 = make_float4(verts[3 * a], verts[3 * a + 1], verts[3 * a + 2], __int_as_float(o));
    t.v1 = make_float4(verts[3 * b], verts[3 * b + 1], verts[3 * b + 2], __int_as_float(tri_mats[o]));
    t.v2 = make_float4(verts[3 * c], verts[3 * c + 1], verts[3 * c + 2], __int_as_float(tri_surf[o]));
    out[i] = t;
}

GD_D void gd_child_box(int child, const float4 *tri_lo, const float4 *tri_hi, const unsigned *order,
                       const float4 *node_lo, const float4 *node_hi, float4 &lo, float4 &hi, int &depth) {
    if (child < 0) {
        int o = (int)order[~child];
        lo = tri_lo[o]; hi = tri_hi[o]; depth = 0;
    } else {
        lo = __ldcg(&node_lo[child]); hi = __ldcg(&node_hi[child]);
        depth = __float_as_int(lo.w);
    }
}

// bottom-up refit: the second thread to reach a node owns it; emits the traversal node
__global__ void gd_k_refit(int n, const int *__restrict__ child_l, const int *__restrict__ child_r,
                           const int *__restrict__ parent_int, const int *__restrict__ parent_leaf,
                           const float4 *__restrict__ tri_lo, const float4 *__restrict__ tri_hi,
                           const unsigned *__restrict__ order, float4 *node_lo, float4 *node_hi, int *visits,
                           GdNode *__restrict__ nodes, int *max_depth) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int cur = parent_leaf[i];
    while (cur >= 0) {
        __threadfence();
        if (atomicAdd(&visits[cur], 1) == 0) return;
        int l = child_l[cur], r = child_r[cur];
        float4 llo, lhi, rlo, rhi;
        int dl, dr;
        gd_child_box(l, tri_lo, tri_hi, order, node_lo, node_hi, llo, lhi, dl);
        gd_child_box(r, tri_lo, tri_hi, order, node_lo, node_hi, rlo, rhi, dr);
        GdNode nd;
        nd.n0xy = make_float4(llo.x, lhi.x, llo.y, lhi.y);
        nd.n1xy = make_float4(rlo.x, rhi.x, rlo.y, rhi.y);
        nd.nz = make_float4(llo.z, lhi.z, rlo.z, rhi.z);
        nd.link = make_int4(l, r, 0, 0);
        nodes[cur] = nd;
        int depth = 1 + max(dl, dr);
        float4 lo = make_float4(fminf(llo.x, rlo.x), fminf(llo.y, rlo.y), fminf(llo.z, rlo.z), __int_as_float(depth));
        float4 hi = make_float4(fmaxf(lhi.x, rhi.x), fmaxf(lhi.y, rhi.y), fmaxf(lhi.z, rhi.z), 0.0f);
        __stcg(&node_lo[cur], lo);
        __stcg(&node_hi[cur], hi);
        if (cur == 0) { *max_depth = depth; return; }
        cur = parent_int[cur];
    }
}

// ---------------------------------------------------------------- 4-wide collapse
// Node4(i) holds up to four descendants of binary node i: starting from its two children, the inner child with the
// largest box surface is replaced by its own two children until there are four entries or only leaves are left
// (surface-area-guided collapse; a fixed "grandchildren" rule wastes entries on tiny subtrees).  Written for every
// binary node; the traversal only ever reaches those that are an entry of another Node4 (or the root).
GD_D float gd_half_area(const float4 lo, const float4 hi) {
    const float ex = hi.x - lo.x, ey = hi.y - lo.y, ez = hi.z - lo.z;
    return ex * ey + ey * ez + ez * ex;
}
__global__ void gd_k_collapse4(int n_inner, const int *__restrict__ child_l, const int *__restrict__ child_r,
                               const float4 *__restrict__ ref_lo, const float4 *__restrict__ ref_hi,
                               const unsigned *__restrict__ order, const float4 *__restrict__ node_lo,
                               const float4 *__restrict__ node_hi, GdNode4 *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_inner) return;
    int c[4] = {child_l[i], child_r[i], GD_NO_CHILD, GD_NO_CHILD};
    int k = 2;
    while (k < 4) {
        int best = -1;
        float best_a = -1.0f;
        for (int j = 0; j < k; ++j)
            if (c[j] >= 0) {
                const float a = gd_half_area(node_lo[c[j]], node_hi[c[j]]);
                if (a > best_a) { best_a = a; best = j; }
            }
        if (best < 0) break;
        const int b = c[best];
        c[best] = child_l[b];
        c[k++] = child_r[b];
    }
    float lo[4][3], hi[4][3];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (c[j] != GD_NO_CHILD) {
            if (c[j] < 0) { int o = (int)order[~c[j]]; a = ref_lo[o]; b = ref_hi[o]; }
            else { a = node_lo[c[j]]; b = node_hi[c[j]]; }
        }
        lo[j][0] = a.x; lo[j][1] = a.y; lo[j][2] = a.z; hi[j][0] = b.x; hi[j][1] = b.y; hi[j][2] = b.z;
    }
    GdNode4 nd;
    nd.lox = make_float4(lo[0][0], lo[1][0], lo[2][0], lo[3][0]); nd.hix = make_float4(hi[0][0], hi[1][0], hi[2][0], hi[3][0]);
    nd.loy = make_float4(lo[0][1], lo[1][1], lo[2][1], lo[3][1]); nd.hiy = make_float4(hi[0][1], hi[1][1], hi[2][1], hi[3][1]);
    nd.loz = make_float4(lo[0][2], lo[1][2], lo[2][2], lo[3][2]); nd.hiz = make_float4(hi[0][2], hi[1][2], hi[2][2], hi[3][2]);
    nd.child = make_int4(c[0], c[1], c[2], c[3]);
    nd.pad = make_int4(0, 0, 0, 0);
    out[i] = nd;
}

// 8-wide compressed nodes (GdNode8, gadep_common.cuh): greedy expansion to eight descendants, octant slots,
// outward 8-bit quantisation.  One per binary inner node, like the 4-wide nodes.
__global__ void gd_k_collapse8(int n_inner, const int *__restrict__ child_l, const int *__restrict__ child_r,
                               const float4 *__restrict__ ref_lo, const float4 *__restrict__ ref_hi,
                               const unsigned *__restrict__ order, const float4 *__restrict__ node_lo,
                               const float4 *__restrict__ node_hi, GdNode8 *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_inner) return;
    int c[8] = {child_l[i], child_r[i], GD_NO_CHILD, GD_NO_CHILD, GD_NO_CHILD, GD_NO_CHILD, GD_NO_CHILD, GD_NO_CHILD};
    int k = 2;
    while (k < 8) {
        int best = -1;
        float best_a = -1.0f;
        for (int j = 0; j < k; ++j)
            if (c[j] >= 0) {
                const float a = gd_half_area(node_lo[c[j]], node_hi[c[j]]);
                if (a > best_a) { best_a = a; best = j; }
            }
        if (best < 0) break;
        const int b = c[best];
        c[best] = child_l[b];
        c[k++] = child_r[b];
    }
    const float4 nlo = node_lo[i], nhi = node_hi[i];
    const float blo[3] = {nlo.x, nlo.y, nlo.z}, bhi[3] = {nhi.x, nhi.y, nhi.z};
    float clo[8][3], chi[8][3];
    for (int j = 0; j < k; ++j) {
        float4 a, b;
        if (c[j] < 0) { const int o = (int)order[~c[j]]; a = ref_lo[o]; b = ref_hi[o]; }
        else { a = node_lo[c[j]]; b = node_hi[c[j]]; }
        clo[j][0] = a.x; clo[j][1] = a.y; clo[j][2] = a.z; chi[j][0] = b.x; chi[j][1] = b.y; chi[j][2] = b.z;
    }
    // octant slots: child j likes slot s by how far its centre lies from the node's centre on the side s names
    int slot_of[8], child_in[8];
    for (int s = 0; s < 8; ++s) child_in[s] = -1;
    for (int j = 0; j < 8; ++j) slot_of[j] = -1;
    for (int it = 0; it < k; ++it) {
        float best = -3.0e38f;
        int bj = -1, bs = -1;
        for (int j = 0; j < k; ++j) {
            if (slot_of[j] >= 0) continue;
            float d[3];
            for (int a = 0; a < 3; ++a) d[a] = 0.5f * (clo[j][a] + chi[j][a]) - 0.5f * (blo[a] + bhi[a]);
            for (int s = 0; s < 8; ++s) {
                if (child_in[s] >= 0) continue;
                const float v = ((s & 1) ? d[0] : -d[0]) + ((s & 2) ? d[1] : -d[1]) + ((s & 4) ? d[2] : -d[2]);
                if (v > best) { best = v; bj = j; bs = s; }
            }
        }
        slot_of[bj] = bs; child_in[bs] = bj;
    }
    GdNode8 nd;
    unsigned q[3][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
    unsigned exyz = 0, valid = 0;
    float org[3];
    for (int a = 0; a < 3; ++a) {
        const float ext = bhi[a] - blo[a];
        int e = -100;
        if (ext > 0.0f) {
            int kk;
            const float m = frexpf(ext, &kk);               // ext = m 2^kk, m in [0.5, 1)
            e = m * 256.0f <= 254.5f ? kk - 8 : kk - 7;     // (hi - o) / 2^e + margins stays <= 255
            e = e < -100 ? -100 : (e > 100 ? 100 : e);
        }
        const float S = __int_as_float((e + 127) << 23), invS = __int_as_float((127 - e) << 23);
        const float o = blo[a] - S * (1.0f / 32.0f);
        org[a] = o;
        exyz |= (unsigned)(e + 127) << (8 * a);
        for (int s = 0; s < 8; ++s) {
            unsigned ql = 255u, qh = 0u;
            const int j = child_in[s];
            if (j >= 0) {
                const float fl = floorf((clo[j][a] - o) * invS - (1.0f / 64.0f));
                const float fh = ceilf((chi[j][a] - o) * invS + (1.0f / 64.0f));
                ql = (unsigned)fminf(fmaxf(fl, 0.0f), 255.0f);
                qh = (unsigned)fminf(fmaxf(fh, 0.0f), 255.0f);
            }
            q[a][s >> 2] |= ql << (8 * (s & 3));
            q[a][2 + (s >> 2)] |= qh << (8 * (s & 3));
        }
    }
    for (int s = 0; s < 8; ++s) {
        nd.child[s] = child_in[s] >= 0 ? c[child_in[s]] : GD_NO_CHILD;
        if (child_in[s] >= 0) valid |= 1u << s;
    }
    nd.ox = org[0]; nd.oy = org[1]; nd.oz = org[2];
    nd.exyz_valid = exyz | (valid << 24);
    for (int w = 0; w < 4; ++w) { nd.qx[w] = q[0][w]; nd.qy[w] = q[1][w]; nd.qz[w] = q[2][w]; }
    out[i] = nd;
}

// 4-wide compressed nodes (GdNode4q): the children of gd_k_collapse4 (same choice, same order), boxes quantised like
// gd_k_collapse8 on the grid of the binary node's own box.
__global__ void gd_k_collapse4q(int n_inner, const int *__restrict__ child_l, const int *__restrict__ child_r,
                                const float4 *__restrict__ ref_lo, const float4 *__restrict__ ref_hi,
                                const unsigned *__restrict__ order, const float4 *__restrict__ node_lo,
                                const float4 *__restrict__ node_hi, GdNode4q *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_inner) return;
    int c[4] = {child_l[i], child_r[i], GD_NO_CHILD, GD_NO_CHILD};
    int k = 2;
    while (k < 4) {
        int best = -1;
        float best_a = -1.0f;
        for (int j = 0; j < k; ++j)
            if (c[j] >= 0) {
                const float a = gd_half_area(node_lo[c[j]], node_hi[c[j]]);
                if (a > best_a) { best_a = a; best = j; }
            }
        if (best < 0) break;
        const int b = c[best];
        c[best] = child_l[b];
        c[k++] = child_r[b];
    }
    const float4 nlo = node_lo[i], nhi = node_hi[i];
    const float blo[3] = {nlo.x, nlo.y, nlo.z}, bhi[3] = {nhi.x, nhi.y, nhi.z};
    float clo[4][3], chi[4][3];
    for (int j = 0; j < 4; ++j) {
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
        if (c[j] != GD_NO_CHILD) {
            if (c[j] < 0) { const int o = (int)order[~c[j]]; a = ref_lo[o]; b = ref_hi[o]; }
            else { a = node_lo[c[j]]; b = node_hi[c[j]]; }
        }
        clo[j][0] = a.x; clo[j][1] = a.y; clo[j][2] = a.z; chi[j][0] = b.x; chi[j][1] = b.y; chi[j][2] = b.z;
    }
    unsigned q[3][2] = {{0, 0}, {0, 0}, {0, 0}};
    unsigned exyz = 0;
    float org[3];
    for (int a = 0; a < 3; ++a) {
        const float ext = bhi[a] - blo[a];
        int e = -100;
        if (ext > 0.0f) {
            int kk;
            const float m = frexpf(ext, &kk);               // ext = m 2^kk, m in [0.5, 1)
            e = m * 256.0f <= 254.5f ? kk - 8 : kk - 7;     // (hi - o) / 2^e + margins stays <= 255
            e = e < -100 ? -100 : (e > 100 ? 100 : e);
        }
        const float S = __int_as_float((e + 127) << 23), invS = __int_as_float((127 - e) << 23);
        const float o = blo[a] - S * (1.0f / 32.0f);
        org[a] = o;
        exyz |= (unsigned)(e + 127) << (8 * a);
        for (int j = 0; j < 4; ++j) {
            unsigned ql = 255u, qh = 0u;
            if (c[j] != GD_NO_CHILD) {
                const float fl = floorf((clo[j][a] - o) * invS - (1.0f / 64.0f));
                const float fh = ceilf((chi[j][a] - o) * invS + (1.0f / 64.0f));
                ql = (unsigned)fminf(fmaxf(fl, 0.0f), 255.0f);
                qh = (unsigned)fminf(fmaxf(fh, 0.0f), 255.0f);
            }
            q[a][0] |= ql << (8 * j);
            q[a][1] |= qh << (8 * j);
        }
    }
    GdNode4q nd;
    nd.ox = org[0]; nd.oy = org[1]; nd.oz = org[2]; nd.exyz = exyz;
    nd.qx_lo = q[0][0]; nd.qx_hi = q[0][1]; nd.qy_lo = q[1][0]; nd.qy_hi = q[1][1]; nd.qz_lo = q[2][0]; nd.qz_hi = q[2][1];
    nd.pad0 = 0; nd.pad1 = 0;
    for (int j = 0; j < 4; ++j) nd.child[j] = c[j];
    out[i] = nd;
}

// ---------------------------------------------------------------- facet-clearance grid (GdGrid, gadep_common.cuh)
// 1. every cell a reference box touches is marked; 2. exact Euclidean distance transform of the marks in cell units,
// separable (x by two sweeps per row, then y and z as windowed lower envelopes), capped at GD_GRID_WINDOW + 1 cells;
// 3. clearance of a cell = (centre-to-centre distance - sqrt(3)) h: two points of the two cells are at least that far
// apart.  Everything is rounded towards "nearer", so the stored value never exceeds the true clearance.
#define GD_GRID_WINDOW 16
// per_lane != 0: one reference box per lane, a box of more than 16 cells is marked by the whole warp (many small facets);
// per_lane == 0: one reference box per warp (few, large facets)
__global__ void gd_k_grid_mark(const float4 *__restrict__ ref_lo, const float4 *__restrict__ ref_hi, int n_ref, GdGrid g,
                               unsigned char *__restrict__ occ, int per_lane) {
    const int lane = threadIdx.x & 31;
    const int i = per_lane ? blockIdx.x * blockDim.x + threadIdx.x : (lane == 0 ? (int)(((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5) : n_ref);
    int x0 = 0, x1 = -1, y0 = 0, y1 = -1, z0 = 0, z1 = -1;
    if (i < n_ref) {
        const float4 lo = ref_lo[i], hi = ref_hi[i];
        const float pad = 2.0e-4f;      // float32 slack of the boxes and of the cell index computed in the transport kernel
        const float ex = pad + 1.0e-6f * fmaxf(fabsf(lo.x), fabsf(hi.x)), ey = pad + 1.0e-6f * fmaxf(fabsf(lo.y), fabsf(hi.y)),
                    ez = pad + 1.0e-6f * fmaxf(fabsf(lo.z), fabsf(hi.z));
        x0 = max((int)floorf((lo.x - ex - g.lox) * g.inv_h), 0); x1 = min((int)floorf((hi.x + ex - g.lox) * g.inv_h), g.nx - 1);
        y0 = max((int)floorf((lo.y - ey - g.loy) * g.inv_h), 0); y1 = min((int)floorf((hi.y + ey - g.loy) * g.inv_h), g.ny - 1);
        z0 = max((int)floorf((lo.z - ez - g.loz) * g.inv_h), 0); z1 = min((int)floorf((hi.z + ez - g.loz) * g.inv_h), g.nz - 1);
    }
    const bool any = x1 >= x0 && y1 >= y0 && z1 >= z0;
    const long long n = any ? (long long)(x1 - x0 + 1) * (y1 - y0 + 1) * (z1 - z0 + 1) : 0;
    if (any && n <= 16)
        for (int z = z0; z <= z1; ++z)
            for (int y = y0; y <= y1; ++y)
                for (int x = x0; x <= x1; ++x) occ[((size_t)z * g.ny + y) * g.nx + x] = 1;
    unsigned big = __ballot_sync(0xFFFFFFFFu, n > 16);
    while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const int bx0 = __shfl_sync(0xFFFFFFFFu, x0, src), bx1 = __shfl_sync(0xFFFFFFFFu, x1, src);
        const int by0 = __shfl_sync(0xFFFFFFFFu, y0, src), by1 = __shfl_sync(0xFFFFFFFFu, y1, src);
        const int bz0 = __shfl_sync(0xFFFFFFFFu, z0, src), bz1 = __shfl_sync(0xFFFFFFFFu, z1, src);
        const int wx = bx1 - bx0 + 1, wy = by1 - by0 + 1;
        const long long nb = (long long)wx * wy * (bz1 - bz0 + 1);
        for (long long k = lane; k < nb; k += 32) {
            const int x = bx0 + (int)(k % wx), y = by0 + (int)((k / wx) % wy), z = bz0 + (int)(k / ((long long)wx * wy));
            occ[((size_t)z * g.ny + y) * g.nx + x] = 1;
        }
    }
}
// rows along x: occ (1 = marked) -> distance in cells to the nearest marked cell of the row, capped, in place
__global__ void gd_k_grid_dt_x(GdGrid g, unsigned char *__restrict__ occ) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= g.ny * g.nz) return;
    unsigned char *row = occ + (size_t)r * g.nx;
    const int cap = GD_GRID_WINDOW + 1;
    int d = cap;
    for (int x = 0; x < g.nx; ++x) { d = row[x] == 1 ? 0 : min(d + 1, cap); row[x] = (unsigned char)(row[x] == 1 ? 0x80 : d); }   // 0x80 = marked
    d = cap;
    for (int x = g.nx - 1; x >= 0; --x) {
        const int v = row[x];
        d = v == 0x80 ? 0 : min(d + 1, cap);
        row[x] = (unsigned char)(v == 0x80 ? 0 : min(v, d));
    }
}
__global__ void gd_k_grid_dt_y(GdGrid g, const unsigned char *__restrict__ gx, unsigned short *__restrict__ d2) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n = (size_t)g.nx * g.ny * g.nz;
    if (i >= n) return;
    const int x = (int)(i % g.nx), y = (int)((i / g.nx) % g.ny);
    const int cap = GD_GRID_WINDOW + 1;
    int best = cap * cap;
    const int a = max(y - GD_GRID_WINDOW, 0), b = min(y + GD_GRID_WINDOW, g.ny - 1);
    const unsigned char *col = gx + (i - (size_t)y * g.nx);
    for (int yy = a; yy <= b; ++yy) {
        const int v = col[(size_t)yy * g.nx], dy = yy - y;
        best = min(best, v * v + dy * dy);
    }
    (void)x;
    d2[i] = (unsigned short)best;
}
__global__ void gd_k_grid_dt_z(GdGrid g, const unsigned short *__restrict__ d2, unsigned char *__restrict__ out,
                               unsigned *__restrict__ info) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t plane = (size_t)g.nx * g.ny, n = plane * g.nz;
    if (i >= n) return;
    const int z = (int)(i / plane);
    const int cap = GD_GRID_WINDOW + 1;
    int best = cap * cap;
    const int a = max(z - GD_GRID_WINDOW, 0), b = min(z + GD_GRID_WINDOW, g.nz - 1);
    const unsigned short *col = d2 + (i - (size_t)z * plane);
    for (int zz = a; zz <= b; ++zz) {
        const int dz = zz - z;
        best = min(best, (int)col[(size_t)zz * plane] + dz * dz);
    }
    // centre distance sqrt(best) cells; any two points of the two cells: at least sqrt(best) - sqrt(3) cells apart
    const float cl = sqrtf((float)best) * 0.999999f - 1.7320509f;
    const unsigned char v = (unsigned char)fminf(fmaxf(floorf(cl * 4.0f), 0.0f), 255.0f);
    out[i] = v;
    info[i] = v;          // GdGrid::info: bit 31 clear = scalar bound only
}

// ---- the cells' 32-bit words (GdGrid::info) and the plane lists of the cells near facets.  One thread per cell.  A cell
// whose scalar clearance is below `thr` (= the reach in units of h / 4; 0 = no lists) gets a list: a box query of the
// 4-wide hierarchy with the cell dilated by the reach collects the facets that can come within reach of a point of the
// cell (every reference box that overlaps the dilated cell; a facet whose plane passes farther than reach + half a cell
// diagonal from the centre is dropped), their planes (gd_k_tri_normals) are referred to the cell centre and merged when
// they agree to 2e-5 mm over the cell.  More than GD_CELL_PLANES distinct planes, more than GD_LIST_MAX_CANDIDATES
// reference boxes, or a query that runs out of stack: no list (the BVH answers).
__global__ void gd_k_grid_list_count(const unsigned char *__restrict__ cells, size_t n, unsigned thr, unsigned *count) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool want = i < n && cells[i] < thr;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, want);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(count, (unsigned)__popc(m));
}
// unit normal of every leaf-ordered triangle, from the float32 vertices in double, rounded to float32; w = 0 marks a
// triangle without a normal.  (The plane through v0 with the rounded normal leaves the triangle's own plane by at most
// 6e-8 x the triangle's extent: < 1e-5 mm.)
__global__ void gd_k_tri_normals(const GdTri *__restrict__ tris, int n, float4 *__restrict__ nrm) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const GdTri tr = tris[i];
    const double e1x = (double)tr.v1.x - tr.v0.x, e1y = (double)tr.v1.y - tr.v0.y, e1z = (double)tr.v1.z - tr.v0.z;
    const double e2x = (double)tr.v2.x - tr.v0.x, e2y = (double)tr.v2.y - tr.v0.y, e2z = (double)tr.v2.z - tr.v0.z;
    const double nx = e1y * e2z - e1z * e2y, ny = e1z * e2x - e1x * e2z, nz = e1x * e2y - e1y * e2x;
    const double len = sqrt(nx * nx + ny * ny + nz * nz);
    nrm[i] = len > 0.0 ? make_float4((float)(nx / len), (float)(ny / len), (float)(nz / len), 1.0f) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
}
#define GD_LIST_MAX_CANDIDATES 96   // reference boxes looked at per cell before the cell is given up (dense meshes)
__global__ void __launch_bounds__(128)
gd_k_grid_planes(GdGrid g, const unsigned char *__restrict__ cells, unsigned thr, const GdNode4 *__restrict__ nodes4,
                 const GdTri *__restrict__ tris, const float4 *__restrict__ nrm, unsigned *__restrict__ info,
                 float4 *__restrict__ planes, unsigned *counter, unsigned capacity) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n = (size_t)g.nx * g.ny * g.nz;
    if (i >= n) return;
    const unsigned scalar = cells[i];
    info[i] = scalar;
    if (scalar >= thr) return;
    const int ix = (int)(i % g.nx), iy = (int)((i / g.nx) % g.ny), iz = (int)(i / ((size_t)g.nx * g.ny));
    // the centre exactly as gd_flight_clear computes it
    const float cx = fmaf((float)ix + 0.5f, g.h, g.lox), cy = fmaf((float)iy + 0.5f, g.h, g.loy), cz = fmaf((float)iz + 0.5f, g.h, g.loz);
    const float half = 0.5f * g.h * 1.0001f, pad = 1.0e-3f;
    const float r = half + g.reach + pad + 1.0e-6f * fmaxf(fmaxf(fabsf(cx), fabsf(cy)), fabsf(cz));
    const float qlx = cx - r, qhx = cx + r, qly = cy - r, qhy = cy + r, qlz = cz - r, qhz = cz + r;
    const float far_plane = g.reach + 0.8661f * g.h + pad;
    float4 pl[GD_CELL_PLANES];
    int cnt = 0, n_cand = 0;
    bool overflow = false;
    int stack[96];
    int sp = 0, node = 0;
    for (;;) {
        const GdNode4 nd = nodes4[node];
        const float lo_x[4] = {nd.lox.x, nd.lox.y, nd.lox.z, nd.lox.w}, hi_x[4] = {nd.hix.x, nd.hix.y, nd.hix.z, nd.hix.w};
        const float lo_y[4] = {nd.loy.x, nd.loy.y, nd.loy.z, nd.loy.w}, hi_y[4] = {nd.hiy.x, nd.hiy.y, nd.hiy.z, nd.hiy.w};
        const float lo_z[4] = {nd.loz.x, nd.loz.y, nd.loz.z, nd.loz.w}, hi_z[4] = {nd.hiz.x, nd.hiz.y, nd.hiz.z, nd.hiz.w};
        const int ch[4] = {nd.child.x, nd.child.y, nd.child.z, nd.child.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (ch[k] == GD_NO_CHILD) continue;
            if (lo_x[k] > qhx || hi_x[k] < qlx || lo_y[k] > qhy || hi_y[k] < qly || lo_z[k] > qhz || hi_z[k] < qlz) continue;
            if (ch[k] >= 0) {
                if (sp == 96) overflow = true; else stack[sp++] = ch[k];
                continue;
            }
            if (++n_cand > GD_LIST_MAX_CANDIDATES) { overflow = true; continue; }
            const float4 nf = nrm[~ch[k]];
            if (nf.w == 0.0f) { overflow = true; continue; }
            const float4 v0 = tris[~ch[k]].v0;
            // signed distance of the cell centre from the plane through v0, in double (the centre and v0 are ~100 mm, the
            // distance ~1 mm and wanted to 1e-5)
            const double d = (double)nf.x * ((double)cx - v0.x) + (double)nf.y * ((double)cy - v0.y) + (double)nf.z * ((double)cz - v0.z);
            const float df = (float)d;
            if (fabsf(df) > far_plane) continue;
            const float4 q = make_float4(nf.x, nf.y, nf.z, df);
            bool seen = false;
            for (int j = 0; j < cnt; ++j) {
                const float sgn = (q.x * pl[j].x + q.y * pl[j].y + q.z * pl[j].z) < 0.0f ? -1.0f : 1.0f;
                const float dn = fabsf(q.x - sgn * pl[j].x) + fabsf(q.y - sgn * pl[j].y) + fabsf(q.z - sgn * pl[j].z);
                seen = seen || dn * r + fabsf(q.w - sgn * pl[j].w) < 2.0e-5f;
            }
            if (seen) continue;
            if (cnt == GD_CELL_PLANES) overflow = true; else pl[cnt++] = q;
        }
        if (overflow || sp == 0) break;
        node = stack[--sp];
    }
    if (overflow) return;
    const unsigned low = scalar < 7u ? scalar : 7u;          // the scalar bound stays valid rounded down
    if (cnt == 0) { info[i] = GD_CELL_LIST | (15u << 3) | low; return; }
    const unsigned slot = atomicAdd(counter, 1u);
    if (slot >= capacity || slot >= (1u << 24)) return;
    for (int k = 0; k < cnt; ++k) planes[(size_t)slot * GD_CELL_PLANES + k] = pl[k];
    info[i] = GD_CELL_LIST | (slot << 7) | ((unsigned)cnt << 3) | low;
}
