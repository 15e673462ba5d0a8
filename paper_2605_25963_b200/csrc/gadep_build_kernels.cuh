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
}

// per facet: AABB (lo, hi as float4 pairs) and centroid bounds of the scene
__global__ void gd_k_tri_bounds(const float *__restrict__ verts, const int *__restrict__ tris, int n_tri,
                                float4 *__restrict__ tri_lo, float4 *__restrict__ tri_hi, int *scene) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float cx = 0, cy = 0, cz = 0;
    bool ok = i < n_tri;
    if (ok) {
        int a = tris[3 * i], b = tris[3 * i + 1], c = tris[3 * i + 2];
        float ax = verts[3 * a], ay = verts[3 * a + 1], az = verts[3 * a + 2];
        float bx = verts[3 * b], by = verts[3 * b + 1], bz = verts[3 * b + 2];
        float qx = verts[3 * c], qy = verts[3 * c + 1], qz = verts[3 * c + 2];
        float lx = fminf(ax, fminf(bx, qx)), ly = fminf(ay, fminf(by, qy)), lz = fminf(az, fminf(bz, qz));
        float hx = fmaxf(ax, fmaxf(bx, qx)), hy = fmaxf(ay, fmaxf(by, qy)), hz = fmaxf(az, fmaxf(bz, qz));
        cx = 0.5f * (lx + hx); cy = 0.5f * (ly + hy); cz = 0.5f * (lz + hz);
        tri_lo[i] = make_float4(lx, ly, lz, cx);
        tri_hi[i] = make_float4(hx, hy, hz, cy);
    }
    int lo[3] = {ok ? gd_f2o(cx) : 0x7FFFFFFF, ok ? gd_f2o(cy) : 0x7FFFFFFF, ok ? gd_f2o(cz) : 0x7FFFFFFF};
    int hi[3] = {ok ? gd_f2o(cx) : (int)0x80000000, ok ? gd_f2o(cy) : (int)0x80000000, ok ? gd_f2o(cz) : (int)0x80000000};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        lo[k] = __reduce_min_sync(0xFFFFFFFFu, lo[k]);
        hi[k] = __reduce_max_sync(0xFFFFFFFFu, hi[k]);
    }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { atomicMin(&scene[k], lo[k]); atomicMax(&scene[3 + k], hi[k]); }
    }
}

__global__ void gd_k_morton(const float4 *__restrict__ tri_lo, const float4 *__restrict__ tri_hi, int n_tri,
                            const int *__restrict__ scene, unsigned long long *__restrict__ keys,
                            unsigned *__restrict__ vals) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_tri) return;
    float sx = gd_o2f(scene[0]), sy = gd_o2f(scene[1]), sz = gd_o2f(scene[2]);
    float ex = gd_o2f(scene[3]) - sx, ey = gd_o2f(scene[4]) - sy, ez = gd_o2f(scene[5]) - sz;
    float4 lo = tri_lo[i], hi = tri_hi[i];
    float cx = lo.w, cy = hi.w, cz = 0.5f * (lo.z + hi.z);
    float nx = ex > 0.0f ? (cx - sx) / ex : 0.0f;
    float ny = ey > 0.0f ? (cy - sy) / ey : 0.0f;
    float nz = ez > 0.0f ? (cz - sz) / ez : 0.0f;
    keys[i] = gd_morton63(nx, ny, nz);
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
__global__ void gd_k_scan(unsigned *data, int count) {
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
                            int *__restrict__ child_r, int *__restrict__ parent_int, int *__restrict__ parent_leaf) {
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
}

// leaf-ordered triangle records
__global__ void gd_k_leaf_tris(const float *__restrict__ verts, const int *__restrict__ tris,
                               const int *__restrict__ tri_mats, const int *__restrict__ tri_surf,
                               const unsigned *__restrict__ order, int n, GdTri *__restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int o = (int)order[i];
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
