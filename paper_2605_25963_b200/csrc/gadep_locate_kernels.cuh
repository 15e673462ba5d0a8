// gadep_locate_kernels.cuh -- material localisation of points (sec 2.4.2).
//   mode 0  side-id rule ("original algorithm"): nearest facet ahead, entering / leaving from its normal,
//           material from that facet's side ids.
//   mode 1  parity rule (the paper's reworked algorithm): intersections of the ray with every closed
//           geometry are counted through an all-hits BVH traversal; among the geometries with an odd count the one
//           whose first intersection is nearest contains the point; none odd -> world medium.
// One ray per thread, plain per-lane loop (this is a query hook and the measurement of the paper's localisation
// cost, not the transport loop).
#pragma once
#include "gadep_trav.cuh"

#define GD_LOC_MAX_HITS 96
#define GD_LOC_OVERFLOW (-3)     // more than GD_LOC_MAX_HITS facets along one ray

__global__ void __launch_bounds__(128)
gd_k_locate(GdBvh bvh, const float *__restrict__ org, const float *__restrict__ dir, long long n, int mode,
            int world_material, int *__restrict__ mat_out, GdCounters *counters) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned n_box = 0, n_tri = 0;
    if (i < n) {
        int stack[GD_STACK4];
        GdTrav T;
        gd_trav_begin(T, bvh, stack, org[3 * i], org[3 * i + 1], org[3 * i + 2], dir[3 * i], dir[3 * i + 1], dir[3 * i + 2], 0.0f,
                      GD_TINF, -2, -1, -1, -1, 0);
        int result = world_material;
        if (mode == 0) {
            while (T.node != GD_TRAV_DONE) {
                if (T.node >= 0) gd_trav_node4(T, bvh, stack, n_box);
                else { gd_trav_leaf(T, bvh, ~T.node, n_tri); T.node = gd_trav_pop(T, stack); }
            }
            if (T.orig != GD_NO_FACET) result = gd_mat_inside(T.fromto);     // low half = from-side material
        } else {
            // all hits: the window never shrinks; a facet reached through several of its references counts once
            int h_facet[GD_LOC_MAX_HITS], h_surf[GD_LOC_MAX_HITS], h_in[GD_LOC_MAX_HITS];
            float h_t[GD_LOC_MAX_HITS];
            int nh = 0;
            bool overflow = false;
            while (T.node != GD_TRAV_DONE) {
                if (T.node >= 0) { gd_trav_node4(T, bvh, stack, n_box); continue; }
                const int leaf = ~T.node;
                T.t = GD_TINF; T.orig = GD_NO_FACET;
                gd_trav_leaf(T, bvh, leaf, n_tri);
                if (T.orig != GD_NO_FACET) {
                    bool seen = false;
                    for (int k = 0; k < nh; ++k) seen = seen || h_facet[k] == T.orig;
                    if (!seen) {
                        if (nh < GD_LOC_MAX_HITS) {
                            const GdTri &tr = bvh.tris[leaf];
                            h_facet[nh] = T.orig; h_t[nh] = T.t;
                            h_surf[nh] = __float_as_int(tr.v2.w);
                            h_in[nh] = gd_mat_inside(__float_as_int(tr.v1.w));
                            nh++;
                        } else overflow = true;
                    }
                }
                T.t = GD_TINF; T.orig = GD_NO_FACET;
                T.node = gd_trav_pop(T, stack);
            }
            float best = GD_TINF;
            for (int a = 0; a < nh; ++a) {
                bool first_of_surface = true;
                for (int b = 0; b < a; ++b) first_of_surface = first_of_surface && h_surf[b] != h_surf[a];
                if (!first_of_surface) continue;
                int count = 0;
                float first = GD_TINF;
                for (int b = a; b < nh; ++b)
                    if (h_surf[b] == h_surf[a]) { count++; first = fminf(first, h_t[b]); }
                if ((count & 1) && first < best) { best = first; result = h_in[a]; }
            }
            if (overflow) result = GD_LOC_OVERFLOW;
        }
        mat_out[i] = result;
    }
    GdLocalCounters cnt = {};
    cnt.n_queries = i < n ? 1u : 0u; cnt.n_box_tests = n_box; cnt.n_tri_tests = n_tri;
    gd_flush_counters(cnt, counters, 0);
}
