// gadep_transport_kernels.cuh -- the history-per-thread transport kernels (cross-check and measurement modes).
// source, localisation, free flight, BVH nearest hit, boundary crossing,
// interactions, tally into a per-block shared-memory spectrum, flush to 64-bit global tallies.
#pragma once
#include "gadep_physics.cuh"

#define GD_RUN_THREADS 256

struct GdTally {                       // device-global, 64-bit
    unsigned long long *spectrum;      // [n_bins + 1]
    unsigned long long *emitted;       // [GD_MAX_LINES]
    unsigned long long *peak;          // [GD_MAX_LINES]
    GdCounters *counters;
    int n_bins;
    float inv_de;                      // n_bins / e_max
};

GD_D void gd_flush_counters(const GdLocalCounters &c, GdCounters *g, unsigned n_hist) {
    unsigned v[12] = {n_hist, c.n_queries, c.n_box_tests, c.n_tri_tests, c.n_crossings, c.n_pe, c.n_compton,
                      c.n_coherent, c.n_pair, c.n_escaped, c.n_leak, c.n_cutoff};
    unsigned long long *dst = (unsigned long long *)g;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        unsigned long long x = v[k];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
        if ((threadIdx.x & 31) == 0 && x) atomicAdd(&dst[k], x);
    }
}

// dynamic shared memory: [table floats][spectrum u32 (n_bins+1)]
// PARITY: material after the start and after every crossing from the paper's parity rule
// ELECTRON: deposits as straight electron segments (R16)
template <bool PARITY, bool PARTIAL, bool ELECTRON = false>
__global__ void __launch_bounds__(GD_RUN_THREADS)
gd_k_transport(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
               unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
               unsigned *__restrict__ flags_out) {
    extern __shared__ __align__(16) unsigned char gd_smem[];
    __shared__ GdSource s_src;
    __shared__ unsigned s_emitted[GD_MAX_LINES], s_peak[GD_MAX_LINES];
    const int n_tab = M.n_mat * 4 * M.n_grid;
    float *s_tab = (float *)gd_smem;
    unsigned *s_spec = (unsigned *)(s_tab + n_tab);
    for (int i = threadIdx.x; i < n_tab; i += blockDim.x) s_tab[i] = M.table[i];
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) s_spec[i] = 0;
    for (int i = threadIdx.x; i < (int)(sizeof(GdSource) / 4); i += blockDim.x) ((int *)&s_src)[i] = ((const int *)src)[i];
    if (threadIdx.x < GD_MAX_LINES) { s_emitted[threadIdx.x] = 0; s_peak[threadIdx.x] = 0; }
    __syncthreads();

    GdLocalCounters cnt = {};
    unsigned n_done = 0, n_parity = 0, n_mismatch = 0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long h = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; h < n_hist; h += stride) {
        GdHistory r;
        gd_run_history_t<PARITY, PARTIAL, ELECTRON>(bvh, M, s_tab, s_src, seed, first + h, r, cnt, n_parity, n_mismatch);
        n_done++;
        atomicAdd(&s_emitted[r.line], 1u);
        if (r.flags & GD_F_PEAK) {
            atomicAdd(&s_peak[r.line], 1u);
            atomicAdd(&s_spec[min(s_src.line_bin[r.line], tally.n_bins)], 1u);
        } else if (r.edep > 0.0f) {
            float b = floorf(r.edep * tally.inv_de);
            int bin = b >= (float)tally.n_bins ? tally.n_bins : (int)b;
            atomicAdd(&s_spec[bin], 1u);
        }
        if (edep_out) edep_out[h] = r.edep;
        if (flags_out) flags_out[h] = r.flags;
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) {
        unsigned v = s_spec[i];
        if (v) atomicAdd(&tally.spectrum[i], (unsigned long long)v);
    }
    if (threadIdx.x < GD_MAX_LINES) {
        if (s_emitted[threadIdx.x]) atomicAdd(&tally.emitted[threadIdx.x], (unsigned long long)s_emitted[threadIdx.x]);
        if (s_peak[threadIdx.x]) atomicAdd(&tally.peak[threadIdx.x], (unsigned long long)s_peak[threadIdx.x]);
    }
    gd_flush_counters(cnt, tally.counters, n_done);
    if (PARITY) {
        if (n_parity) atomicAdd(&tally.counters->n_parity, (unsigned long long)n_parity);
        if (n_mismatch) atomicAdd(&tally.counters->n_parity_mismatch, (unsigned long long)n_mismatch);
    }
}

// ---------------------------------------------------------------- v1: persistent lanes with refill
// Every lane owns one live history; when it ends the lane takes the next history index from its warp's chunk
// (chunks come from one global counter), so no lane idles while a neighbour finishes a long history.  Each loop
// iteration issues exactly one nearest-hit query per live lane (start localisation or flight), which keeps the
// warp together in the BVH traversal -- the expensive part.  Results are independent of this scheduling because
// the random streams are keyed by the history index and the tallies are integers.
__global__ void __launch_bounds__(GD_RUN_THREADS)
gd_k_transport_refill(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
                      unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
                      unsigned *__restrict__ flags_out, unsigned long long *next_history, unsigned chunk) {
    extern __shared__ __align__(16) unsigned char gd_smem[];
    __shared__ GdSource s_src;
    __shared__ unsigned s_emitted[GD_MAX_LINES], s_peak[GD_MAX_LINES];
    const int n_tab = M.n_mat * 4 * M.n_grid;
    float *s_tab = (float *)gd_smem;
    unsigned *s_spec = (unsigned *)(s_tab + n_tab);
    for (int i = threadIdx.x; i < n_tab; i += blockDim.x) s_tab[i] = M.table[i];
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) s_spec[i] = 0;
    for (int i = threadIdx.x; i < (int)(sizeof(GdSource) / 4); i += blockDim.x) ((int *)&s_src)[i] = ((const int *)src)[i];
    if (threadIdx.x < GD_MAX_LINES) { s_emitted[threadIdx.x] = 0; s_peak[threadIdx.x] = 0; }
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    GdLocalCounters cnt = {};
    unsigned n_done = 0;
    unsigned long long w_cur = 0, w_end = 0;     // warp-uniform chunk of history indices [w_cur, w_end)
    GdLane L;
    L.mode = GD_MODE_NEED;
    L.ex = gd_no_exclude();
    for (;;) {
        // ---- refill
        unsigned need_mask = __ballot_sync(0xFFFFFFFFu, L.mode == GD_MODE_NEED);
        if (need_mask) {
            unsigned n_need = __popc(need_mask);
            unsigned long long new_base = 0;
            bool refill = w_cur + n_need > w_end;
            if (refill) {
                if (lane == 0) new_base = atomicAdd(next_history, (unsigned long long)chunk);
                new_base = __shfl_sync(0xFFFFFFFFu, new_base, 0);
            }
            if (L.mode == GD_MODE_NEED) {
                unsigned long long h = w_cur + __popc(need_mask & lt_mask);
                if (h >= w_end) h = new_base + (h - w_end);
                if (h < n_hist) gd_lane_start(L, s_src, seed, first + h);
                else L.mode = GD_MODE_DONE;
            }
            if (refill) { w_cur = new_base + (w_cur + n_need - w_end); w_end = new_base + chunk; }
            else w_cur += n_need;
        }
        if (__all_sync(0xFFFFFFFFu, L.mode == GD_MODE_DONE)) break;
        // ---- one query per live lane; the traversal is warp-synchronous
        const bool live = L.mode != GD_MODE_DONE;
        float t_min = 0.0f, t_max = 0.0f;
        int filter = -2;
        GdRay ray;
        if (live) {
            gd_lane_query(L, M, s_tab, t_min, t_max, filter);
            gd_ray_setup(ray, L.pos, L.dir);
            cnt.n_queries++;
        } else {
            gd_ray_setup(ray, gd_make(0.f, 0.f, 0.f), gd_make(0.f, 0.f, 1.f));
        }
        GdHit hit;
        gd_nearest_hit<true>(bvh, ray, t_min, t_max, filter, L.ex, live, hit, cnt.n_box_tests, cnt.n_tri_tests);
        if (live) {
            GdHistory r;
            if (gd_lane_post(L, M, s_tab, s_src, seed, hit, r, cnt)) {
                n_done++;
                atomicAdd(&s_emitted[r.line], 1u);
                if (r.flags & GD_F_PEAK) {
                    atomicAdd(&s_peak[r.line], 1u);
                    atomicAdd(&s_spec[min(s_src.line_bin[r.line], tally.n_bins)], 1u);
                } else if (r.edep > 0.0f) {
                    float b = floorf(r.edep * tally.inv_de);
                    int bin = b >= (float)tally.n_bins ? tally.n_bins : (int)b;
                    atomicAdd(&s_spec[bin], 1u);
                }
                unsigned long long hrel = L.history - first;
                if (edep_out) edep_out[hrel] = r.edep;
                if (flags_out) flags_out[hrel] = r.flags;
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) {
        unsigned v = s_spec[i];
        if (v) atomicAdd(&tally.spectrum[i], (unsigned long long)v);
    }
    if (threadIdx.x < GD_MAX_LINES) {
        if (s_emitted[threadIdx.x]) atomicAdd(&tally.emitted[threadIdx.x], (unsigned long long)s_emitted[threadIdx.x]);
        if (s_peak[threadIdx.x]) atomicAdd(&tally.peak[threadIdx.x], (unsigned long long)s_peak[threadIdx.x]);
    }
    gd_flush_counters(cnt, tally.counters, n_done);
}
