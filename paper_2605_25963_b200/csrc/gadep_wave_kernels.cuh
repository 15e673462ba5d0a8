// gadep_wave_kernels.cuh -- warp-resident wavefront transport and the ray-cast hook.
//
// Every warp owns GD_W_SLOTS photon slots in shared memory (SoA, GD_W_NF words per slot).  A slot is in one of
// three places: the READY queue (its next nearest-hit query is prepared), in flight on a lane (GdTrav registers),
// or the RESULT queue (hit known, physics pending).  The warp alternates
//   T-burst: lanes traverse in rounds of `n_steps` 4-wide node visits + one leaf step; a lane whose ray ends writes
//            the hit to its slot, pushes it to RESULT and -- as soon as `k_fetch` lanes are idle -- takes a READY slot
//            (dynamic fetch).  The burst ends when READY is empty and 32 results wait (or `k_exit` times as many
//            results as rays still in flight: sparse warps batch their few chains); unfinished rays stay in their
//            lanes' registers across the physics burst.
//   P-burst: lanes take RESULT slots and process one event each (boundary crossing / interaction / tally / refill
//            from the history counter / attenuation lookup); a slot whose next flight ends before the clearance of
//            its grid cell (GdGrid) stays on its lane and goes round again without a query, the others are pushed to
//            READY and their lanes take the next waiting result.  Both queues are rings (first in, first out).
// There is no block-level barrier inside the loop and no particle state in global memory (only the two pending
// annihilation photons of a pair event, which are rare, sit in a global side buffer).  Results do not depend on any
// of this scheduling: random streams are keyed by the history index and the tallies are integers.
#pragma once
#include "gadep_physics.cuh"
#include "gadep_trav.cuh"
#include "gadep_transport_kernels.cuh"

#define GD_W_THREADS 512
#define GD_W_WARPS (GD_W_THREADS / 32)
#define GD_W_SLOTS 64
// fields per slot.  25 words keep the block's shared memory under the 164 KB carve-out for up to 9 materials, which
// leaves the SM a 64 KB L1 instead of 32 KB.
#define GD_W_NF 25

// Measurement build only (-DGD_PROF, never in the shipped library): per-warp clocks of the two bursts and lane counts.
#ifdef GD_PROF
__device__ unsigned long long gd_prof[16];
#define GD_PROF_ADD(k, v) do { pacc[k] += (unsigned long long)(v); } while (0)
#else
#define GD_PROF_ADD(k, v) do {} while (0)
#endif

// scheduling knobs (defaults in gadep_api.cu; GADEP_TUNE="k_fetch,k_exit,n_steps" overrides them for measurement
// sweeps).  None of them can change a result.
struct GdWaveTune {
    int k_fetch;        // idle lanes needed before READY slots are fetched
    int k_exit;         // T-burst ends when n_results >= k_exit * rays in flight (or 32 results) and READY is empty
    int n_steps;        // node visits per traversal round
    int p_min;          // a physics pass runs while this many lanes have work (or the warp has nothing else to do)
};

// ---- slot <-> registers
#define GD_SF(f) sl[(f) * GD_W_SLOTS + s]
GD_D unsigned gd_pack_state(const GdLane &L) {
    return (unsigned)(L.m + 1) | ((unsigned)L.mode << 5) | ((unsigned)L.line << 7) | ((unsigned)L.pending << 13) |
           ((unsigned)L.n_stall << 15) | (L.g.stream << 21) | ((unsigned)L.need_mu << 23);
}
GD_D void gd_slot_store(float *sl, int s, const GdLane &L, unsigned long long first) {
    GD_SF(0) = L.pos.x; GD_SF(1) = L.pos.y; GD_SF(2) = L.pos.z;
    GD_SF(3) = L.dir.x; GD_SF(4) = L.dir.y; GD_SF(5) = L.dir.z;
    GD_SF(6) = L.e; GD_SF(7) = L.tau;
    GD_SF(8) = L.mu[0]; GD_SF(9) = L.mu[1]; GD_SF(10) = L.mu[2]; GD_SF(11) = L.mu[3];
    GD_SF(12) = L.mu_tot; GD_SF(13) = L.sdist;
    GD_SF(14) = __uint_as_float(gd_pack_state(L));
    GD_SF(15) = __uint_as_float(L.g.draw);
    GD_SF(16) = __uint_as_float((unsigned)(L.history - first));
    GD_SF(17) = L.dep;
    GD_SF(18) = __uint_as_float((L.flags & 0xFFu) | ((L.n_events > 0xFFFFu ? 0xFFFFu : L.n_events) << 16));
    GD_SF(19) = __int_as_float(L.ex.a); GD_SF(20) = __int_as_float(L.ex.b); GD_SF(21) = __int_as_float(L.ex.c);
}
GD_D void gd_slot_load(const float *sl, int s, GdLane &L, unsigned long long seed, unsigned long long first) {
    L.pos = gd_make(GD_SF(0), GD_SF(1), GD_SF(2));
    L.dir = gd_make(GD_SF(3), GD_SF(4), GD_SF(5));
    L.e = GD_SF(6); L.tau = GD_SF(7);
    L.mu[0] = GD_SF(8); L.mu[1] = GD_SF(9); L.mu[2] = GD_SF(10); L.mu[3] = GD_SF(11);
    L.mu_tot = GD_SF(12); L.sdist = GD_SF(13);
    const unsigned st = __float_as_uint(GD_SF(14));
    L.m = (int)(st & 31u) - 1; L.mode = (int)((st >> 5) & 3u); L.line = (int)((st >> 7) & 63u);
    L.pending = (int)((st >> 13) & 3u); L.n_stall = (int)((st >> 15) & 63u); L.need_mu = (int)((st >> 23) & 1u);
    L.history = first + (unsigned long long)__float_as_uint(GD_SF(16));
    gd_rng_init(L.g, seed, L.history, (st >> 21) & 3u, __float_as_uint(GD_SF(15)));
    L.dep = GD_SF(17);
    const unsigned fe = __float_as_uint(GD_SF(18));
    L.flags = fe & 0xFFu; L.n_events = fe >> 16;
    L.ex.a = __float_as_int(GD_SF(19)); L.ex.b = __float_as_int(GD_SF(20)); L.ex.c = __float_as_int(GD_SF(21));
}

// O14 tally of the histories that ended in this batch, aggregated per warp: lanes that hit the same
// counter are found with __match_any_sync and their leader adds the group's size, so the five hot `emitted` words of
// a point-source run see one shared-memory atomic per line and batch instead of one per history.
// `fin` may differ from lane to lane; every lane of the warp must call.
GD_D void gd_tally_warp(bool fin, const GdHistory &r, const GdSource &S, const GdTally &tally, unsigned *s_spec,
                        unsigned *s_emitted, unsigned *s_peak, unsigned lane) {
    const unsigned fin_mask = __ballot_sync(0xFFFFFFFFu, fin);
    if (fin_mask == 0u) return;
    int bin = -1;                                     // spectrum bin of this lane's history, -1 = nothing to book
    const bool peak = fin && (r.flags & GD_F_PEAK);
    if (peak) bin = min(S.line_bin[r.line], tally.n_bins);
    else if (fin && r.edep > 0.0f) {
        const float b = floorf(r.edep * tally.inv_de);
        bin = b >= (float)tally.n_bins ? tally.n_bins : (int)b;
    }
    if (fin) {
        const unsigned same = __match_any_sync(fin_mask, r.line);
        if ((same & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_emitted[r.line], (unsigned)__popc(same));
    }
    const unsigned peak_mask = __ballot_sync(0xFFFFFFFFu, peak);
    if (peak) {
        const unsigned same = __match_any_sync(peak_mask, r.line);
        if ((same & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_peak[r.line], (unsigned)__popc(same));
    }
    const unsigned bin_mask = __ballot_sync(0xFFFFFFFFu, bin >= 0);
    if (bin >= 0) {
        const unsigned same = __match_any_sync(bin_mask, bin);
        if ((same & ((1u << lane) - 1u)) == 0u) atomicAdd(&s_spec[bin], (unsigned)__popc(same));
    }
}

// dynamic shared memory: [table floats][spectrum u32 (n_bins+1)][slots: warps x GD_W_NF x GD_W_SLOTS floats]
// pair_buf: global, 8 floats per slot of every warp of the grid
// WIDTH: 8 = compressed 8-wide nodes (default), 4 = uncompressed 4-wide nodes (cross-check variant)
template <int WIDTH>
__global__ void __launch_bounds__(GD_W_THREADS, 1)
gd_k_transport_wave(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
                    unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
                    unsigned *__restrict__ flags_out, unsigned long long *next_history, unsigned chunk,
                    float *__restrict__ pair_buf, GdWaveTune tune) {
    extern __shared__ __align__(16) unsigned char gd_smem[];
    __shared__ GdSource s_src;
    __shared__ unsigned s_emitted[GD_MAX_LINES], s_peak[GD_MAX_LINES];
    __shared__ unsigned s_cnt[12];
    __shared__ unsigned char s_qready[GD_W_WARPS][GD_W_SLOTS], s_qres[GD_W_WARPS][GD_W_SLOTS];
    const int n_tab = M.n_mat * 4 * M.n_grid;
    float *s_tab = (float *)gd_smem;
    unsigned *s_spec = (unsigned *)(s_tab + n_tab);
    float *s_slots = (float *)(s_spec + tally.n_bins + 1);
    for (int i = threadIdx.x; i < n_tab; i += blockDim.x) s_tab[i] = M.table[i];
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) s_spec[i] = 0;
    for (int i = threadIdx.x; i < (int)(sizeof(GdSource) / 4); i += blockDim.x) ((int *)&s_src)[i] = ((const int *)src)[i];
    if (threadIdx.x < GD_MAX_LINES) { s_emitted[threadIdx.x] = 0; s_peak[threadIdx.x] = 0; }
    if (threadIdx.x < 12) s_cnt[threadIdx.x] = 0;
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    float *sl = s_slots + (size_t)warp * GD_W_NF * GD_W_SLOTS;
    unsigned char *q_ready = s_qready[warp], *q_res = s_qres[warp];
    float *pair = pair_buf + ((size_t)blockIdx.x * GD_W_WARPS + warp) * GD_W_SLOTS * 8;
    int stack[WIDTH == 8 ? GD_STACK8 : GD_STACK4];
    GdTrav T;
    gd_trav_idle(T);
    unsigned n_box = 0, n_tri = 0, n_query = 0, n_done = 0, n_skip = 0;
    unsigned long long w_cur = 0, w_end = 0;     // warp-uniform chunk of history indices [w_cur, w_end)
    // every slot starts in RESULT with mode NEED: the first P-bursts start the first histories
    for (int s = lane; s < GD_W_SLOTS; s += 32) {
        GD_SF(14) = __uint_as_float((unsigned)GD_MODE_NEED << 5);
        q_res[s] = (unsigned char)s;
    }
    // both queues are rings (first in, first out): a slot of a long scattering chain is served every round instead of
    // waiting at the bottom of a stack while fresh histories stream over it -- the chains are the critical path
    int n_res = GD_W_SLOTS, n_ready = 0, h_res = 0, h_ready = 0;
    static_assert((GD_W_SLOTS & (GD_W_SLOTS - 1)) == 0, "slot count must be a power of two");
#ifdef GD_PROF
    unsigned long long pacc[16] = {};
    long long p_t0 = clock64();
#endif
    __syncwarp();

    for (;;) {
        // ================================================================ P-burst
        // Lanes take waiting results, run the physics of one event each, and either hand the slot to READY (the next
        // flight needs the BVH) or -- when the clearance grid says that no facet lies within the next flight -- keep
        // it and go round again: the answer of that query is known ("none").  Lanes that gave their slot away take the
        // next waiting result.  The burst goes on while at least `p_min` lanes have work, or while the warp has
        // nothing else to do; what is left then is parked in RESULT with its known answer.
        {
            bool has = false;
            int s = 0;
            GdLane L;
            L.mode = GD_MODE_DONE;
            GdHit hit;
            hit.t = 0.0f; hit.leaf = -1; hit.orig = GD_NO_FACET; hit.leaving = 1; hit.mats = 0;
            const bool no_rays = __ballot_sync(0xFFFFFFFFu, T.slot >= 0) == 0u;
            for (bool first_pass = true;; first_pass = false) {
                // ---- fetch
                const unsigned free_mask = __ballot_sync(0xFFFFFFFFu, !has);
                const int n_free = __popc(free_mask), n_has = 32 - n_free;
                const int take = n_free < n_res ? n_free : n_res;
                // the first pass takes whatever made the traversal burst end; later passes need p_min lanes with work,
                // unless the warp has no ray in flight and none prepared
                if (!(n_has + take > 0 && (first_pass || n_has + take >= tune.p_min || (no_rays && n_ready == 0)))) {
                    // not worth a pass: park the lanes that still hold a slot (their query is answered: no facet)
                    if (has) {
                        gd_slot_store(sl, s, L, first);
                        GD_SF(22) = L.sdist; GD_SF(23) = __int_as_float(GD_NO_FACET); GD_SF(24) = 0.0f;
                        q_res[(h_res + n_res + __popc(~free_mask & lt_mask)) & (GD_W_SLOTS - 1)] = (unsigned char)s;
                    }
                    n_res += n_has;
                    __syncwarp();
                    break;
                }
                if (take > 0) {
                    const int rank = __popc(free_mask & lt_mask);
                    if (!has && rank < take) {
                        s = (int)q_res[(h_res + rank) & (GD_W_SLOTS - 1)];
                        gd_slot_load(sl, s, L, seed, first);
                        if (L.pending) {
                            const float *p = pair + s * 8;
                            L.p_pos = gd_make(p[0], p[1], p[2]); L.p_axis = gd_make(p[3], p[4], p[5]); L.p_m = __float_as_int(p[6]);
                        }
                        // gd_lane_post reads the from-side id as "inside if leaving else outside" in LOCATE mode and the
                        // to-side id as "outside if leaving else inside" in FLIGHT mode: present (from, to) that way
                        hit.t = GD_SF(22);
                        hit.orig = __float_as_int(GD_SF(23));
                        hit.leaf = hit.orig == GD_NO_FACET ? -1 : 0;
                        hit.mats = __float_as_int(GD_SF(24));          // inside := from, outside := to
                        has = true;
                    }
                    h_res = (h_res + take) & (GD_W_SLOTS - 1); n_res -= take;
                }
                GD_PROF_ADD(2, 1); GD_PROF_ADD(3, __popc(__ballot_sync(0xFFFFFFFFu, has)));
                // ---- one event per lane
                GdLocalCounters cnt = {};
                GdHistory r;
                r.edep = 0.0f; r.flags = 0u; r.line = 0;
                bool fin = false;
                if (has && L.mode != GD_MODE_NEED) {
                    const int was_pending = L.pending;
                    fin = gd_lane_post(L, M, s_tab, s_src, seed, hit, r, cnt);
                    if (fin) {
                        n_done++;
                        const unsigned long long hrel = L.history - first;
                        if (edep_out) edep_out[hrel] = r.edep;
                        if (flags_out) flags_out[hrel] = r.flags;
                    } else if (L.pending && !was_pending) {  // a pair event: park the two annihilation photons
                        float *p = pair + s * 8;
                        p[0] = L.p_pos.x; p[1] = L.p_pos.y; p[2] = L.p_pos.z;
                        p[3] = L.p_axis.x; p[4] = L.p_axis.y; p[5] = L.p_axis.z; p[6] = __int_as_float(L.p_m);
                    }
                }
                gd_tally_warp(fin, r, s_src, tally, s_spec, s_emitted, s_peak, lane);
                {   // event counters, one shared-memory atomic per kind and pass (crossing / PE / Compton / coherent /
                    // pair; escapes, re-localisations and cut-offs can accompany any of them)
                    const unsigned v[8] = {cnt.n_crossings, cnt.n_pe, cnt.n_compton, cnt.n_coherent, cnt.n_pair, cnt.n_escaped,
                                           cnt.n_leak, cnt.n_cutoff};
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const unsigned mk = __ballot_sync(0xFFFFFFFFu, v[k] != 0u);
                        if (mk && lane == 0) atomicAdd(&s_cnt[4 + k], (unsigned)__popc(mk));
                    }
                }
                // ---- refill finished slots from the history counter (warp-level chunks)
                const unsigned need_mask = __ballot_sync(0xFFFFFFFFu, has && L.mode == GD_MODE_NEED);
                if (need_mask) {
                    const unsigned n_need = __popc(need_mask);
                    unsigned long long new_base = 0;
                    const bool refill = w_cur + n_need > w_end;
                    unsigned my_chunk = chunk;
                    if (refill) {
                        // guided: towards the end of the launch the chunks shrink with what is left, so that the last
                        // histories spread over all warps instead of going to the few that ask last
                        if (lane == 0) {
                            const unsigned long long cur = *(volatile unsigned long long *)next_history;
                            const unsigned long long rem = cur < n_hist ? n_hist - cur : 0ull;
                            const unsigned long long g = rem / ((unsigned long long)gridDim.x * GD_W_WARPS * 2ull);
                            if (g < my_chunk) my_chunk = g < 32ull ? 32u : (unsigned)g;
                            new_base = atomicAdd(next_history, (unsigned long long)my_chunk);
                        }
                        new_base = __shfl_sync(0xFFFFFFFFu, new_base, 0);
                        my_chunk = __shfl_sync(0xFFFFFFFFu, my_chunk, 0);
                    }
                    if (has && L.mode == GD_MODE_NEED) {
                        unsigned long long h = w_cur + __popc(need_mask & lt_mask);
                        if (h >= w_end) h = new_base + (h - w_end);
                        if (h < n_hist) gd_lane_start(L, s_src, seed, first + h);
                        else L.mode = GD_MODE_DONE;
                    }
                    if (refill) { w_cur = new_base + (w_cur + n_need - w_end); w_end = new_base + my_chunk; }
                    else w_cur += n_need;
                }
                // ---- the next query: answered by the clearance grid, or handed to READY
                const bool live = has && L.mode != GD_MODE_DONE;
                bool skip = false;
                if (live) {
                    float t_min, t_max;
                    int filter;
                    gd_lane_query(L, M, s_tab, t_min, t_max, filter);
                    if (L.mode == GD_MODE_FLIGHT && L.sdist < GD_INF)
                        skip = fmaf(L.sdist, 1.0001f, 4.0f * GD_TBACK) < gd_clearance(bvh.grid, L.pos);
                }
                const unsigned ready_mask = __ballot_sync(0xFFFFFFFFu, live && !skip);
                if (live && !skip) {
                    gd_slot_store(sl, s, L, first);
                    q_ready[(h_ready + n_ready + __popc(ready_mask & lt_mask)) & (GD_W_SLOTS - 1)] = (unsigned char)s;
                }
                n_ready += __popc(ready_mask);
                has = skip;
                if (skip) { n_skip++; hit.t = L.sdist; hit.leaf = -1; hit.orig = GD_NO_FACET; hit.mats = 0; }
                __syncwarp();
            }
        }
#ifdef GD_PROF
        { const long long t1 = clock64(); GD_PROF_ADD(0, t1 - p_t0); p_t0 = t1; }
#endif
        const unsigned busy_mask = __ballot_sync(0xFFFFFFFFu, T.slot >= 0);
        if (n_ready == 0 && busy_mask == 0u) {
            if (n_res == 0) break;                           // every slot is dead
            continue;
        }
        // ================================================================ T-burst
        for (;;) {
            const unsigned idle_mask = __ballot_sync(0xFFFFFFFFu, T.slot < 0);
            const int n_idle = __popc(idle_mask);
            if (n_idle) {
                if (n_ready > 0) {
                    if (n_idle >= tune.k_fetch || n_idle == 32) {
                        const int rank = __popc(idle_mask & lt_mask);
                        if (T.slot < 0 && rank < n_ready) {
                            const int s = (int)q_ready[(h_ready + rank) & (GD_W_SLOTS - 1)];
                            const unsigned st = __float_as_uint(GD_SF(14));
                            const bool loc = (int)((st >> 5) & 3u) == GD_MODE_LOCATE;
                            gd_trav_begin(T, bvh, stack, GD_SF(0), GD_SF(1), GD_SF(2), GD_SF(3), GD_SF(4), GD_SF(5),
                                          loc ? 0.0f : -GD_TBACK, loc ? GD_INF : GD_SF(13), loc ? -2 : (int)(st & 31u) - 1,
                                          __float_as_int(GD_SF(19)), __float_as_int(GD_SF(20)), __float_as_int(GD_SF(21)), s);
                            n_query++;
                        }
                        const int tk = n_idle < n_ready ? n_idle : n_ready;
                        h_ready = (h_ready + tk) & (GD_W_SLOTS - 1); n_ready -= tk;
                    }
                } else if ((n_res > 0 && (n_res >= 32 || n_res >= tune.k_exit * (32 - n_idle))) || n_idle == 32) {
                    break;
                }
            }
            GD_PROF_ADD(4, 1); GD_PROF_ADD(5, __popc(__ballot_sync(0xFFFFFFFFu, T.slot >= 0 && T.node >= 0)));
            GD_PROF_ADD(6, __popc(__ballot_sync(0xFFFFFFFFu, T.slot >= 0)));
            gd_trav_step<WIDTH>(T, bvh, stack, tune.n_steps, n_box, n_tri);
            const bool fin = T.slot >= 0 && T.node == GD_TRAV_DONE;
            const unsigned fin_mask = __ballot_sync(0xFFFFFFFFu, fin);
            if (fin_mask) {
                if (fin) {
                    const int s = T.slot;
                    GD_SF(22) = T.t; GD_SF(23) = __int_as_float(T.orig); GD_SF(24) = __int_as_float(T.fromto);
                    q_res[(h_res + n_res + __popc(fin_mask & lt_mask)) & (GD_W_SLOTS - 1)] = (unsigned char)s;
                    T.slot = -1;
                }
                n_res += __popc(fin_mask);
                __syncwarp();
            }
        }
#ifdef GD_PROF
        { const long long t1 = clock64(); GD_PROF_ADD(1, t1 - p_t0); p_t0 = t1; }
#endif
    }
#ifdef GD_PROF
    if (lane == 0) for (int k = 0; k < 16; ++k) if (pacc[k]) atomicAdd(&gd_prof[k], pacc[k]);
#endif
    // ---- flush: per-lane 32-bit work counters straight to the 64-bit global totals
    {
        const unsigned v[5] = {n_done, n_query, n_box, n_tri, n_skip};
        const int where[5] = {0, 1, 2, 3, 13};           // GdCounters: n_histories, n_queries, n_box_tests, n_tri_tests, n_skipped
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            unsigned long long x = v[k];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
            if (lane == 0 && x) atomicAdd(&((unsigned long long *)tally.counters)[where[k]], x);
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
    if (threadIdx.x >= 4 && threadIdx.x < 12 && s_cnt[threadIdx.x])
        atomicAdd(&((unsigned long long *)tally.counters)[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
}

// ---------------------------------------------------------------- ray-cast hook with dynamic fetch
// Persistent warps take chunks of ray indices from one global counter; a lane whose ray ends stores the result and
// takes the next ray of its warp's chunk once `k_fetch` lanes are idle.
template <int WIDTH>
__global__ void __launch_bounds__(256, 4)
gd_k_trace_wave(GdBvh bvh, const float *__restrict__ org, const float *__restrict__ dir, long long n, int filter_mat,
                float t_min, int *__restrict__ tri_out, float *__restrict__ t_out, GdCounters *counters,
                unsigned long long *next_ray, unsigned chunk, GdWaveTune tune) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    int stack[WIDTH == 8 ? GD_STACK8 : GD_STACK4];
    GdTrav T;
    gd_trav_idle(T);
    long long my_ray = -1;
    unsigned n_box = 0, n_tri = 0, n_query = 0;
    long long w_cur = 0, w_end = 0;
    bool dry = false;                 // the global counter ran past n
    for (;;) {
        const unsigned idle_mask = __ballot_sync(0xFFFFFFFFu, T.slot < 0);
        const int n_idle = __popc(idle_mask);
        if (n_idle) {
            if (w_cur >= w_end && !dry) {
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(next_ray, (unsigned long long)chunk);
                base = __shfl_sync(0xFFFFFFFFu, base, 0);
                w_cur = (long long)base;
                w_end = w_cur + chunk < n ? w_cur + chunk : n;
                if (w_cur >= n) { dry = true; w_cur = w_end = 0; }
            }
            const long long avail = w_end - w_cur;
            if (avail > 0) {
                if (n_idle >= tune.k_fetch || n_idle == 32) {
                    const int rank = __popc(idle_mask & lt_mask);
                    if (T.slot < 0 && rank < avail) {
                        const long long i = w_cur + rank;
                        my_ray = i;
                        gd_trav_begin(T, bvh, stack, org[3 * i], org[3 * i + 1], org[3 * i + 2], dir[3 * i], dir[3 * i + 1],
                                      dir[3 * i + 2], t_min, GD_INF, filter_mat, -1, -1, -1, 0);
                        n_query++;
                    }
                    w_cur += n_idle < avail ? n_idle : avail;
                }
            } else if (n_idle == 32) {
                break;
            }
        }
        gd_trav_step<WIDTH>(T, bvh, stack, tune.n_steps, n_box, n_tri);
        if (T.slot >= 0 && T.node == GD_TRAV_DONE) {
            tri_out[my_ray] = T.orig == GD_NO_FACET ? -1 : T.orig;
            t_out[my_ray] = T.orig == GD_NO_FACET ? GD_INF : T.t;
            T.slot = -1;
        }
    }
    GdLocalCounters cnt = {};
    cnt.n_queries = n_query; cnt.n_box_tests = n_box; cnt.n_tri_tests = n_tri;
    gd_flush_counters(cnt, counters, 0);
}
