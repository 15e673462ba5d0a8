// gadep_wave_kernels.cuh -- block-resident wavefront transport and the ray-cast hook.
//
// A block owns GD_W_NSLOT photon slots in shared memory (SoA, GD_W_NF words per slot) and three block-wide queues of
// slot numbers: READY (the slot's next nearest-hit query is prepared), RESULT (hit known; the event is a boundary
// crossing into another medium or an interaction) and SLOW (any other event: start of a history, start localisation,
// escape, crossing into KILL).  A slot is in one queue, or on a lane of some warp.  Every warp of the block does
// whichever kind of work there is:
//   T-burst:      lanes traverse in rounds of `n_steps` node visits + one leaf step; a lane whose ray ends writes the hit
//                 to its slot, pushes it to RESULT or SLOW and -- as soon as `k_fetch` lanes are idle -- takes a READY
//                 slot (dynamic fetch).  Unfinished rays stay in their lanes' registers while the warp does physics.
//   chain burst:  lanes take RESULT slots and handle crossings and coherent scattering in place; a slot whose next
//                 flight provably meets no facet (clearance grid: scalar bound of its cell, or the distances to the
//                 planes of the cell's list) stays on its lane and goes round again without a query; photoelectric,
//                 Compton and pair events go to SLOW, flights that need the BVH to READY.
//   general pass: lanes take SLOW slots and process one event each (any kind), tally finished histories, start the next
//                 histories of the block's chunk and prepare their first query.
// Because the queues are shared, a warp finds 32 slots for either kind of work as long as the block has them -- the
// long scattering chains that are left when the history counter runs dry end up on the lanes of one warp instead of
// idling in all of them.  The queues are rings with a ticket counter on each side; an entry carries a valid bit that its
// producer sets last and its consumer clears, so no lock is held while a slot is read or written.
// There is no block-level barrier inside the loop and no particle state in global memory (only the two pending
// annihilation photons of a pair event, which are rare, sit in a global side buffer).  Results do not depend on any
// of this scheduling: random streams are keyed by the history index and the tallies are integers.
// The kernel is bound by instruction fetch as much as by anything else: code that several call
// sites share is written once (one push routine for all queues, out-of-line Philox / rotation / attenuation lookup).
#pragma once
#include "gadep_physics.cuh"
#include "gadep_trav.cuh"
#include "gadep_transport_kernels.cuh"

#define GD_W_THREADS 384           // 12 warps x 160 registers: the default
#define GD_W_THREADS_LAT 896       // 28 warps x 72 registers (540 bytes of spills): for hierarchies far larger than the L2,
                                   // where the kernel waits for node fetches from HBM and rays in flight are what pays.
                                   // Config 4, 1e8 histories: 1727 ms at 12 warps, 1515 at 16, 1408 at 20, 1318 at 24,
                                   // 1262 at 28, 1430 at 32; the cache-resident configs lose 2 - 4 % already at 16.
#define GD_W_NSLOT 1024           // photon slots per block
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
    int t_keep;         // a warp stays in its T-burst while at least this many of its lanes hold a ray (or READY has more)
    int n_steps;        // node visits per traversal round (lower bound of the adaptive length)
    int n_steps_max;    // ... and its upper bound; equal to n_steps = fixed length
    int p_min;          // a physics pass runs while this many lanes have work (or the warp has nothing else to do)
    int t_help;         // READY slots that must wait before the warps that do not prefer traversal fetch any
    int k_claim;        // chain burst: free lanes needed before the queues are consulted and waiting results claimed
};

// Ordering between a slot's words and the queue entry that publishes it: an acquire-release fence at block scope
// (lighter than the sequentially consistent __threadfence_block()).
#ifndef GD_FENCE_MODE
#define GD_FENCE_MODE 1
#endif
#if GD_FENCE_MODE == 0
#define GD_FENCE_BLOCK() __threadfence_block()
#elif GD_FENCE_MODE == 1
#define GD_FENCE_BLOCK() asm volatile("fence.acq_rel.cta;" ::: "memory")
#else
#define GD_FENCE_BLOCK() asm volatile("" ::: "memory")
#endif

// ---- block-wide queue of slot numbers (multi-producer, multi-consumer, warp-granular).  Tickets count up for ever;
// ticket k lives in entry k mod GD_W_NSLOT and carries the lap number (k / GD_W_NSLOT) mod 32 beside the valid bit, so
// a consumer can tell the entry it waits for from the previous lap's entry that its owner has not emptied yet.
#define GD_Q_READY 0
#define GD_Q_RESULT 1
#define GD_Q_SLOW 2
struct GdQueue {
    unsigned head, tail;                      // consumers have claimed tickets < head, producers hold tickets < tail
    unsigned short ent[GD_W_NSLOT];           // 0 = empty, else 0x8000 | lap << 10 | slot
};
GD_D unsigned gd_q_tag(unsigned ticket) { return 0x8000u | (((ticket / GD_W_NSLOT) & 31u) << 10); }
GD_D int gd_q_count(const GdQueue *q) {
    const unsigned h = *(volatile const unsigned *)&q->head, t = *(volatile const unsigned *)&q->tail;
    return (int)(t - h);
}
// every lane with dest >= 0 (0 .. 2) appends its slot to queue q0[dest]; the slot's words must have been written by the
// same lane before the call.  One copy of the push code serves all destinations (the kernel is bound by instruction
// fetch); grouping the lanes with __match_any_sync instead of one ballot per queue measured 5 % slower.
GD_D void gd_q_push_to(GdQueue *q0, int dest, int slot, unsigned lane) {
#pragma unroll 1
    for (int k = 0; k < 3; ++k) {
        const unsigned mask = __ballot_sync(0xFFFFFFFFu, dest == k);
        if (mask == 0u) continue;
        GdQueue *q = q0 + k;
        unsigned base = 0;
        const int leader = __ffs(mask) - 1;
        if ((int)lane == leader) base = atomicAdd(&q->tail, (unsigned)__popc(mask));
        base = __shfl_sync(0xFFFFFFFFu, base, leader);
        if (dest == k) {
            const unsigned ticket = base + __popc(mask & ((1u << lane) - 1u));
            volatile unsigned short *e = &q->ent[ticket & (GD_W_NSLOT - 1)];
            while (*e != 0) {}               // the consumer of the previous lap has claimed this entry but not yet emptied it
            GD_FENCE_BLOCK();                // slot words before the valid bit
            *e = (unsigned short)(gd_q_tag(ticket) | (unsigned)slot);
        }
    }
}
// up to `want` entries for the lanes with `free` set (lowest lanes first); returns how many were claimed (warp-uniform)
// and sets slot for the lanes that got one (got = true)
GD_D int gd_q_claim(GdQueue *q, bool free, int want, unsigned lane, int &slot, bool &got) {
    const unsigned mask = __ballot_sync(0xFFFFFFFFu, free);
    got = false;
    if (mask == 0u || want <= 0) return 0;
    unsigned base = 0;
    int n = 0;
    if (lane == 0) {
        for (;;) {
            const unsigned h = *(volatile unsigned *)&q->head, t = *(volatile unsigned *)&q->tail;
            const int avail = (int)(t - h);
            n = avail < want ? avail : want;
            if (n <= 0) { n = 0; break; }
            if (atomicCAS(&q->head, h, h + (unsigned)n) == h) { base = h; break; }
        }
    }
    n = __shfl_sync(0xFFFFFFFFu, n, 0);
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    const int rank = __popc(mask & ((1u << lane) - 1u));
    if (free && rank < n) {
        const unsigned ticket = base + (unsigned)rank, tag = gd_q_tag(ticket);
        volatile unsigned short *e = &q->ent[ticket & (GD_W_NSLOT - 1)];
        unsigned v;
        while (((v = *e) & 0xFC00u) != tag) {}   // the producer holds the ticket but has not written the entry yet
        *e = 0;
        GD_FENCE_BLOCK();                    // valid bit before the slot words
        slot = (int)(v & 0x3FFu);
        got = true;
    }
    return n;
}

// ---- history indices for the block: one chunk [cur, end) of the launch's global counter, packed in a 64-bit shared
// word (indices relative to the launch's first history, < 2^32).  Requests are served by compare-and-swap on that word;
// the warp that finds the chunk too short takes the lock, fetches the next chunk and hands out the old chunk's rest
// together with the head of the new one, so no index is ever dropped.
struct GdHistPool {
    unsigned long long state;                 // cur | end << 32
    unsigned lock, dry;                       // dry: the global counter has passed n_hist
};
// n <= 32 indices for the calling warp (lane 0 works, the result is broadcast): lane of rank r gets a0 + r for r < n0,
// else a1 + (r - n0); an index >= n_hist means "no history left"
GD_D void gd_hist_take(GdHistPool *hp, unsigned n, unsigned long long *next_history, unsigned long long n_hist,
                       unsigned chunk, unsigned n_blocks, unsigned lane, unsigned &a0, unsigned &n0, unsigned &a1) {
    unsigned r0 = 0, rn0 = 0, r1 = 0;
    if (lane == 0) {
        const unsigned nh = (unsigned)n_hist;
        for (;;) {
            const unsigned long long st = *(volatile unsigned long long *)&hp->state;
            const unsigned cur = (unsigned)st, end = (unsigned)(st >> 32);
            if (end - cur >= n) {                                            // enough left in the chunk
                if (atomicCAS(&hp->state, st, (unsigned long long)(cur + n) | ((unsigned long long)end << 32)) == st) {
                    r0 = cur; rn0 = n; r1 = nh; break;
                }
                continue;
            }
            if (*(volatile unsigned *)&hp->dry) {                            // hand out what is left, then nothing
                if (atomicCAS(&hp->state, st, (unsigned long long)end | ((unsigned long long)end << 32)) == st) {
                    r0 = cur; rn0 = end - cur; r1 = nh; break;
                }
                continue;
            }
            if (atomicCAS(&hp->lock, 0u, 1u) != 0u) continue;                // another warp is fetching a chunk
            const unsigned long long s1 = *(volatile unsigned long long *)&hp->state;
            if ((unsigned)(s1 >> 32) - (unsigned)s1 >= n || *(volatile unsigned *)&hp->dry) {   // refilled meanwhile
                atomicExch(&hp->lock, 0u);
                continue;
            }
            // guided: towards the end of the launch the chunks shrink with what is left, so that the last histories
            // spread over all blocks instead of going to the few that ask last
            const unsigned long long seen = *(volatile unsigned long long *)next_history;
            const unsigned long long rem = seen < n_hist ? n_hist - seen : 0ull;
            const unsigned long long gsz = rem / ((unsigned long long)n_blocks * 2ull);
            unsigned my_chunk = chunk;
            if (gsz < my_chunk) my_chunk = gsz < 256ull ? 256u : (unsigned)gsz;
            const unsigned long long g = atomicAdd(next_history, (unsigned long long)my_chunk);
            const unsigned g0 = g >= n_hist ? nh : (unsigned)g;
            const unsigned g1 = g + my_chunk >= n_hist ? nh : (unsigned)(g + my_chunk);
            for (;;) {    // under the lock the old chunk can only shrink (it is shorter than n): its rest + the head of the new one
                const unsigned long long s2 = *(volatile unsigned long long *)&hp->state;
                const unsigned c2 = (unsigned)s2, e2 = (unsigned)(s2 >> 32);
                const unsigned from_old = e2 - c2, from_new = n - from_old;
                const unsigned nc = g0 + from_new < g1 ? g0 + from_new : g1;
                if (atomicCAS(&hp->state, s2, (unsigned long long)nc | ((unsigned long long)g1 << 32)) == s2) {
                    r0 = c2; rn0 = from_old; r1 = g0; break;
                }
            }
            if (g1 >= nh) *(volatile unsigned *)&hp->dry = 1u;
            GD_FENCE_BLOCK();
            atomicExch(&hp->lock, 0u);
            break;
        }
    }
    a0 = __shfl_sync(0xFFFFFFFFu, r0, 0);
    n0 = __shfl_sync(0xFFFFFFFFu, rn0, 0);
    a1 = __shfl_sync(0xFFFFFFFFu, r1, 0);
}

// ---- slot <-> registers
#define GD_SF(f) sl[(f) * GD_W_NSLOT + s]
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

// The two physics routines are inlined.  Compiled out of line (GD_PASS_INLINE 0: the caller's traversal state is saved
// around the call instead of competing with the photon state for registers) they measured 25 % slower on configs 2 / 3:
// the block context and the launch constants then travel through local memory.
#ifndef GD_PASS_INLINE
#define GD_PASS_INLINE 1
#endif
#if GD_PASS_INLINE
#define GD_PASS __device__ __forceinline__
#else
#define GD_PASS __device__ __noinline__
#endif

// ---- what the warps of a block share
struct GdBlk {
    float *sl;                                 // photon slots, SoA
    const float *tab;                          // attenuation tables
    const GdSource *src;
    unsigned *spec, *emitted, *peak, *cnt;     // per-block tallies and event counters
    GdQueue *q;                                // q[GD_Q_READY], q[GD_Q_RESULT], q[GD_Q_SLOW]
    GdQueue *ready, *result, *slow;
    GdHistPool *hist;
    unsigned *live;                            // slots that still carry or may get a history
    float *pair;                               // global: parked annihilation photons of the block's slots
};
struct GdRunArgs {                             // launch constants of a transport kernel
    unsigned long long first, n_hist, seed;
    float *edep_out;
    unsigned *flags_out;
    unsigned long long *next_history;
    unsigned chunk;
};
struct GdLaneCounters { unsigned n_done, n_skip, n_fast_cross, n_fast_coh; };

// ============================================================ general pass: any event, one per claimed slot
// (start of a history, start localisation, escape, crossing into KILL, photoelectric / Compton / pair event, cut-off,
// the next annihilation photon, tally + the next history of the block's chunk)
GD_PASS void gd_general_pass(const GdBlk &B, const GdBvh &bvh, const GdMaterials &M, const GdTally &tally, const GdRunArgs &A,
                          unsigned lane, GdLaneCounters &C) {
    float *sl = B.sl;
    const unsigned lt_mask = (1u << lane) - 1u;
    int s = 0;
    bool has = false;
    gd_q_claim(B.slow, true, 32, lane, s, has);
    GdLane L;
    L.mode = GD_MODE_DONE;
    GdHit hit;
    hit.t = 0.0f; hit.leaf = -1; hit.orig = GD_NO_FACET; hit.leaving = 1; hit.mats = 0;
    if (has) {
        gd_slot_load(sl, s, L, A.seed, A.first);
        if (L.pending) {
            const float *p = B.pair + s * 8;
            L.p_pos = gd_make(p[0], p[1], p[2]); L.p_axis = gd_make(p[3], p[4], p[5]); L.p_m = __float_as_int(p[6]);
        }
        // gd_lane_post reads the from-side id as "inside if leaving else outside" in LOCATE mode and the to-side id as
        // "outside if leaving else inside" in FLIGHT mode: present (from, to) that way
        hit.t = GD_SF(22);
        hit.orig = __float_as_int(GD_SF(23));
        hit.leaf = hit.orig == GD_NO_FACET ? -1 : 0;
        hit.mats = __float_as_int(GD_SF(24));          // inside := from, outside := to
    }
    GdLocalCounters cnt = {};
    GdHistory r;
    r.edep = 0.0f; r.flags = 0u; r.line = 0;
    bool fin = false;
    if (has && L.mode != GD_MODE_NEED) {
        const int was_pending = L.pending;
        fin = gd_lane_post(L, M, B.tab, *B.src, A.seed, hit, r, cnt);
        if (fin) {
            C.n_done++;
            const unsigned long long hrel = L.history - A.first;
            if (A.edep_out) A.edep_out[hrel] = r.edep;
            if (A.flags_out) A.flags_out[hrel] = r.flags;
        } else if (L.pending && !was_pending) {  // a pair event: park the two annihilation photons
            float *p = B.pair + s * 8;
            p[0] = L.p_pos.x; p[1] = L.p_pos.y; p[2] = L.p_pos.z;
            p[3] = L.p_axis.x; p[4] = L.p_axis.y; p[5] = L.p_axis.z; p[6] = __int_as_float(L.p_m);
        }
    }
    gd_tally_warp(fin, r, *B.src, tally, B.spec, B.emitted, B.peak, lane);
    {   // event counters, one shared-memory atomic per kind and pass (crossing / PE / Compton / coherent / pair; escapes,
        // re-localisations and cut-offs can accompany any of them)
        const unsigned v[8] = {cnt.n_crossings, cnt.n_pe, cnt.n_compton, cnt.n_coherent, cnt.n_pair, cnt.n_escaped,
                               cnt.n_leak, cnt.n_cutoff};
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const unsigned mk = __ballot_sync(0xFFFFFFFFu, v[k] != 0u);
            if (mk && lane == 0) atomicAdd(&B.cnt[4 + k], (unsigned)__popc(mk));
        }
    }
    // ---- finished slots take the next histories of the block's chunk
    const unsigned need_mask = __ballot_sync(0xFFFFFFFFu, has && L.mode == GD_MODE_NEED);
    if (need_mask) {
        unsigned a0, n0, a1;
        gd_hist_take(B.hist, (unsigned)__popc(need_mask), A.next_history, A.n_hist, A.chunk, gridDim.x, lane, a0, n0, a1);
        bool died = false;
        if (has && L.mode == GD_MODE_NEED) {
            const unsigned rk = __popc(need_mask & lt_mask);
            const unsigned long long h = rk < n0 ? a0 + rk : (unsigned long long)a1 + (rk - n0);
            if (h < A.n_hist) gd_lane_start(L, *B.src, A.seed, A.first + h);
            else { L.mode = GD_MODE_DONE; died = true; }
        }
        const unsigned died_mask = __ballot_sync(0xFFFFFFFFu, died);
        if (died_mask && lane == 0) atomicSub(B.live, (unsigned)__popc(died_mask));
    }
    // ---- the next query: answered by the clearance grid (the slot then waits in RESULT with its answer), or handed
    // to READY
    const bool live_lane = has && L.mode != GD_MODE_DONE;
    bool skip = false;
    if (live_lane) {
        float t_min, t_max;
        int filter;
        gd_lane_query(L, M, B.tab, t_min, t_max, filter);
        if (L.mode == GD_MODE_FLIGHT && L.sdist < GD_INF)
            skip = gd_flight_clear(bvh.grid, L.pos, L.sdist);
        gd_slot_store(sl, s, L, A.first);
        if (skip) { C.n_skip++; GD_SF(22) = L.sdist; GD_SF(23) = __int_as_float(GD_NO_FACET); GD_SF(24) = 0.0f; }
    }
    gd_q_push_to(B.q, live_lane ? (skip ? GD_Q_RESULT : GD_Q_READY) : -1, s, lane);
}

// ============================================================ chain burst: crossings and coherent events
// Lanes take RESULT slots (flights that met a facet or ended in an interaction) and handle the two event kinds of a
// scattering chain; anything else goes to the general queue untouched.  A slot whose next flight ends before the
// clearance of its grid cell stays on its lane and goes round again: the answer of that query is known ("none").  Lanes
// that gave their slot away take the next waiting result.  `can_leave`: the warp has other work to go to (rays in
// flight, or READY slots to fetch) once fewer than p_min lanes are busy.
template <bool CAN_TRAVERSE>
GD_PASS void gd_chain_burst(const GdBlk &B, const GdBvh &bvh, const GdMaterials &M, const GdRunArgs &A, const GdWaveTune &tune,
                         int my_rays, unsigned lane, GdLaneCounters &C, unsigned long long *pacc) {
    float *sl = B.sl;
    bool has = false, dirty = false;        // dirty: the lane's registers are newer than its slot
    int s = 0;
    GdLane L;
    L.mode = GD_MODE_DONE;
    GdHit hit;
    hit.t = 0.0f; hit.leaf = -1; hit.orig = GD_NO_FACET; hit.leaving = 1; hit.mats = 0;
    for (bool first_pass = true;; first_pass = false) {
        // ---- a pass needs p_min lanes with work -- or a warp with nothing else to do.  Decided on a snapshot of the
        // queues before anything is claimed: what is parked below are lanes whose answer is known (no facet within the
        // flight), never a freshly claimed traversal result.
        const unsigned free_mask = __ballot_sync(0xFFFFFFFFu, !has);
        const int n_has = 32 - __popc(free_mask);
        // the queues are consulted (and waiting results claimed) only once k_claim lanes are free: the claim and the
        // slot loads of one or two lanes are otherwise paid in every pass
        const bool refill = first_pass || 32 - n_has >= tune.k_claim || n_has < tune.p_min;
        int avail = 0, other = 1;
        if (refill) {
            if (lane == 0) { avail = gd_q_count(B.result); other = CAN_TRAVERSE ? gd_q_count(B.ready) : gd_q_count(B.slow); }
            avail = __shfl_sync(0xFFFFFFFFu, avail, 0);
            other = __shfl_sync(0xFFFFFFFFu, other, 0);
        }
        const int expect = n_has + (avail < 32 - n_has ? avail : 32 - n_has);
        const bool nothing_else = CAN_TRAVERSE ? (my_rays == 0 && other == 0) : other < tune.p_min;
        const bool go = expect > 0 && (first_pass || expect >= tune.p_min || nothing_else);
        bool to_slow = false, to_ready = false, skip = false;
        if (go) {
            // ---- fetch: lanes without a slot take waiting results
            bool got = false;
            int s_new = 0;
            int take = 0;
            if (refill) take = gd_q_claim(B.result, !has, 32 - n_has, lane, s_new, got);
            if (got) {
                s = s_new;
                gd_slot_load(sl, s, L, A.seed, A.first);
                hit.t = GD_SF(22);
                hit.orig = __float_as_int(GD_SF(23));
                hit.leaf = hit.orig == GD_NO_FACET ? -1 : 0;
                hit.mats = __float_as_int(GD_SF(24));          // inside := from, outside := to
                has = true; dirty = false;
            }
            if (n_has + take == 0) break;        // another warp was quicker
#ifdef GD_PROF
            pacc[2] += 1; pacc[3] += n_has + take;
#endif
            // ---- one event per lane
            int kind = 0;
            if (has) kind = gd_lane_fast_event(L, M, hit);
            to_slow = has && kind == 0;
            C.n_fast_cross += kind == 1; C.n_fast_coh += kind == 2;
            // ---- the next query: answered by the clearance grid, or handed to READY
            if (has && !to_slow) {
                float t_min, t_max;
                int filter;
                gd_lane_query(L, M, B.tab, t_min, t_max, filter);
                if (L.sdist < GD_INF) skip = gd_flight_clear(bvh.grid, L.pos, L.sdist);
                to_ready = !skip;
            }
        }
        // ---- one place where registers go back to the slot: a lane that hands its slot to READY, a lane that is parked
        // (!go) or whose next event is a general one while its registers are newer than the slot (both with the known
        // answer "no facet within the flight")
        const bool known = (!go && has) || (to_slow && dirty);
        if (to_ready || known) {
            gd_slot_store(sl, s, L, A.first);
            if (known) { GD_SF(22) = L.sdist; GD_SF(23) = __int_as_float(GD_NO_FACET); GD_SF(24) = 0.0f; }
        }
        gd_q_push_to(B.q, !go ? (has ? GD_Q_RESULT : -1) : (to_slow ? GD_Q_SLOW : (to_ready ? GD_Q_READY : -1)), s, lane);
        if (!go) break;
        has = skip;
        if (skip) { C.n_skip++; dirty = true; hit.t = L.sdist; hit.leaf = -1; hit.orig = GD_NO_FACET; hit.mats = 0; }
    }
}

// ============================================================ traversal service: retire finished rays, fetch READY slots
// Returns the number of slots fetched.  A start localisation, an escape (no facet, no interaction) and a crossing into
// KILL are general events; a crossing into another medium or an interaction goes to the chain burst.
GD_D int gd_trav_service(GdTrav &T, const GdBlk &B, const GdBvh &bvh, int *stack, int n_free, int rdy_min, unsigned lane, unsigned &n_query) {
    float *sl = B.sl;
    const bool done_l = T.slot >= 0 && T.node == GD_TRAV_DONE;
    bool slow = false;
    if (done_l) {
        const int s = T.slot;
        GD_SF(22) = T.t; GD_SF(23) = __int_as_float(T.orig); GD_SF(24) = __int_as_float(T.fromto);
        slow = T.filter == -2 || (T.orig == GD_NO_FACET ? !(T.t < GD_INF) : (T.fromto >> 16) == GD_MAT_KILL);
    }
    gd_q_push_to(B.q + GD_Q_RESULT, done_l ? (slow ? 1 : 0) : -1, T.slot, lane);
    if (done_l) T.slot = -1;
    bool got = false;
    int s = 0;
    if (rdy_min > 1) {                       // a helper warp fetches only from a READY queue that has piled up
        int r = 0;
        if (lane == 0) r = gd_q_count(B.ready);
        if (__shfl_sync(0xFFFFFFFFu, r, 0) < rdy_min) return 0;
    }
    const int tk = gd_q_claim(B.ready, T.slot < 0, n_free, lane, s, got);
    if (got) {
        const unsigned st = __float_as_uint(GD_SF(14));
        const bool loc = (int)((st >> 5) & 3u) == GD_MODE_LOCATE;
        gd_trav_begin(T, bvh, stack, GD_SF(0), GD_SF(1), GD_SF(2), GD_SF(3), GD_SF(4), GD_SF(5),
                      loc ? 0.0f : -GD_TBACK, loc ? GD_INF : GD_SF(13), loc ? -2 : (int)(st & 31u) - 1,
                      __float_as_int(GD_SF(19)), __float_as_int(GD_SF(20)), __float_as_int(GD_SF(21)), s);
        n_query++;
    }
    return tk;
}

// ---- block set-up and tear-down shared by the two transport kernels
#define GD_W_SHARED                                                                                              \
    extern __shared__ __align__(16) unsigned char gd_smem[];                                                     \
    __shared__ GdSource s_src;                                                                                   \
    __shared__ unsigned s_emitted[GD_MAX_LINES], s_peak[GD_MAX_LINES];                                           \
    __shared__ unsigned s_cnt[12];                                                                               \
    __shared__ GdQueue s_q[3];                                                                                   \
    GdQueue &s_ready = s_q[GD_Q_READY], &s_result = s_q[GD_Q_RESULT], &s_slow = s_q[GD_Q_SLOW];                    \
    __shared__ GdHistPool s_hist;                                                                                \
    __shared__ unsigned s_live;                                                                                  \
    const int n_tab = M.n_mat * 4 * M.n_grid;                                                                    \
    float *s_tab = (float *)gd_smem;                                                                             \
    unsigned *s_spec = (unsigned *)(s_tab + n_tab);                                                              \
    float *sl = (float *)(s_spec + tally.n_bins + 1);                                                            \
    for (int i = threadIdx.x; i < n_tab; i += blockDim.x) s_tab[i] = M.table[i];                                 \
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) s_spec[i] = 0;                                 \
    for (int i = threadIdx.x; i < (int)(sizeof(GdSource) / 4); i += blockDim.x) ((int *)&s_src)[i] = ((const int *)src)[i]; \
    if (threadIdx.x < GD_MAX_LINES) { s_emitted[threadIdx.x] = 0; s_peak[threadIdx.x] = 0; }                     \
    if (threadIdx.x < 12) s_cnt[threadIdx.x] = 0;                                                                \
    /* every slot starts in the general queue with mode NEED: the first passes start the first histories */     \
    for (int s = threadIdx.x; s < GD_W_NSLOT; s += blockDim.x) {                                                 \
        GD_SF(14) = __uint_as_float((unsigned)GD_MODE_NEED << 5);                                                \
        s_slow.ent[s] = (unsigned short)(gd_q_tag((unsigned)s) | (unsigned)s);                                   \
        s_ready.ent[s] = 0; s_result.ent[s] = 0;                                                                 \
    }                                                                                                            \
    if (threadIdx.x == 0) {                                                                                      \
        s_slow.head = 0; s_slow.tail = GD_W_NSLOT; s_result.head = 0; s_result.tail = 0; s_ready.head = 0; s_ready.tail = 0; \
        s_hist.state = 0ull; s_hist.lock = 0u; s_hist.dry = 0u;                                                  \
        s_live = GD_W_NSLOT;                                                                                     \
    }                                                                                                            \
    __syncthreads();                                                                                             \
    GdBlk B;                                                                                                     \
    B.sl = sl; B.tab = s_tab; B.src = &s_src; B.spec = s_spec; B.emitted = s_emitted; B.peak = s_peak; B.cnt = s_cnt; \
    B.q = s_q; B.ready = &s_ready; B.result = &s_result; B.slow = &s_slow; B.hist = &s_hist; B.live = &s_live;              \
    B.pair = pair_buf + (size_t)blockIdx.x * GD_W_NSLOT * 8;                                                     \
    GdRunArgs A;                                                                                                 \
    A.first = first; A.n_hist = n_hist; A.seed = seed; A.edep_out = edep_out; A.flags_out = flags_out;          \
    A.next_history = next_history; A.chunk = chunk;

// per-lane 32-bit work counters straight to the 64-bit global totals
GD_D void gd_flush_lane_counters(const GdTally &tally, unsigned lane, unsigned n_done, unsigned n_query, unsigned n_box,
                                 unsigned n_tri, unsigned n_skip, unsigned n_fast_cross, unsigned n_fast_coh) {
    const unsigned v[7] = {n_done, n_query, n_box, n_tri, n_skip, n_fast_cross, n_fast_coh};
    const int where[7] = {0, 1, 2, 3, 13, 4, 7};     // GdCounters: n_histories, n_queries, n_box_tests, n_tri_tests, n_skipped, n_crossings, n_coherent
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        unsigned long long x = v[k];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
        if (lane == 0 && x) atomicAdd(&((unsigned long long *)tally.counters)[where[k]], x);
    }
}
GD_D void gd_flush_block_tallies(const GdTally &tally, const unsigned *s_spec, const unsigned *s_emitted, const unsigned *s_peak,
                                 const unsigned *s_cnt) {
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

// dynamic shared memory: [table floats][spectrum u32 (n_bins+1)][slots: GD_W_NF x GD_W_NSLOT floats]
// pair_buf: global, 8 floats per slot of every block of the grid
// WIDTH: 4 = uncompressed 4-wide nodes (default), 8 = compressed 8-wide nodes
// Every warp does whichever kind of work there is (the default kernel).
template <int WIDTH, int THREADS = GD_W_THREADS>
__global__ void __launch_bounds__(THREADS, 1)
gd_k_transport_wave(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
                    unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
                    unsigned *__restrict__ flags_out, unsigned long long *next_history, unsigned chunk,
                    float *__restrict__ pair_buf, GdWaveTune tune) {
    GD_W_SHARED
    const unsigned lane = threadIdx.x & 31u;
    int stack[WIDTH == 8 ? GD_STACK8 : GD_STACK4];
    GdTrav T;
    gd_trav_idle(T);
    unsigned n_box = 0, n_tri = 0, n_query = 0;
    GdLaneCounters C = {0, 0, 0, 0};
    static_assert(GD_W_NSLOT == 1024, "queue entries hold a 10-bit slot number");
    // warps of the last SM sub-partition take the general passes first, so that the other three keep the two compact
    // loops in their instruction caches
    const bool slow_first = ((threadIdx.x >> 5) & 3u) == 3u;
    // every third warp takes READY slots whenever it has free lanes; the others only help when READY has piled up, so that
    // a trickle of rays fills the lanes of a few warps instead of a quarter of the lanes of all
    const bool t_pref = ((threadIdx.x >> 5) % 3u) == 0u;
    const int rdy_min = t_pref ? 1 : tune.t_help;
    unsigned idle_ns = 250u;
    int n_steps = tune.n_steps;
    unsigned round_no = 0, box_mark = 0, tri_mark = 0;
    unsigned long long *pacc = nullptr;
#ifdef GD_PROF
    unsigned long long pacc_[16] = {};
    pacc = pacc_;
    long long p_t0 = clock64();
#endif
    for (;;) {
        // ---- what next?  (queue lengths are snapshots: a wrong guess costs a pass with fewer lanes, never a result)
        const int my_rays = __popc(__ballot_sync(0xFFFFFFFFu, T.slot >= 0));
        int n_res = 0, n_rdy = 0, n_slow = 0;
        unsigned live = 0;
        if (lane == 0) {
            n_res = gd_q_count(&s_result); n_rdy = gd_q_count(&s_ready); n_slow = gd_q_count(&s_slow);
            live = *(volatile unsigned *)&s_live;
        }
        n_res = __shfl_sync(0xFFFFFFFFu, n_res, 0);
        n_rdy = __shfl_sync(0xFFFFFFFFu, n_rdy, 0);
        n_slow = __shfl_sync(0xFFFFFFFFu, n_slow, 0);
        live = __shfl_sync(0xFFFFFFFFu, live, 0);
        const bool t_work = my_rays > 0 || n_rdy >= rdy_min;
        const bool few_rays = my_rays < tune.t_keep;      // a warp with many rays in flight finishes them first: their slots are what the others wait for
        const bool other_work = t_work || n_res > 0;
        const bool do_slow = n_slow > 0 && (n_slow >= (slow_first ? tune.p_min : 8 * tune.p_min) || !other_work) && (few_rays || !t_work);
        const bool do_fast = !do_slow && n_res > 0 && few_rays && (n_res >= tune.p_min || !t_work);
        GD_PROF_ADD(10, 1);
        if (!do_slow && !do_fast && !t_work) {
            GD_PROF_ADD(11, 1);
            if (live == 0u) break;               // every slot of the block is dead
            __nanosleep(idle_ns);                // other warps hold all the work there is: back off
            if (idle_ns < 4000u) idle_ns *= 2u;
#ifdef GD_PROF
            { const long long t1 = clock64(); GD_PROF_ADD(8, t1 - p_t0); p_t0 = t1; }
#endif
            continue;
        }
        idle_ns = 250u;
        if (do_slow) {
            GD_PROF_ADD(7, 1);
            gd_general_pass(B, bvh, M, tally, A, lane, C);
#ifdef GD_PROF
            { const long long t1 = clock64(); GD_PROF_ADD(9, t1 - p_t0); p_t0 = t1; }
#endif
            continue;
        }
        if (do_fast) {
            GD_PROF_ADD(12, 1);
            gd_chain_burst<true>(B, bvh, M, A, tune, my_rays, lane, C, pacc);
#ifdef GD_PROF
            { const long long t1 = clock64(); GD_PROF_ADD(0, t1 - p_t0); p_t0 = t1; }
#endif
            continue;
        }
        GD_PROF_ADD(13, 1);
        // ================================================================ T-burst
        // Finished rays are retired and READY slots fetched in one go, once `k_fetch` lanes are free (finished or
        // idle): the queue operations are paid every few rounds instead of every round.  Unfinished rays stay in their
        // lanes' registers while the warp does physics.
        for (;;) {
            const bool done_l = T.slot >= 0 && T.node == GD_TRAV_DONE;
            const int n_free = __popc(__ballot_sync(0xFFFFFFFFu, T.slot < 0 || done_l));
            if (n_free >= tune.k_fetch || n_free == 32) {
#ifdef GD_PROF
                const long long ts0 = clock64();
#endif
                const int tk = gd_trav_service(T, B, bvh, stack, n_free, rdy_min, lane, n_query);
#ifdef GD_PROF
                GD_PROF_ADD(14, clock64() - ts0); GD_PROF_ADD(15, 1);
#endif
                // nothing to fetch and few rays left: see whether physics has piled up
                if (tk == 0 && 32 - n_free < tune.t_keep) {
                    if (n_free == 32) break;
                    int r = 0;
                    if (lane == 0) r = max(gd_q_count(&s_result), gd_q_count(&s_slow));
                    if (__shfl_sync(0xFFFFFFFFu, r, 0) >= tune.p_min) break;
                }
            }
            GD_PROF_ADD(4, 1); GD_PROF_ADD(5, __popc(__ballot_sync(0xFFFFFFFFu, T.slot >= 0 && T.node >= 0)));
            GD_PROF_ADD(6, __popc(__ballot_sync(0xFFFFFFFFu, T.slot >= 0 && T.node != GD_TRAV_DONE)));
            gd_trav_step<WIDTH>(T, bvh, stack, n_steps, n_box, n_tri);
            // node visits per round follow the warp's own ratio of node visits to triangle tests (deep walks between
            // leaves: long rounds; a leaf every other visit: short rounds), re-evaluated every 32 rounds
            if ((++round_no & 31u) == 0u && tune.n_steps_max > tune.n_steps) {
                const unsigned dv = __reduce_add_sync(0xFFFFFFFFu, n_box - box_mark), dt = __reduce_add_sync(0xFFFFFFFFu, n_tri - tri_mark);
                box_mark = n_box; tri_mark = n_tri;
                const int want = (int)((dv / (WIDTH == 8 ? 6u : 4u) + dt / 2u) / (dt > 0u ? dt : 1u));
                n_steps = want < tune.n_steps ? tune.n_steps : (want > tune.n_steps_max ? tune.n_steps_max : want);
            }
        }
#ifdef GD_PROF
        { const long long t1 = clock64(); GD_PROF_ADD(1, t1 - p_t0); p_t0 = t1; }
#endif
    }
#ifdef GD_PROF
    if (lane == 0) for (int k = 0; k < 16; ++k) if (pacc[k]) atomicAdd(&gd_prof[k], pacc[k]);
#endif
    gd_flush_lane_counters(tally, lane, C.n_done, n_query, n_box, n_tri, C.n_skip, C.n_fast_cross, C.n_fast_coh);
    __syncthreads();
    gd_flush_block_tallies(tally, s_spec, s_emitted, s_peak, s_cnt);
}

// Warp-specialised variant (GADEP_RUN_WARP_SPECIALISED): GD_WS_TWARPS lean traversal warps that only run the BVH loop
// and GD_WS_PWARPS physics warps that only run the chain bursts and general passes, on the same block-wide queues.
// setmaxnreg moves registers from the former to the latter.  Same results, bit for bit.
#ifndef GD_WS_TWARPS
#define GD_WS_TWARPS 16
#define GD_WS_PWARPS 8
#define GD_WS_REGS_T 56
#define GD_WS_REGS_P 128
#endif
#define GD_WS_THREADS (32 * (GD_WS_TWARPS + GD_WS_PWARPS))
// what the traversal warps give up must cover what the physics warps take, or the physics warps wait for ever
static_assert((65536 / GD_WS_THREADS / 8 * 8 - GD_WS_REGS_T) * GD_WS_TWARPS >= (GD_WS_REGS_P - 65536 / GD_WS_THREADS / 8 * 8) * GD_WS_PWARPS,
              "register budget of the warp-specialised kernel does not balance");
static_assert(GD_WS_TWARPS % 4 == 0 && GD_WS_PWARPS % 4 == 0, "setmaxnreg works on warpgroups");
template <int WIDTH>
__global__ void __launch_bounds__(GD_WS_THREADS, 1)
gd_k_transport_ws(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
                  unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
                  unsigned *__restrict__ flags_out, unsigned long long *next_history, unsigned chunk,
                  float *__restrict__ pair_buf, GdWaveTune tune) {
    GD_W_SHARED
    const unsigned lane = threadIdx.x & 31u;
    const int warp = threadIdx.x >> 5;
    unsigned idle_ns = 250u;
    if (warp < GD_WS_TWARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(GD_WS_REGS_T));
        int stack[WIDTH == 8 ? GD_STACK8 : GD_STACK4];
        GdTrav T;
        gd_trav_idle(T);
        unsigned n_box = 0, n_tri = 0, n_query = 0;
        for (;;) {
            const bool done_l = T.slot >= 0 && T.node == GD_TRAV_DONE;
            const int n_free = __popc(__ballot_sync(0xFFFFFFFFu, T.slot < 0 || done_l));
            if (n_free >= tune.k_fetch || n_free == 32) {
                const int tk = gd_trav_service(T, B, bvh, stack, n_free, 1, lane, n_query);
                if (tk == 0 && n_free == 32) {               // no ray in flight, none to fetch
                    unsigned live = 0;
                    if (lane == 0) live = *(volatile unsigned *)&s_live;
                    if (__shfl_sync(0xFFFFFFFFu, live, 0) == 0u) break;
                    __nanosleep(idle_ns);
                    if (idle_ns < 2000u) idle_ns *= 2u;
                    continue;
                }
                idle_ns = 250u;
            }
            gd_trav_step<WIDTH>(T, bvh, stack, tune.n_steps, n_box, n_tri);
        }
        gd_flush_lane_counters(tally, lane, 0, n_query, n_box, n_tri, 0, 0, 0);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(GD_WS_REGS_P));
        GdLaneCounters C = {0, 0, 0, 0};
        const bool slow_first = (warp & 3) == 3;
        for (;;) {
            int n_res = 0, n_slow = 0;
            unsigned live = 0;
            if (lane == 0) { n_res = gd_q_count(&s_result); n_slow = gd_q_count(&s_slow); live = *(volatile unsigned *)&s_live; }
            n_res = __shfl_sync(0xFFFFFFFFu, n_res, 0);
            n_slow = __shfl_sync(0xFFFFFFFFu, n_slow, 0);
            live = __shfl_sync(0xFFFFFFFFu, live, 0);
            const bool do_slow = n_slow > 0 && (n_slow >= (slow_first ? tune.p_min : 8 * tune.p_min) || n_res < tune.p_min);
            if (do_slow) { gd_general_pass(B, bvh, M, tally, A, lane, C); idle_ns = 250u; continue; }
            if (n_res > 0) { gd_chain_burst<false>(B, bvh, M, A, tune, 0, lane, C, nullptr); idle_ns = 250u; continue; }
            if (live == 0u) break;
            __nanosleep(idle_ns);
            if (idle_ns < 2000u) idle_ns *= 2u;
        }
        gd_flush_lane_counters(tally, lane, C.n_done, 0, 0, 0, C.n_skip, C.n_fast_cross, C.n_fast_coh);
    }
    __syncthreads();
    gd_flush_block_tallies(tally, s_spec, s_emitted, s_peak, s_cnt);
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
