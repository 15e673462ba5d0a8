// gadep_ws_kernels.cuh -- warp-specialised wavefront transport.
//
// One block of 896 threads per SM = 8 teams of 1 physics warp + 2-3 traversal warps (20 in all), each team with its own
// pool of GD_WS_SLOTS photon slots in shared memory.  The traversal warps only run the BVH loop (lean: they give
// registers back with setmaxnreg, 72 -> 56) and keep 20 x 32 rays in flight per SM; the physics warps (which take those
// registers, 72 -> 112) turn hits into the next queries.  Measurement variant (GADEP_RUN_WARP_SPECIALISED): same
// results as the default kernel bit for bit, same bulk rate, longer drain.  The two roles talk through two
// rings per team in shared memory:
//   READY   single producer (the physics warp), many consumers: an idle traversal lane draws a ticket (atomicAdd on
//           the head) and starts the ray of that ring position as soon as the published tail has passed it;
//   RESULT  many producers (traversal lanes claim positions with atomicAdd and mark their entry valid), single
//           consumer (the physics warp takes the valid entries at its head, up to 32 at a time).
// A slot is in exactly one place (a ring, a lane's registers, or the physics warp's hands), so neither ring can
// overflow.  Results do not depend on any of this: streams are keyed by the history index, tallies are integers.
#pragma once
#include "gadep_wave_kernels.cuh"

#ifndef GD_WS_TEAMS
#define GD_WS_TEAMS 8                       // physics warps per block (a multiple of 4: whole warpgroups)
#define GD_WS_TWARPS_TOTAL 20               // traversal warps per block (a multiple of 4)
#define GD_WS_SLOTS 192                     // photon slots per team
#define GD_WS_RING 256                      // ring capacity (power of two, > GD_WS_SLOTS)
#define GD_WS_REGS_T 56
#define GD_WS_REGS_P 112
#endif
#define GD_WS_THREADS (32 * (GD_WS_TEAMS + GD_WS_TWARPS_TOTAL))
// setmaxnreg moves registers inside the block's own allocation: what the traversal warps give up must cover what the
// physics warps take, or the physics warps wait for ever
static_assert((65536 / GD_WS_THREADS / 8 * 8 - GD_WS_REGS_T) * GD_WS_TWARPS_TOTAL >= (GD_WS_REGS_P - 65536 / GD_WS_THREADS / 8 * 8) * GD_WS_TEAMS,
              "register budget of the warp-specialised kernel does not balance");
#define GD_WS_NF 24                         // words per slot
#define GD_WS_VALID 0x8000u
#ifndef GD_WS_SETMAXNREG
#define GD_WS_SETMAXNREG 1
#endif

struct GdWsTeam {                           // shared-memory control block of one team
    unsigned short ready_ring[GD_WS_RING], res_ring[GD_WS_RING];
    int ready_tail;                         // entries [0, ready_tail) are published
    int ready_head;                         // next ticket
    int res_tail;                           // next result position to claim
    int done;                               // every slot of the team is dead
};

// slot layout: 0-2 pos, 3-5 dir, 6 e, 7 tau, 8-11 mu[4], 12 mu_tot, 13 state, 14 draw, 15 history, 16 dep,
// 17 flags | events, 18-20 crossed facets, 21-23 hit (t, facet, from | to)
#define GD_WSF(f) sl[(f) * GD_WS_SLOTS + s]
GD_D void gd_ws_store(float *sl, int s, const GdLane &L, unsigned long long first) {
    GD_WSF(0) = L.pos.x; GD_WSF(1) = L.pos.y; GD_WSF(2) = L.pos.z;
    GD_WSF(3) = L.dir.x; GD_WSF(4) = L.dir.y; GD_WSF(5) = L.dir.z;
    GD_WSF(6) = L.e; GD_WSF(7) = L.tau;
    GD_WSF(8) = L.mu[0]; GD_WSF(9) = L.mu[1]; GD_WSF(10) = L.mu[2]; GD_WSF(11) = L.mu[3];
    GD_WSF(12) = L.mu_tot;
    GD_WSF(13) = __uint_as_float(gd_pack_state(L));
    GD_WSF(14) = __uint_as_float(L.g.draw);
    GD_WSF(15) = __uint_as_float((unsigned)(L.history - first));
    GD_WSF(16) = L.dep;
    GD_WSF(17) = __uint_as_float((L.flags & 0xFFu) | ((L.n_events > 0xFFFFu ? 0xFFFFu : L.n_events) << 16));
    GD_WSF(18) = __int_as_float(L.ex.a); GD_WSF(19) = __int_as_float(L.ex.b); GD_WSF(20) = __int_as_float(L.ex.c);
}
GD_D void gd_ws_load(const float *sl, int s, GdLane &L, unsigned long long seed, unsigned long long first) {
    L.pos = gd_make(GD_WSF(0), GD_WSF(1), GD_WSF(2));
    L.dir = gd_make(GD_WSF(3), GD_WSF(4), GD_WSF(5));
    L.e = GD_WSF(6); L.tau = GD_WSF(7);
    L.mu[0] = GD_WSF(8); L.mu[1] = GD_WSF(9); L.mu[2] = GD_WSF(10); L.mu[3] = GD_WSF(11);
    L.mu_tot = GD_WSF(12);
    L.sdist = L.mu_tot > 0.0f ? L.tau / L.mu_tot : GD_INF;          // as gd_lane_query computed it
    const unsigned st = __float_as_uint(GD_WSF(13));
    L.m = (int)(st & 31u) - 1; L.mode = (int)((st >> 5) & 3u); L.line = (int)((st >> 7) & 63u);
    L.pending = (int)((st >> 13) & 3u); L.n_stall = (int)((st >> 15) & 63u); L.need_mu = (int)((st >> 23) & 1u);
    L.history = first + (unsigned long long)__float_as_uint(GD_WSF(15));
    gd_rng_init(L.g, seed, L.history, (st >> 21) & 3u, __float_as_uint(GD_WSF(14)));
    L.dep = GD_WSF(16);
    const unsigned fe = __float_as_uint(GD_WSF(17));
    L.flags = fe & 0xFFu; L.n_events = fe >> 16;
    L.ex.a = __float_as_int(GD_WSF(18)); L.ex.b = __float_as_int(GD_WSF(19)); L.ex.c = __float_as_int(GD_WSF(20));
    L.cool = 0; L.qkind = 0; L.sc = L.pos; L.sr = 0.0f;
}

// ---------------------------------------------------------------- physics warp of a team
GD_D void gd_ws_physics(GdWsTeam *tm, float *sl, const GdMaterials &M, const float *s_tab, const GdSource &s_src,
                        unsigned long long first, unsigned long long n_hist, unsigned long long seed, const GdTally &tally,
                        unsigned *s_spec, unsigned *s_emitted, unsigned *s_peak, unsigned *s_cnt, float *edep_out,
                        unsigned *flags_out, unsigned long long *next_history, unsigned chunk, float *pair) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    unsigned long long w_cur = 0, w_end = 0;
    unsigned n_done = 0;
    int head = 0, n_dead = 0, ready_tail = 0;
    int boot = 0;                            // slots [boot, GD_WS_SLOTS) have not had their first history yet
    for (;;) {
        // ---- take up to 32 slots: first the never-started ones, then the valid entries at the head of RESULT
        int s = -1;
        int take;
        if (boot < GD_WS_SLOTS) {
            take = GD_WS_SLOTS - boot < 32 ? GD_WS_SLOTS - boot : 32;
            if ((int)lane < take) { s = boot + (int)lane; GD_WSF(13) = __uint_as_float((unsigned)GD_MODE_NEED << 5); }
            boot += take;
        } else {
            const unsigned e = *(volatile unsigned short *)&tm->res_ring[(head + (int)lane) & (GD_WS_RING - 1)];
            const unsigned vm = __ballot_sync(0xFFFFFFFFu, (e & GD_WS_VALID) != 0u);
            take = vm == 0xFFFFFFFFu ? 32 : __ffs(~vm) - 1;
            if (take == 0) {
                if (n_dead == GD_WS_SLOTS) break;
                __nanosleep(100);
                continue;
            }
            if ((int)lane < take) {
                s = (int)(e & ~GD_WS_VALID);
                *(volatile unsigned short *)&tm->res_ring[(head + (int)lane) & (GD_WS_RING - 1)] = 0;
            }
            head += take;
            __threadfence_block();            // the hit fields were written before the entry was marked valid
        }
        const bool act = s >= 0;
        const int sc = act ? s : 0;
        GdLane L;
        L.mode = GD_MODE_DONE;
        if (act) {
            const int s = sc;
            gd_ws_load(sl, s, L, seed, first);
            if (L.pending) {
                const float *p = pair + s * 8;
                L.p_pos = gd_make(p[0], p[1], p[2]); L.p_axis = gd_make(p[3], p[4], p[5]); L.p_m = __float_as_int(p[6]);
            }
            if (L.mode != GD_MODE_NEED) {
                GdHit hit;
                hit.t = GD_WSF(21);
                hit.orig = __float_as_int(GD_WSF(22));
                hit.leaf = hit.orig == GD_NO_FACET ? -1 : 0;
                hit.leaving = 1;
                hit.mats = __float_as_int(GD_WSF(23));          // inside := from, outside := to
                GdLocalCounters cnt = {};
                const int was_pending = L.pending;
                GdHistory r;
                if (gd_lane_post(L, M, s_tab, s_src, seed, hit, r, cnt)) {
                    n_done++;
                    gd_tally_history(r, s_src, tally, s_spec, s_emitted, s_peak);
                    const unsigned long long hrel = L.history - first;
                    if (edep_out) edep_out[hrel] = r.edep;
                    if (flags_out) flags_out[hrel] = r.flags;
                } else if (L.pending && !was_pending) {
                    float *p = pair + s * 8;
                    p[0] = L.p_pos.x; p[1] = L.p_pos.y; p[2] = L.p_pos.z;
                    p[3] = L.p_axis.x; p[4] = L.p_axis.y; p[5] = L.p_axis.z; p[6] = __int_as_float(L.p_m);
                }
                const int kind = cnt.n_crossings ? 4 : (cnt.n_coherent ? 7 : (cnt.n_compton ? 6 : (cnt.n_pe ? 5 : (cnt.n_pair ? 8 : -1))));
                if (kind >= 0) atomicAdd(&s_cnt[kind], 1u);
                if (cnt.n_escaped) atomicAdd(&s_cnt[9], cnt.n_escaped);
                if (cnt.n_leak) atomicAdd(&s_cnt[10], cnt.n_leak);
                if (cnt.n_cutoff) atomicAdd(&s_cnt[11], cnt.n_cutoff);
            }
        }
        // ---- next history for the slots that finished one
        const unsigned need_mask = __ballot_sync(0xFFFFFFFFu, act && L.mode == GD_MODE_NEED);
        if (need_mask) {
            const unsigned n_need = __popc(need_mask);
            unsigned long long new_base = 0;
            const bool refill = w_cur + n_need > w_end;
            if (refill) {
                if (lane == 0) new_base = atomicAdd(next_history, (unsigned long long)chunk);
                new_base = __shfl_sync(0xFFFFFFFFu, new_base, 0);
            }
            if (act && L.mode == GD_MODE_NEED) {
                unsigned long long h = w_cur + __popc(need_mask & lt_mask);
                if (h >= w_end) h = new_base + (h - w_end);
                if (h < n_hist) gd_lane_start(L, s_src, seed, first + h);
                else L.mode = GD_MODE_DONE;
            }
            if (refill) { w_cur = new_base + (w_cur + n_need - w_end); w_end = new_base + chunk; }
            else w_cur += n_need;
        }
        // ---- prepare the next query and publish the slot in READY
        const bool live = act && L.mode != GD_MODE_DONE;
        if (live) {
            float t_min, t_max;
            int filter;
            gd_lane_query(L, M, s_tab, t_min, t_max, filter);
            gd_ws_store(sl, sc, L, first);
        }
        const unsigned live_mask = __ballot_sync(0xFFFFFFFFu, live);
        n_dead += take - __popc(live_mask);
        if (live) tm->ready_ring[(ready_tail + __popc(live_mask & lt_mask)) & (GD_WS_RING - 1)] = (unsigned short)sc;
        __threadfence_block();                // slot fields and ring entries before the tail
        __syncwarp();
        ready_tail += __popc(live_mask);
        if (lane == 0) *(volatile int *)&tm->ready_tail = ready_tail;
    }
    __threadfence_block();
    if (lane == 0) *(volatile int *)&tm->done = 1;
    {
        unsigned long long x = n_done;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) x += __shfl_down_sync(0xFFFFFFFFu, x, o);
        if (lane == 0 && x) atomicAdd(&((unsigned long long *)tally.counters)[0], x);
    }
}

// ---------------------------------------------------------------- traversal warp of a team
GD_D void gd_ws_traverse(GdWsTeam *tm, float *sl, const GdBvh &bvh, const GdWaveTune &tune, GdCounters *counters) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    int stack[GD_STACK4];
    GdTrav T;
    gd_trav_idle(T);
    int ticket = -1;                          // position in READY this idle lane waits for
    unsigned n_box = 0, n_tri = 0, n_query = 0;
    for (;;) {
        // ---- idle lanes without a ticket draw one (warp-aggregated), lanes with a ticket start as soon as it is served
        const unsigned want_mask = __ballot_sync(0xFFFFFFFFu, T.slot < 0 && ticket < 0);
        if (want_mask && (__popc(want_mask) >= tune.k_fetch || __ballot_sync(0xFFFFFFFFu, T.slot >= 0) == 0u)) {
            int base = 0;
            if (lane == 0) base = atomicAdd(&tm->ready_head, __popc(want_mask));
            base = __shfl_sync(0xFFFFFFFFu, base, 0);
            if (T.slot < 0 && ticket < 0) ticket = base + __popc(want_mask & lt_mask);
        }
        const int tail = *(volatile int *)&tm->ready_tail;
        if (ticket >= 0 && ticket < tail) {
            __threadfence_block();            // ring entry and slot fields were written before the tail moved
            const int s = (int)tm->ready_ring[ticket & (GD_WS_RING - 1)];
            const unsigned st = __float_as_uint(GD_WSF(13));
            const bool loc = (int)((st >> 5) & 3u) == GD_MODE_LOCATE;
            const float mu_tot = GD_WSF(12);
            const float sdist = mu_tot > 0.0f ? GD_WSF(7) / mu_tot : GD_TINF;
            gd_trav_begin(T, bvh, stack, GD_WSF(0), GD_WSF(1), GD_WSF(2), GD_WSF(3), GD_WSF(4), GD_WSF(5), loc ? 0.0f : -GD_TBACK,
                          loc ? GD_TINF : sdist, loc ? -2 : (int)(st & 31u) - 1, __float_as_int(GD_WSF(18)),
                          __float_as_int(GD_WSF(19)), __float_as_int(GD_WSF(20)), s);
            n_query++;
            ticket = -1;
        }
        const unsigned busy = __ballot_sync(0xFFFFFFFFu, T.slot >= 0);
        if (busy == 0u) {
            if (*(volatile int *)&tm->done) break;
            __nanosleep(200);
            continue;
        }
        gd_trav_step(T, bvh, stack, tune.n_steps, n_box, n_tri);
        // ---- finished rays: hit into the slot, slot into RESULT
        const bool fin = T.slot >= 0 && T.node == GD_TRAV_DONE;
        const unsigned fin_mask = __ballot_sync(0xFFFFFFFFu, fin);
        if (fin_mask) {
            int base = 0;
            if (fin) {
                const int s = T.slot;
                GD_WSF(21) = T.t; GD_WSF(22) = __int_as_float(T.orig); GD_WSF(23) = __int_as_float(T.fromto);
            }
            __threadfence_block();
            if (lane == 0) base = atomicAdd(&tm->res_tail, __popc(fin_mask));
            base = __shfl_sync(0xFFFFFFFFu, base, 0);
            if (fin) {
                *(volatile unsigned short *)&tm->res_ring[(base + __popc(fin_mask & lt_mask)) & (GD_WS_RING - 1)] =
                    (unsigned short)((unsigned)T.slot | GD_WS_VALID);
                T.slot = -1;
            }
        }
    }
    GdLocalCounters cnt = {};
    cnt.n_queries = n_query; cnt.n_box_tests = n_box; cnt.n_tri_tests = n_tri;
    gd_flush_counters(cnt, counters, 0);
}

// dynamic shared memory: [table floats][spectrum u32 (n_bins+1)][teams x GD_WS_NF x GD_WS_SLOTS floats][team control]
__global__ void __launch_bounds__(GD_WS_THREADS, 1)
gd_k_transport_ws(GdBvh bvh, GdMaterials M, const GdSource *__restrict__ src, unsigned long long first,
                  unsigned long long n_hist, unsigned long long seed, GdTally tally, float *__restrict__ edep_out,
                  unsigned *__restrict__ flags_out, unsigned long long *next_history, unsigned chunk,
                  float *__restrict__ pair_buf, GdWaveTune tune) {
    extern __shared__ __align__(16) unsigned char gd_smem[];
    __shared__ GdSource s_src;
    __shared__ unsigned s_emitted[GD_MAX_LINES], s_peak[GD_MAX_LINES];
    __shared__ unsigned s_cnt[14];
    __shared__ GdWsTeam s_team[GD_WS_TEAMS];
    const int n_tab = M.n_mat * 4 * M.n_grid;
    float *s_tab = (float *)gd_smem;
    unsigned *s_spec = (unsigned *)(s_tab + n_tab);
    float *s_slots = (float *)(s_spec + tally.n_bins + 1);
    for (int i = threadIdx.x; i < n_tab; i += blockDim.x) s_tab[i] = M.table[i];
    for (int i = threadIdx.x; i <= tally.n_bins; i += blockDim.x) s_spec[i] = 0;
    for (int i = threadIdx.x; i < (int)(sizeof(GdSource) / 4); i += blockDim.x) ((int *)&s_src)[i] = ((const int *)src)[i];
    for (int i = threadIdx.x; i < (int)(sizeof(s_team) / 4); i += blockDim.x) ((int *)s_team)[i] = 0;
    if (threadIdx.x < GD_MAX_LINES) { s_emitted[threadIdx.x] = 0; s_peak[threadIdx.x] = 0; }
    if (threadIdx.x < 14) s_cnt[threadIdx.x] = 0;
    __syncthreads();

    const int warp = threadIdx.x >> 5;
    if (warp < GD_WS_TEAMS) {                 // warps 0..3: one warpgroup of physics warps, one per team
#if GD_WS_SETMAXNREG
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(GD_WS_REGS_P));
#endif
        const int team = warp;
        gd_ws_physics(&s_team[team], s_slots + (size_t)team * GD_WS_NF * GD_WS_SLOTS, M, s_tab, s_src, first, n_hist, seed, tally,
                      s_spec, s_emitted, s_peak, s_cnt, edep_out, flags_out, next_history, chunk,
                      pair_buf + ((size_t)blockIdx.x * GD_WS_TEAMS + team) * GD_WS_SLOTS * 8);
    } else {                                  // warps 4..31: seven warpgroups of traversal warps
#if GD_WS_SETMAXNREG
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(GD_WS_REGS_T));
#endif
        const int team = (warp - GD_WS_TEAMS) % GD_WS_TEAMS;
        gd_ws_traverse(&s_team[team], s_slots + (size_t)team * GD_WS_NF * GD_WS_SLOTS, bvh, tune, tally.counters);
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
    if (threadIdx.x >= 4 && threadIdx.x < 14 && s_cnt[threadIdx.x])
        atomicAdd(&((unsigned long long *)tally.counters)[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
}
