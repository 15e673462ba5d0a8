// gadep_physics.cuh -- one photon history in float32 (PAPER.md:179 physics processes; PAPER.md:191 localisation
// from the nearest facet's side materials; PAPER.md:165 scoring in the sensitive volume).
// Step order and random-number consumption follow DESIGN.md "the path" so that the
// counter-based streams line up with any other implementation of the same description.
#pragma once
#include "gadep_bvh.cuh"

#define GD_TWO_PI 6.28318530717958647692f
#define GD_INF __int_as_float_inf()
GD_HD float __int_as_float_inf() { return gd_as_float(0x7F800000); }

// ---------------------------------------------------------------- O2: attenuation lookup
// tab: [n_mat][4][n_grid]; channels 0..2 hold ln(mu) (-1e30 for zero), channel 3 holds mu.
struct GdF4 { float a, b, c, d; };
GD_HD_NI GdF4 gd_mu_lookup_v(int n_grid, float ln_e0, float inv_dln, const float *tab, int m, float e) {
    float x = (logf(e) - ln_e0) * inv_dln;
    int j = (int)floorf(x);
    j = j < 0 ? 0 : (j > n_grid - 2 ? n_grid - 2 : j);
    float f = x - (float)j;
    float g = 1.0f - f;
    const float *t = tab + (m * 4) * n_grid + j;
    GdF4 mu;
    mu.a = expf(g * t[0] + f * t[1]);
    mu.b = expf(g * t[n_grid] + f * t[n_grid + 1]);
    mu.c = expf(g * t[2 * n_grid] + f * t[2 * n_grid + 1]);
    // pair production only above 2 m_e c^2: the grid cell that straddles the threshold would interpolate to > 0 (R17)
    mu.d = e > GD_TWO_MEC2 ? g * t[3 * n_grid] + f * t[3 * n_grid + 1] : 0.0f;
    return mu;
}
GD_HD float gd_mu_lookup(const GdMaterials &M, const float *tab, int m, float e, float mu[4]) {
    GdF4 r = gd_mu_lookup_v(M.n_grid, M.ln_e0, M.inv_dln, tab, m, e);
    mu[0] = r.a; mu[1] = r.b; mu[2] = r.c; mu[3] = r.d;
    return ((mu[0] + mu[1]) + mu[2]) + mu[3];
}

struct GdF2 { float s, c; };
GD_HD_NI GdF2 gd_sincos_2pi_v(float u) {
    GdF2 r;
#ifdef __CUDA_ARCH__
    sincospif(2.0f * u, &r.s, &r.c);
#else
    r.s = sinf(GD_TWO_PI * u); r.c = cosf(GD_TWO_PI * u);
#endif
    return r;
}
GD_HD void gd_sincos_2pi(float u, float &s, float &c) { GdF2 r = gd_sincos_2pi_v(u); s = r.s; c = r.c; }

// O4 / O12: isotropic direction from 2 draws
GD_HD GdVec3 gd_isotropic_from(float u1, float u2) {
    float w = 1.0f - 2.0f * u1;
    float st = sqrtf(fmaxf(0.0f, 1.0f - w * w));
    float s, c;
    gd_sincos_2pi(u2, s, c);
    return gd_make(st * c, st * s, w);
}
GD_HD GdVec3 gd_sample_isotropic(GdRng &g) {
    float u1 = gd_rng_next(g), u2 = gd_rng_next(g);
    float w = 1.0f - 2.0f * u1;
    float st = sqrtf(fmaxf(0.0f, 1.0f - w * w));
    float s, c;
    gd_sincos_2pi(u2, s, c);
    return gd_make(st * c, st * s, w);
}

// O13: rotate d by polar cosine c and azimuth 2*pi*u_phi
GD_HD_NI GdVec3 gd_rotate(GdVec3 d, float c, float u_phi) {
    float sp, cp;
    gd_sincos_2pi(u_phi, sp, cp);
    float s = sqrtf(fmaxf(0.0f, 1.0f - c * c));
    float q = 1.0f - d.z * d.z;
    GdVec3 r;
    if (q > 1.0e-12f) {
        float rho = sqrtf(q), ir = 1.0f / rho;
        r.x = d.x * c + s * (d.x * d.z * cp - d.y * sp) * ir;
        r.y = d.y * c + s * (d.y * d.z * cp + d.x * sp) * ir;
        r.z = d.z * c - s * rho * cp;
    } else {
        r.x = s * cp; r.y = s * sp; r.z = d.z >= 0.0f ? c : -c;
    }
    float n = 1.0f / sqrtf(r.x * r.x + r.y * r.y + r.z * r.z);
    r.x *= n; r.y *= n; r.z *= n;
    return r;
}

// O10: Klein-Nishina composition-rejection; returns eps = E'/E, cos(theta) in *cos_t
GD_HD float gd_sample_compton(GdRng &g, float e, float &cos_t) {
    float k = e * (1.0f / GD_MEC2);
    float eps0 = 1.0f / (1.0f + 2.0f * k);
    float a1 = logf(1.0f / eps0);
    float a2 = 0.5f * (1.0f - eps0 * eps0);
    float pa = a1 / (a1 + a2);
    float eps, t;
    for (;;) {
        float u1 = gd_rng_next(g), u2 = gd_rng_next(g), u3 = gd_rng_next(g);
        if (pa > u1) eps = expf(-a1 * u2);
        else eps = sqrtf(eps0 * eps0 + (1.0f - eps0 * eps0) * u2);
        t = (1.0f - eps) / (k * eps);
        float sin2 = t * (2.0f - t);
        if (1.0f - eps * sin2 / (1.0f + eps * eps) >= u3) break;
    }
    cos_t = 1.0f - t;
    return eps;
}

// O11: Thomson (1 + cos^2) law by exact inversion of the CDF (3c + c^3 + 4)/8
// (the two cube roots of Cardano's formula multiply to -1: one cube root and one reciprocal, taken on the side without
// cancellation)
GD_HD float gd_thomson_from(float u) {
    const float q = 4.0f * u - 2.0f;
    const float a = cbrtf(sqrtf(q * q + 1.0f) + fabsf(q));
    return copysignf(a - 1.0f / a, q);
}

// "No facet within the flight of length s from p" decided on the clearance grid alone (true = certain, false = ask the
// BVH): s (+ the float32 slack of s, of the cell lookup and of the plane distances) is shorter than the clearance of
// p's cell, or -- where that scalar is too small -- than the distance from p to every plane of the cell's list and
// than the list's reach.
GD_D bool gd_flight_clear(const GdGrid &g, const GdVec3 &p, float s) {
    if (!g.info) return false;
    const float need = fmaf(s, 1.0001f, 4.0f * GD_TBACK);
    const float fx = floorf((p.x - g.lox) * g.inv_h), fy = floorf((p.y - g.loy) * g.inv_h), fz = floorf((p.z - g.loz) * g.inv_h);
    const int ix = (int)fx, iy = (int)fy, iz = (int)fz;
    if ((unsigned)ix >= (unsigned)g.nx || (unsigned)iy >= (unsigned)g.ny || (unsigned)iz >= (unsigned)g.nz) return false;
    const unsigned w = __ldg(g.info + ((unsigned)iz * (unsigned)g.ny + (unsigned)iy) * (unsigned)g.nx + (unsigned)ix);   // <= 2^28 cells
    if (!(w & GD_CELL_LIST)) return need < (float)w * g.quarter_h;
    if (need < (float)(w & 7u) * g.quarter_h) return true;
    if (!(need < g.reach)) return false;
    const unsigned cnt = (w >> 3) & 15u;
    if (cnt == 15u) return true;
    const float rx = p.x - fmaf(fx + 0.5f, g.h, g.lox), ry = p.y - fmaf(fy + 0.5f, g.h, g.loy), rz = p.z - fmaf(fz + 0.5f, g.h, g.loz);
    const float4 *pl = g.planes + (size_t)((w >> 7) & 0xFFFFFFu) * GD_CELL_PLANES;
    float lb = g.reach;
#pragma unroll 1
    for (unsigned k = 0; k < cnt; ++k) {                     // one 128-byte line: the first load brings the others
        const float4 q = __ldg(pl + k);
        lb = fminf(lb, fabsf(fmaf(q.x, rx, fmaf(q.y, ry, fmaf(q.z, rz, q.w)))));
    }
    return need < lb;
}

struct GdHistory {
    float edep;        // scoring deposit; line energy for a full-absorption history
    unsigned flags;
    int line;
};

GD_HD void gd_deposit(const GdMaterials &M, int m, float e, float &dep, unsigned &flags) {
    if ((M.scoring_mask >> m) & 1u) dep += e;
    else flags |= GD_F_NONSCORING;
}
// Katz & Penfold: R [mg/cm^2] = 412 T^(1.265 - 0.0954 ln T); in mm for the material's density (R16)
GD_HD float gd_electron_range_mm(float t_mev, float rho) {
    if (!(t_mev > 0.0f) || !(rho > 0.0f)) return 0.0f;
    const float lt = logf(t_mev);
    return 412.0f * expf((1.265f - 0.0954f * lt) * lt) / (100.0f * rho);
}

// ---------------------------------------------------------------- lane state machine
// One lane carries one history at a time; every step of a live lane issues exactly one nearest-hit query
// (mode LOCATE: O5 start material; mode FLIGHT: O7.3), so a warp's lanes stay together in the traversal.
#define GD_MODE_NEED 0
#define GD_MODE_LOCATE 1
#define GD_MODE_FLIGHT 2
#define GD_MODE_DONE 3

struct GdLane {
    GdVec3 pos, dir;
    float e, tau, mu[4], mu_tot, sdist;
    int m, need_mu, mode;
    GdRng g;
    unsigned long long history;
    float dep;
    unsigned flags, n_events;
    int line, pending, p_m;
    GdVec3 p_pos, p_axis;
    GdExclude ex;          // facets crossed on this flight segment within the last GD_TBACK of path
    int n_stall;           // consecutive crossings without progress (safety net)
    // partial cross-section method only: remaining optical depth of every process, process that fires next
    float tau_c[4];
    int sel;
    // electron-range mode only (R16): energies set free at el_pos in material el_m by the last
    // gd_lane_post call, waiting for their segments; running number of the history's electrons
    int el_n, el_m;
    float el_T[2];
    GdVec3 el_pos;
    unsigned el_count;
};

// O4: source sampling on stream 0; leaves the lane in mode LOCATE
GD_HD void gd_lane_start(GdLane &L, const GdSource &S, unsigned long long seed, unsigned long long history) {
    L.history = history;
    gd_rng_init(L.g, seed, history, 0, 0);
    int nl = S.n_lines;
    const GdF4u u4 = gd_rng_peek4(L.g);               // draws 0..3: line, then (point source) the direction
    float ul = u4.a * S.line_cum[nl - 1]; L.g.draw += 1;
    int line = nl - 1;
    for (int l = 0; l < nl; ++l) if (ul < S.line_cum[l]) { line = l; break; }
    L.line = line;
    L.e = S.line_mev[line];
    if (S.kind == 1) {
        for (;;) {
            float u1 = gd_rng_next(L.g), u2 = gd_rng_next(L.g), u3 = gd_rng_next(L.g);
            float r = S.cyl_r * sqrtf(u1);
            float z = S.cyl_z0 + (S.cyl_z1 - S.cyl_z0) * u3;
            if (S.ex_r > 0.0f && r < S.ex_r && z >= S.ex_z0 && z <= S.ex_z1) continue;
            float s, c;
            gd_sincos_2pi(u2, s, c);
            L.pos = gd_make(r * c, r * s, z);
            break;
        }
    } else {
        L.pos = gd_make(S.pos[0], S.pos[1], S.pos[2]);
    }
    if (S.kind == 2) L.dir = gd_make(S.dir[0], S.dir[1], S.dir[2]);
    else if (S.kind == 0) { L.dir = gd_isotropic_from(u4.b, u4.c); L.g.draw += 2; }
    else L.dir = gd_sample_isotropic(L.g);
    if (S.n_copies > 1) {
        const int copy = (int)(history % (unsigned long long)S.n_copies);
        L.pos.x += S.copy_off[copy][0]; L.pos.y += S.copy_off[copy][1]; L.pos.z += S.copy_off[copy][2];
        L.line = copy * nl + line;
    }
    L.dep = 0.0f; L.flags = 0; L.n_events = 0; L.pending = 0;
    L.m = 0; L.need_mu = 1; L.mu_tot = 0.0f; L.tau = 0.0f; L.sdist = 0.0f;
    L.ex = gd_no_exclude(); L.n_stall = 0;
    L.mode = GD_MODE_LOCATE;
}

// ---- "partial cross-section method" (R2 / section 12): every process c keeps its own remaining
// optical depth tau_c; the flight ends where the first budget runs out (s = min_c tau_c / mu_c), that process fires, and
// only its budget is sampled again.  Same distribution as total-mu sampling + a selection draw, one draw fewer per event.
GD_HD void gd_partial_birth(GdLane &L) {
#pragma unroll
    for (int c = 0; c < 4; ++c) L.tau_c[c] = -logf(gd_rng_next(L.g));
}
GD_HD void gd_partial_step(GdLane &L) {
    float best = GD_INF;
    int sel = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float sc = L.mu[c] > 0.0f ? L.tau_c[c] / L.mu[c] : GD_INF;
        if (sc < best) { best = sc; sel = c; }
    }
    L.sdist = best; L.sel = sel;
}
GD_HD void gd_partial_advance(GdLane &L, float t) {
#pragma unroll
    for (int c = 0; c < 4; ++c) L.tau_c[c] -= L.mu[c] * t;
}

// parameters of the lane's next query
template <bool PARTIAL>
GD_HD void gd_lane_query_t(GdLane &L, const GdMaterials &M, const float *tab, float &t_min, float &t_max, int &filter) {
    if (L.mode == GD_MODE_LOCATE) { t_min = 0.0f; t_max = GD_INF; filter = -2; return; }
    if (L.need_mu) { L.mu_tot = gd_mu_lookup(M, tab, L.m, L.e, L.mu); L.need_mu = 0; }     // O2
    if (PARTIAL) gd_partial_step(L);
    else L.sdist = L.mu_tot > 0.0f ? L.tau / L.mu_tot : GD_INF;                             // O7.2
    t_min = -GD_TBACK; t_max = L.sdist; filter = L.m;                                       // O7.3
}
GD_HD void gd_lane_query(GdLane &L, const GdMaterials &M, const float *tab, float &t_min, float &t_max, int &filter) {
    gd_lane_query_t<false>(L, M, tab, t_min, t_max, filter);
}

// the current photon ended: start the next annihilation photon if one waits; returns true when the history is over
template <bool PARTIAL>
GD_HD bool gd_lane_next_photon_t(GdLane &L, unsigned long long seed) {
    if (L.pending == 0) return true;
    L.pos = L.p_pos; L.m = L.p_m; L.e = GD_MEC2; L.need_mu = 1;
    unsigned stream;
    if (L.pending == 2) { L.dir = L.p_axis; stream = 1; }
    else { L.dir = gd_make(-L.p_axis.x, -L.p_axis.y, -L.p_axis.z); stream = 2; }
    L.pending--;
    gd_rng_init(L.g, seed, L.history, stream, 0);
    if (PARTIAL) gd_partial_birth(L);
    else L.tau = -logf(gd_rng_next(L.g));                                                   // O7.1
    L.ex = gd_no_exclude(); L.n_stall = 0;
    return false;
}

// O14: flags and scoring deposit of a finished history
GD_HD void gd_lane_finish(GdLane &L, const GdSource &S, GdHistory &out) {
    if (!(L.flags & (GD_F_ESCAPED | GD_F_NONSCORING))) { L.flags |= GD_F_PEAK; L.dep = S.line_mev[L.line]; }
    L.flags &= ~GD_F_RELOC;
    L.flags |= ((unsigned)L.line & 0xFFu) << 8;
    L.flags |= (L.n_events > 0xFFFFu ? 0xFFFFu : L.n_events) << 16;
    out.edep = L.dep; out.flags = L.flags; out.line = L.line;
    L.mode = GD_MODE_NEED;
}

// an energy deposit: at once, or (ELECTRON, R16) noted for the caller, who lays it along an electron segment
#define GD_DEPOSIT(e_)                                                                         \
    do {                                                                                       \
        if (ELECTRON) { L.el_T[L.el_n++] = (e_); L.el_m = L.m; L.el_pos = L.pos; }             \
        else gd_deposit(M, L.m, (e_), L.dep, L.flags);                                         \
    } while (0)

// consume the query result; returns true when the history is finished (out is then valid; with ELECTRON the caller
// first resolves the noted deposits and then calls gd_lane_finish itself)
template <bool PARTIAL, bool ELECTRON = false>
GD_HD bool gd_lane_post_t(GdLane &L, const GdMaterials &M, const float *tab, const GdSource &S, unsigned long long seed,
                          const GdHit &hit_in, GdHistory &out, GdLocalCounters &cnt) {
    GdHit hit = hit_in;
    bool photon_done = false;
    if (L.mode == GD_MODE_LOCATE) {                                                         // O5
        L.m = hit.leaf < 0 ? M.world_material : (hit.leaving ? gd_mat_inside(hit.mats) : gd_mat_outside(hit.mats));
        if (L.flags & GD_F_RELOC) L.flags &= ~GD_F_RELOC;                                   // re-localisation: tau carries on
        else if (PARTIAL) gd_partial_birth(L);
        else L.tau = -logf(gd_rng_next(L.g));                                               // O7.1
        L.mode = GD_MODE_FLIGHT;
        // The first flight runs along the same ray as the localisation query, and the nearest facet ahead is by
        // construction the first one whose from-side is the start material: one traversal answers both (O5 + O7.3).
        L.mu_tot = gd_mu_lookup(M, tab, L.m, L.e, L.mu); L.need_mu = 0;                     // O2
        if (PARTIAL) gd_partial_step(L);
        else L.sdist = L.mu_tot > 0.0f ? L.tau / L.mu_tot : GD_INF;                         // O7.2
        if (hit.leaf >= 0 && !(hit.t <= L.sdist)) hit.leaf = -1;
    }
    if (hit.leaf >= 0) {                                                                    // O7.6 boundary first
        float t = fmaxf(hit.t, 0.0f);
        L.pos.x += t * L.dir.x; L.pos.y += t * L.dir.y; L.pos.z += t * L.dir.z;
        if (PARTIAL) gd_partial_advance(L, t);
        else L.tau -= L.mu_tot * t;
        L.m = hit.leaving ? gd_mat_outside(hit.mats) : gd_mat_inside(hit.mats);
        cnt.n_crossings++;
        L.need_mu = 1;
        // Facets crossed earlier on this straight segment stay excluded whatever the distance: for a grazing ray the
        // float32 error of t (position ulp / cos) exceeds GD_TBACK, and a facet 1e-4 behind can reappear inside the window.
        if (t > GD_TBACK) L.n_stall = 0;
        L.ex.c = L.ex.b; L.ex.b = L.ex.a; L.ex.a = hit.orig;
        if (L.m == GD_MAT_KILL) { L.flags |= GD_F_ESCAPED; cnt.n_escaped++; photon_done = true; }
        else if (++L.n_stall > 32) {       // > 32 facets inside 0.1 um: degenerate mesh; stop instead of spinning
            L.flags |= GD_F_ESCAPED | GD_F_LEAK; cnt.n_escaped++; cnt.n_leak++; photon_done = true;
        }
    } else if (!(L.sdist < GD_INF) && L.m != M.world_material && !(L.flags & GD_F_RELOC)) {
        // No facet ahead although the photon is not in the world material: a float32 inconsistency at a corner (the
        // rounded crossing point of one facet lies just outside its neighbour across the shared edge).  Localise again
        // from the current point and direction (O5), keep the optical depth; counted in n_leak / GD_F_LEAK.
        L.flags |= GD_F_LEAK | GD_F_RELOC; cnt.n_leak++;
        L.mode = GD_MODE_LOCATE; L.ex = gd_no_exclude(); L.n_stall = 0;
        return false;
    } else if (!(L.sdist < GD_INF)) {                                                       // O7.5
        L.flags |= GD_F_ESCAPED; cnt.n_escaped++;
        photon_done = true;
    } else {                                                                                // O7.4 / O8 interaction
        L.pos.x += L.sdist * L.dir.x; L.pos.y += L.sdist * L.dir.y; L.pos.z += L.sdist * L.dir.z;
        L.n_events++;
        L.ex = gd_no_exclude(); L.n_stall = 0;                            // new flight segment
        if (L.e < M.e_cut) { GD_DEPOSIT(L.e); cnt.n_cutoff++; photon_done = true; }
        else {
            GdF4u u4 = gd_rng_peek4(L.g);             // selection draw + the three draws of a coherent event
            bool tau_done = false;
            int ch = -1;
            if (PARTIAL) {                            // the process whose budget ran out fires; the others pay for the flight
                ch = L.sel;
                gd_partial_advance(L, L.sdist);
                u4.d = u4.c; u4.c = u4.b; u4.b = u4.a;    // no selection draw: the event's own draws start at once
            } else {
                float us = u4.a * L.mu_tot; L.g.draw += 1;
                float acc = 0.0f;
#pragma unroll
                for (int c = 0; c < 4; ++c) { acc += L.mu[c]; if (ch < 0 && us < acc) ch = c; }
                if (ch < 0) ch = L.mu[3] > 0.0f ? 3 : (L.mu[2] > 0.0f ? 2 : (L.mu[1] > 0.0f ? 1 : 0));
            }
            if (ch == 0) {                                                                  // O9 photoelectric
                GD_DEPOSIT(L.e); cnt.n_pe++;
                photon_done = true;
            } else if (ch == 1) {                                                           // O10 Compton
                float cost;
                float eps = gd_sample_compton(L.g, L.e, cost);
                float uphi = gd_rng_next(L.g);
                float e_new = eps * L.e;
                GD_DEPOSIT(L.e - e_new);
                L.dir = gd_rotate(L.dir, cost, uphi);
                L.e = e_new;
                cnt.n_compton++;
                L.need_mu = 1;
                if (L.e < M.e_cut) { GD_DEPOSIT(L.e); cnt.n_cutoff++; photon_done = true; }
            } else if (ch == 2) {                                                           // O11 coherent
                const float cost = gd_thomson_from(u4.b);
                L.dir = gd_rotate(L.dir, cost, u4.c);
                if (PARTIAL) L.tau_c[2] = -logf(u4.d); else L.tau = -logf(u4.d);             // O7.1
                tau_done = true;
                L.g.draw += 3;
                cnt.n_coherent++;
            } else {                                                                        // O12 pair
                GD_DEPOSIT(L.e - GD_TWO_MEC2);
                L.p_axis = gd_sample_isotropic(L.g);
                L.p_pos = L.pos; L.p_m = L.m; L.pending = 2;
                cnt.n_pair++;
                photon_done = true;
            }
            if (!photon_done && !tau_done) {                                                // O7.1
                if (PARTIAL) L.tau_c[ch] = -logf(gd_rng_next(L.g)); else L.tau = -logf(gd_rng_next(L.g));
            }
        }
    }
    if (!photon_done) return false;
    if (!gd_lane_next_photon_t<PARTIAL>(L, seed)) return false;
    // ---- O14
    if (!ELECTRON) gd_lane_finish(L, S, out);
    return true;
}
// The two event kinds that make up almost all events of a scattering chain, with the arithmetic of gd_lane_post_t
// (same expressions, same order: results are bit-identical): a boundary crossing into another medium, and a coherent
// scattering.  Returns 0 when the event is neither (or is a crossing into KILL, a stalled crossing, a photon below the
// cut-off): the lane is then untouched and the event belongs to gd_lane_post.  1 = crossing done, 2 = coherent done.
// Only for mode FLIGHT and a hit that is a crossing, or no hit with a finite flight length.
GD_D int gd_lane_fast_event(GdLane &L, const GdMaterials &M, const GdHit &hit) {
    if (hit.leaf >= 0) {                                                                    // O7.6 boundary first
        const int to = hit.leaving ? gd_mat_outside(hit.mats) : gd_mat_inside(hit.mats);
        const float t = fmaxf(hit.t, 0.0f);
        const int stall = t > GD_TBACK ? 1 : L.n_stall + 1;
        if (to == GD_MAT_KILL || stall > 32) return 0;
        L.pos.x += t * L.dir.x; L.pos.y += t * L.dir.y; L.pos.z += t * L.dir.z;
        L.tau -= L.mu_tot * t;
        L.m = to;
        L.need_mu = 1;
        L.n_stall = stall;
        L.ex.c = L.ex.b; L.ex.b = L.ex.a; L.ex.a = hit.orig;
        return 1;
    }
    if (L.e < M.e_cut) return 0;
    const GdF4u u4 = gd_rng_peek4(L.g);                   // selection draw + the three draws of a coherent event
    const float us = u4.a * L.mu_tot;
    float acc = 0.0f;
    int ch = -1;
#pragma unroll
    for (int c = 0; c < 4; ++c) { acc += L.mu[c]; if (ch < 0 && us < acc) ch = c; }
    if (ch != 2) return 0;
    L.pos.x += L.sdist * L.dir.x; L.pos.y += L.sdist * L.dir.y; L.pos.z += L.sdist * L.dir.z;     // O7.4
    L.n_events++;
    L.ex = gd_no_exclude(); L.n_stall = 0;
    const float cost = gd_thomson_from(u4.b);                                               // O11
    L.dir = gd_rotate(L.dir, cost, u4.c);
    L.tau = -logf(u4.d);                                                                    // O7.1
    L.g.draw += 4;
    return 2;
}

GD_HD bool gd_lane_post(GdLane &L, const GdMaterials &M, const float *tab, const GdSource &S, unsigned long long seed,
                        const GdHit &hit, GdHistory &out, GdLocalCounters &cnt) {
    return gd_lane_post_t<false>(L, M, tab, S, seed, hit, out, cnt);
}

// ---------------------------------------------------------------- parity localisation inside the transport loop
// intersections of the ray from the photon with every closed surface are counted (all hits, binary BVH);
// among the surfaces with an odd count the one with the nearest first intersection contains the photon.  Facets the
// photon has just crossed (ex) lie at t ~ 0 and are skipped -- the crossing itself already moved the photon to their
// far side.  Returns the material, or -3 when the hit list overflows.
#define GD_PAR_MAX_HITS 64
GD_HD int gd_locate_parity(const GdBvh &bvh, const GdRay &ray, const GdExclude &ex, int world, unsigned &n_box_tests,
                           unsigned &n_tri_tests) {
    int h_facet[GD_PAR_MAX_HITS], h_surf[GD_PAR_MAX_HITS], h_in[GD_PAR_MAX_HITS];
    float h_t[GD_PAR_MAX_HITS];
    int nh = 0;
    if (!bvh.root_is_leaf) {
        int stack[GD_STACK];
        int sp = 0, node = 0;
        for (;;) {
            if (node >= 0) {
                const GdNode &nd = bvh.nodes[node];
                const float4 a = nd.n0xy, b = nd.n1xy, z = nd.nz;
                const int4 lk = nd.link;
                n_box_tests += 2;
                float x0 = (a.x - ray.o.x) * ray.inv.x, x1 = (a.y - ray.o.x) * ray.inv.x;
                float y0 = (a.z - ray.o.y) * ray.inv.y, y1 = (a.w - ray.o.y) * ray.inv.y;
                float z0 = (z.x - ray.o.z) * ray.inv.z, z1 = (z.y - ray.o.z) * ray.inv.z;
                const float n0 = fmaxf(fmaxf(fminf(x0, x1), fminf(y0, y1)), fmaxf(fminf(z0, z1), 0.0f));
                float f0 = fminf(fminf(fmaxf(x0, x1), fmaxf(y0, y1)), fmaxf(z0, z1));
                f0 = f0 + fabsf(f0) * 4.0e-7f;
                x0 = (b.x - ray.o.x) * ray.inv.x; x1 = (b.y - ray.o.x) * ray.inv.x;
                y0 = (b.z - ray.o.y) * ray.inv.y; y1 = (b.w - ray.o.y) * ray.inv.y;
                z0 = (z.z - ray.o.z) * ray.inv.z; z1 = (z.w - ray.o.z) * ray.inv.z;
                const float n1 = fmaxf(fmaxf(fminf(x0, x1), fminf(y0, y1)), fmaxf(fminf(z0, z1), 0.0f));
                float f1 = fminf(fminf(fmaxf(x0, x1), fmaxf(y0, y1)), fmaxf(z0, z1));
                f1 = f1 + fabsf(f1) * 4.0e-7f;
                const bool g0 = n0 <= f0, g1 = n1 <= f1;
                if (g0 && g1) { stack[sp++] = lk.y; node = lk.x; }
                else if (g0) node = lk.x;
                else if (g1) node = lk.y;
                else if (sp == 0) break;
                else node = stack[--sp];
                continue;
            }
            const GdTri &tr = bvh.tris[~node];
            const int facet = gd_as_int(tr.v0.w);
            if (facet != ex.a && facet != ex.b && facet != ex.c) {
                float t, det;
                n_tri_tests++;
                if (gd_ray_tri(ray, tr.v0, tr.v1, tr.v2, t, det) && t > 0.0f) {
                    bool seen = false;
                    for (int k = 0; k < nh; ++k) seen = seen || h_facet[k] == facet;
                    if (!seen) {
                        if (nh == GD_PAR_MAX_HITS) return -3;
                        h_facet[nh] = facet; h_t[nh] = t; h_surf[nh] = gd_as_int(tr.v2.w);
                        h_in[nh] = gd_mat_inside(gd_as_int(tr.v1.w));
                        nh++;
                    }
                }
            }
            if (sp == 0) break;
            node = stack[--sp];
        }
    }
    int result = world;
    float best = GD_INF;
    for (int a = 0; a < nh; ++a) {
        bool first_of_surface = true;
        for (int b = 0; b < a; ++b) first_of_surface = first_of_surface && h_surf[b] != h_surf[a];
        if (!first_of_surface) continue;
        int count = 0;
        float first = GD_INF;
        for (int b = a; b < nh; ++b)
            if (h_surf[b] == h_surf[a]) { count++; first = fminf(first, h_t[b]); }
        if ((count & 1) && first < best) { best = first; result = h_in[a]; }
    }
    return result;
}

// One whole history on one lane (history-per-thread kernel, host emulation).
// PARITY: after the start localisation and after every boundary crossing the material comes from the parity rule
// instead of the facet's side ids (the side ids still say where the KILL boundary is); mismatches between the two
// rules are counted in cnt.n_cutoff's neighbour fields by the caller.
// ELECTRON: deposits become straight electron segments (R16).
template <bool PARITY, bool PARTIAL, bool ELECTRON = false>
GD_HD void gd_run_history_t(const GdBvh &bvh, const GdMaterials &M, const float *tab, const GdSource &S,
                            unsigned long long seed, unsigned long long history, GdHistory &out, GdLocalCounters &cnt,
                            unsigned &n_parity, unsigned &n_mismatch) {
    GdLane L;
    gd_lane_start(L, S, seed, history);
    L.el_n = 0; L.el_m = 0; L.el_count = 0;
    GdRay ray;
    GdHit hit;
    for (;;) {
        float t_min, t_max;
        int filter;
        gd_lane_query_t<PARTIAL>(L, M, tab, t_min, t_max, filter);
        gd_ray_setup(ray, L.pos, L.dir);
        cnt.n_queries++;
        gd_nearest_hit<false>(bvh, ray, t_min, t_max, filter, L.ex, true, hit, cnt.n_box_tests, cnt.n_tri_tests);
        const unsigned crossings_before = cnt.n_crossings;
        const bool was_locate = L.mode == GD_MODE_LOCATE;
        if (PARITY && was_locate) {
            // start material from the parity rule: present it as the from-side of the hit (or as the world material)
            const int m_par = gd_locate_parity(bvh, ray, L.ex, M.world_material, cnt.n_box_tests, cnt.n_tri_tests);
            n_parity++;
            const int m_side = hit.leaf < 0 ? M.world_material : (hit.leaving ? gd_mat_inside(hit.mats) : gd_mat_outside(hit.mats));
            if (m_par != m_side) {
                n_mismatch++;
                if (m_par >= 0 && hit.leaf >= 0) {      // the parity rule decides: present it as the facet's from-side
                    if (hit.leaving) hit.mats = (m_par & 0xFFFF) | (int)((unsigned)hit.mats & 0xFFFF0000u);
                    else hit.mats = (hit.mats & 0xFFFF) | (int)((unsigned)(m_par & 0xFFFF) << 16);
                }
            }
        }
        const bool finished = gd_lane_post_t<PARTIAL, ELECTRON>(L, M, tab, S, seed, hit, out, cnt);
        if (ELECTRON) {
            for (int k = 0; k < L.el_n; ++k) {
                // the k-th electron of the history: isotropic direction from stream 3, segment of the CSDA range, cut
                // at the first facet with the material on its from-side; the rest is left behind that facet
                const float t_kin = L.el_T[k];
                const float range = gd_electron_range_mm(t_kin, M.rho[L.el_m]);
                const float u1 = gd_rng_uniform_v((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)history, (uint32_t)(history >> 32), 3u, 2u * L.el_count);
                const float u2 = gd_rng_uniform_v((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)history, (uint32_t)(history >> 32), 3u, 2u * L.el_count + 1u);
                L.el_count++;
                float in_m = t_kin, beyond = 0.0f;
                int m2 = L.el_m;
                if (range > 0.0f) {
                    GdRay er;
                    GdHit eh;
                    gd_ray_setup(er, L.el_pos, gd_isotropic_from(u1, u2));
                    cnt.n_queries++;
                    gd_nearest_hit<false>(bvh, er, 0.0f, range, L.el_m, gd_no_exclude(), true, eh, cnt.n_box_tests, cnt.n_tri_tests);
                    if (eh.leaf >= 0 && eh.t < range) {
                        in_m = t_kin * (fmaxf(eh.t, 0.0f) / range); beyond = t_kin - in_m;
                        m2 = eh.leaving ? gd_mat_outside(eh.mats) : gd_mat_inside(eh.mats);
                    }
                }
                gd_deposit(M, L.el_m, in_m, L.dep, L.flags);
                if (beyond > 0.0f) {
                    if (m2 >= 0) gd_deposit(M, m2, beyond, L.dep, L.flags);
                    else L.flags |= GD_F_NONSCORING;          // left through the KILL boundary
                }
            }
            L.el_n = 0;
            if (finished) gd_lane_finish(L, S, out);
        }
        if (finished) return;
        if (PARITY && cnt.n_crossings != crossings_before && L.mode == GD_MODE_FLIGHT) {
            gd_ray_setup(ray, L.pos, L.dir);
            const int m_par = gd_locate_parity(bvh, ray, L.ex, M.world_material, cnt.n_box_tests, cnt.n_tri_tests);
            n_parity++;
            if (m_par != L.m) { n_mismatch++; if (m_par >= 0) { L.m = m_par; L.need_mu = 1; } }
        }
    }
}

GD_HD void gd_run_history(const GdBvh &bvh, const GdMaterials &M, const float *tab, const GdSource &S,
                          unsigned long long seed, unsigned long long history, GdHistory &out, GdLocalCounters &cnt) {
    unsigned a = 0, b = 0;
    gd_run_history_t<false, false>(bvh, M, tab, S, seed, history, out, cnt, a, b);
}
