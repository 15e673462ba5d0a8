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
GD_HD float gd_mu_lookup(const GdMaterials &M, const float *tab, int m, float e, float mu[4]) {
    float x = (logf(e) - M.ln_e0) * M.inv_dln;
    int j = (int)floorf(x);
    j = j < 0 ? 0 : (j > M.n_grid - 2 ? M.n_grid - 2 : j);
    float f = x - (float)j;
    float g = 1.0f - f;
    const float *t = tab + (m * 4) * M.n_grid + j;
    mu[0] = expf(g * t[0] + f * t[1]);
    mu[1] = expf(g * t[M.n_grid] + f * t[M.n_grid + 1]);
    mu[2] = expf(g * t[2 * M.n_grid] + f * t[2 * M.n_grid + 1]);
    mu[3] = g * t[3 * M.n_grid] + f * t[3 * M.n_grid + 1];
    return ((mu[0] + mu[1]) + mu[2]) + mu[3];
}

GD_HD void gd_sincos_2pi(float u, float &s, float &c) {
#ifdef __CUDA_ARCH__
    sincospif(2.0f * u, &s, &c);
#else
    s = sinf(GD_TWO_PI * u); c = cosf(GD_TWO_PI * u);
#endif
}

// O4 / O12: isotropic direction from 2 draws
GD_HD GdVec3 gd_sample_isotropic(GdRng &g) {
    float u1 = gd_rng_next(g), u2 = gd_rng_next(g);
    float w = 1.0f - 2.0f * u1;
    float st = sqrtf(fmaxf(0.0f, 1.0f - w * w));
    float s, c;
    gd_sincos_2pi(u2, s, c);
    return gd_make(st * c, st * s, w);
}

// O13: rotate d by polar cosine c and azimuth 2*pi*u_phi
GD_HD GdVec3 gd_rotate(GdVec3 d, float c, float u_phi) {
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
GD_HD float gd_sample_thomson(GdRng &g) {
    float u = gd_rng_next(g);
    float c = 8.0f * u - 4.0f;
    float r = sqrtf(0.25f * c * c + 1.0f);
    return cbrtf(0.5f * c + r) + cbrtf(0.5f * c - r);
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

// One history: O4 source, O5 start material, O7 flight loop, O8-O12 interactions, O14 flags.
GD_HD void gd_run_history(const GdBvh &bvh, const GdMaterials &M, const float *tab, const GdSource &S,
                          unsigned long long seed, unsigned long long history, GdHistory &out, GdLocalCounters &cnt) {
    GdRng g;
    gd_rng_init(g, seed, history, 0, 0);
    // ---- O4 source
    int nl = S.n_lines;
    float ul = gd_rng_next(g) * S.line_cum[nl - 1];
    int line = nl - 1;
    for (int l = 0; l < nl; ++l) if (ul < S.line_cum[l]) { line = l; break; }
    GdVec3 pos, dir;
    float e = S.line_mev[line];
    if (S.kind == 1) {
        for (;;) {
            float u1 = gd_rng_next(g), u2 = gd_rng_next(g), u3 = gd_rng_next(g);
            float r = S.cyl_r * sqrtf(u1);
            float z = S.cyl_z0 + (S.cyl_z1 - S.cyl_z0) * u3;
            if (S.ex_r > 0.0f && r < S.ex_r && z >= S.ex_z0 && z <= S.ex_z1) continue;
            float s, c;
            gd_sincos_2pi(u2, s, c);
            pos = gd_make(r * c, r * s, z);
            break;
        }
    } else {
        pos = gd_make(S.pos[0], S.pos[1], S.pos[2]);
    }
    if (S.kind == 2) dir = gd_make(S.dir[0], S.dir[1], S.dir[2]);
    else dir = gd_sample_isotropic(g);

    GdRay ray;
    GdHit hit;
    // ---- O5 start material: nearest facet ahead, no filter
    int m;
    {
        gd_ray_setup(ray, pos, dir);
        cnt.n_queries++;
        gd_nearest_hit(bvh, ray, 0.0f, GD_INF, -2, hit, cnt.n_box_tests, cnt.n_tri_tests);
        m = hit.leaf < 0 ? M.world_material : (hit.leaving ? gd_mat_inside(hit.mats) : gd_mat_outside(hit.mats));
    }

    float dep = 0.0f;
    unsigned flags = 0, n_events = 0;
    int pending = 0;              // 2: annihilation photons A and B wait; 1: B waits
    GdVec3 p_pos = pos, p_axis = dir;
    int p_m = m;
    unsigned draw0 = g.draw;
    unsigned stream = 0;

    for (;;) {                    // photons of this history: primary, then A (stream 1), then B (stream 2)
        gd_rng_init(g, seed, history, stream, draw0);
        float tau = -logf(gd_rng_next(g));                       // O7.1
        float mu[4], mu_tot = 0.0f;
        bool need_mu = true;
        for (;;) {                // flight loop
            if (need_mu) { mu_tot = (m >= 0) ? gd_mu_lookup(M, tab, m, e, mu) : 0.0f; need_mu = false; }
            float sdist = mu_tot > 0.0f ? tau / mu_tot : GD_INF;     // O7.2
            gd_ray_setup(ray, pos, dir);
            cnt.n_queries++;
            gd_nearest_hit(bvh, ray, -GD_TBACK, sdist, m, hit, cnt.n_box_tests, cnt.n_tri_tests);   // O7.3
            if (hit.leaf >= 0) {                                    // O7.6 boundary first
                float t = fmaxf(hit.t, 0.0f);
                pos.x += t * dir.x; pos.y += t * dir.y; pos.z += t * dir.z;
                tau -= mu_tot * t;
                m = hit.leaving ? gd_mat_outside(hit.mats) : gd_mat_inside(hit.mats);
                cnt.n_crossings++;
                need_mu = true;
                if (m == GD_MAT_KILL) { flags |= GD_F_ESCAPED; cnt.n_escaped++; break; }
                continue;
            }
            if (!(sdist < GD_INF)) {                                // O7.5 nothing ahead, no interaction
                flags |= GD_F_ESCAPED; cnt.n_escaped++;
                if (m != M.world_material) { flags |= GD_F_LEAK; cnt.n_leak++; }
                break;
            }
            // ---- O7.4 / O8 interaction at pos + s d
            pos.x += sdist * dir.x; pos.y += sdist * dir.y; pos.z += sdist * dir.z;
            n_events++;
            if (e < M.e_cut) { gd_deposit(M, m, e, dep, flags); cnt.n_cutoff++; break; }
            float us = gd_rng_next(g) * mu_tot;
            int ch = -1;
            float acc = 0.0f;
#pragma unroll
            for (int c = 0; c < 4; ++c) { acc += mu[c]; if (ch < 0 && us < acc) ch = c; }
            if (ch < 0) ch = mu[3] > 0.0f ? 3 : (mu[2] > 0.0f ? 2 : (mu[1] > 0.0f ? 1 : 0));
            if (ch == 0) {                                          // O9 photoelectric
                gd_deposit(M, m, e, dep, flags); cnt.n_pe++;
                break;
            } else if (ch == 1) {                                   // O10 Compton
                float cost;
                float eps = gd_sample_compton(g, e, cost);
                float uphi = gd_rng_next(g);
                float e_new = eps * e;
                gd_deposit(M, m, e - e_new, dep, flags);
                dir = gd_rotate(dir, cost, uphi);
                e = e_new;
                cnt.n_compton++;
                need_mu = true;
                if (e < M.e_cut) { gd_deposit(M, m, e, dep, flags); cnt.n_cutoff++; break; }
            } else if (ch == 2) {                                   // O11 coherent: E, m, mu unchanged
                float cost = gd_sample_thomson(g);
                float uphi = gd_rng_next(g);
                dir = gd_rotate(dir, cost, uphi);
                cnt.n_coherent++;
            } else {                                                // O12 pair
                gd_deposit(M, m, e - GD_TWO_MEC2, dep, flags);
                p_axis = gd_sample_isotropic(g);
                p_pos = pos; p_m = m; pending = 2;
                cnt.n_pair++;
                break;
            }
            tau = -logf(gd_rng_next(g));                            // O7.1 after every interaction
        }
        if (pending == 0) break;
        pos = p_pos; m = p_m; e = GD_MEC2; draw0 = 0;
        if (pending == 2) { dir = p_axis; stream = 1; }
        else { dir = gd_make(-p_axis.x, -p_axis.y, -p_axis.z); stream = 2; }
        pending--;
    }
    // ---- O14
    if (!(flags & (GD_F_ESCAPED | GD_F_NONSCORING))) { flags |= GD_F_PEAK; dep = S.line_mev[line]; }
    flags |= ((unsigned)line & 0xFFu) << 8;
    flags |= (n_events > 0xFFFFu ? 0xFFFFu : n_events) << 16;
    out.edep = dep; out.flags = flags; out.line = line;
}
