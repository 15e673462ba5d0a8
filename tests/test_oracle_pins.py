"""Pins of the CPU oracle against what the paper and the mathematics fix.
None of these compares the oracle with itself or with the CUDA path."""
import math

import numpy as np
import pytest

import detmesh as dm
from detmesh.configs import SRC_BEAM, SRC_POINT
from detmesh.geometry import Line, discretise, merge_surfaces, revolve
from oracle import gadep_oracle as orc

MEC2 = 0.51099895
RE2 = 2.8179403262e-13 ** 2


# ------------------------------------------------------------------ P10 RNG
def test_philox_known_answer_vectors():
    # Random123 known-answer vectors for philox4x32-10 (Salmon et al., SC'11 reference distribution)
    assert list(orc.philox([0, 0, 0, 0], [0, 0])) == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
    assert list(orc.philox([0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [0xA4093822, 0x299F31D0])) == \
        [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]
    out = orc.philox([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2)
    assert [int(out[0]), int(out[1]), int(out[3])] == [0x408F276D, 0x41C83B0E, 0x6D5451FD]


def test_philox_stream_layout_against_independent_python_implementation():
    # counter = (history_lo, history_hi, draw/4, stream), key = (seed_lo, seed_hi); u = ((w>>9)+0.5) 2^-23
    for seed, hist, stream in [(1, 0, 0), (7, 123456789012, 2), (2 ** 40 + 3, 2 ** 33 + 5, 1)]:
        ref = dm.philox_u01_host(seed & 0xFFFFFFFF, seed >> 32, (hist & 0xFFFFFFFF, hist >> 32, 0, stream), 12)
        got = [orc.u01(seed, hist, stream, k) for k in range(12)]
        assert np.array_equal(ref, np.array(got))
        assert all(0.0 < u < 1.0 and float(np.float32(u)) == float(u) for u in got)   # exactly representable in float32


# ------------------------------------------------------------------ O1 / O2 tables
def kn_dsigma_domega(k, c):
    eps = 1.0 / (1.0 + k * (1.0 - c))
    return 0.5 * RE2 * eps * eps * (eps + 1.0 / eps - (1.0 - c * c))


def kn_quadrature(k, n=20001):
    x, w = np.polynomial.legendre.leggauss(400)
    f = kn_dsigma_domega(k, x) * 2 * np.pi
    eps = 1.0 / (1.0 + k * (1.0 - x))
    tot = (w * f).sum()
    return tot, (w * f * eps).sum() / tot, (w * f * x).sum() / tot, (w * f * eps * eps).sum() / tot


def test_klein_nishina_total_closed_form_vs_quadrature_and_limits():
    assert dm.sigma_kn_total(MEC2) == pytest.approx(2.865399e-25, rel=1e-6)          # SURVEY.md O1 check value
    assert dm.sigma_kn_total(1e-7) == pytest.approx(8 * np.pi / 3 * RE2, rel=1e-5)     # Thomson limit 6.652459e-25
    for e in (0.0595, 0.6617, 1.3325, 3.0):
        assert dm.sigma_kn_total(e) == pytest.approx(kn_quadrature(e / MEC2)[0], rel=1e-9)


def test_table_check_values_ge():
    w = dm.make_config(1)
    s = orc.OracleScene(w)
    ge = dm.MAT["Ge_active"]
    # SURVEY.md O1 (1/cm); oracle returns 1/mm
    for e, pe, co in [(0.6617, 0.004066, 0.361832), (0.0595, 5.59278, 0.771685), (1.3325, 4.9794e-4, 0.257987)]:
        assert 10 * s.mu(ge, 0, e) == pytest.approx(pe, rel=2e-4)
        assert 10 * s.mu(ge, 1, e) == pytest.approx(co, rel=2e-5)
    mu_t = s.mu(ge, 0, 0.6617) + s.mu(ge, 1, 0.6617)
    assert math.exp(-mu_t * 10) == pytest.approx(0.693573, rel=2e-5)
    assert math.exp(-mu_t * 60) == pytest.approx(0.111315, rel=1e-4)
    # pair (Q2): Ge 6.94e-4 /cm at 1332.5 keV, 1.57e-2 /cm at 3 MeV; zero below threshold
    assert 10 * s.mu(ge, 3, 1.3325) == pytest.approx(6.94e-4, rel=5e-3)
    assert 10 * s.mu(ge, 3, 3.0) == pytest.approx(1.57e-2, rel=5e-3)
    assert s.mu(ge, 3, 1.0) == 0.0
    # Ge K-edge step x1/7 below 11.1 keV at the grid points
    g = dm.energy_grid()
    assert s.mu(ge, 0, g[3]) / s.mu(ge, 0, g[4]) == pytest.approx((g[4] / g[3]) ** 3 / 7.0, rel=1e-5)
    # vacuum and config-0 coherent are identically zero
    assert s.mu(dm.MAT["vacuum"], 1, 0.5) == 0.0
    assert orc.OracleScene(dm.make_config(0)).mu(ge, 2, 0.5) == 0.0


def test_interpolation_exact_on_power_laws_and_grid_points():
    w = dm.make_config(1)
    s = orc.OracleScene(w)
    g = dm.energy_grid()
    al = dm.MAT["Al"]
    for i in (0, 17, 100, 199):
        for ch in range(4):
            assert s.mu(al, ch, g[i]) == pytest.approx(float(w.mu[al, ch, i]), rel=1e-12, abs=1e-300)
    # log-log interpolation reproduces a pure power law between grid points (float32 table rounding only)
    for e in (0.0123, 0.2, 1.7):
        z, a = dm.ELEMENTS["Al"]
        pe = 2.699 * 6.02214076e23 / a * 4.5e-33 * z ** 4.5 / e ** 3 * 0.1
        coh = 2.699 * 6.02214076e23 / a * 7.0e-27 * z ** 2.5 / e ** 2 * 0.1
        assert s.mu(al, 0, e) == pytest.approx(pe, rel=3e-7)
        assert s.mu(al, 2, e) == pytest.approx(coh, rel=3e-7)
    # pair channel is linear in f across the threshold bracket (zero-safe)
    j = int(np.searchsorted(g, 2 * MEC2)) - 1
    e = math.exp(0.5 * (math.log(g[j]) + math.log(g[j + 1])))
    assert w.mu[al, 3, j] == 0 and w.mu[al, 3, j + 1] > 0
    assert s.mu(al, 3, e) == pytest.approx(0.5 * float(w.mu[al, 3, j + 1]), rel=1e-9)


# ------------------------------------------------------------------ P2 ray-triangle
def _one_triangle_scene(v):
    s = orc.OracleScene()
    s.load_mesh(np.asarray(v, dtype=np.float32), np.array([[0, 1, 2]], dtype=np.int32), np.zeros(1, np.int32),
                np.array([1], np.int32), np.array([0], np.int32), 0)
    return s


def test_ray_triangle_hand_computed():
    s = _one_triangle_scene([[0, 0, 0], [1, 0, 0], [0, 1, 0]])      # n = +z
    hit, t, dn = s.ray_triangle(0, [0.25, 0.25, 2.0], [0, 0, -1.0])
    assert hit and t == pytest.approx(2.0) and dn < 0               # moving against the normal: entering
    hit, t, dn = s.ray_triangle(0, [0.25, 0.25, -3.0], [0, 0, 1.0])
    assert hit and t == pytest.approx(3.0) and dn > 0               # along the normal: leaving
    assert not s.ray_triangle(0, [0.75, 0.75, 1.0], [0, 0, -1.0])[0]   # outside the hypotenuse
    assert s.ray_triangle(0, [0.5, 0.5, 1.0], [0, 0, -1.0])[0]          # on the edge: inclusive
    assert s.ray_triangle(0, [0.0, 0.0, 1.0], [0, 0, -1.0])[0]          # on a vertex
    assert not s.ray_triangle(0, [0.2, 0.2, 1.0], [1.0, 0, 0])[0]       # parallel
    hit, t, _ = s.ray_triangle(0, [0.2, 0.2, 1.0], [0, 0, 1.0])         # behind: negative t is reported
    assert hit and t == pytest.approx(-1.0)
    d = np.array([0.3, -0.2, -1.0]); d /= np.linalg.norm(d)
    o = np.array([0.3, 0.3, 0.0]) - 5.0 * d
    hit, t, _ = s.ray_triangle(0, o, d)
    assert hit and t == pytest.approx(5.0, rel=1e-12)


def test_ray_triangle_vs_plane_and_edge_function_formulation():
    rng = np.random.default_rng(11)
    n_hit = 0
    for _ in range(300):
        v = rng.normal(size=(3, 3)).astype(np.float32)
        s = _one_triangle_scene(v)
        vd = v.astype(np.float64)
        nrm = np.cross(vd[1] - vd[0], vd[2] - vd[0])
        for _ in range(40):
            o = rng.normal(size=3) * 1.2
            d = rng.normal(size=3); d /= np.linalg.norm(d)
            hit, t, dn = s.ray_triangle(0, o, d)
            den = nrm @ d
            t2 = nrm @ (vd[0] - o) / den
            p = o + t2 * d
            inside = all(np.cross(vd[(i + 1) % 3] - vd[i], p - vd[i]) @ nrm >= -1e-12 * (nrm @ nrm) for i in range(3))
            margin = min(np.cross(vd[(i + 1) % 3] - vd[i], p - vd[i]) @ nrm / (nrm @ nrm) for i in range(3))
            if abs(margin) < 1e-9:
                continue
            assert hit == inside
            if hit:
                n_hit += 1
                assert t == pytest.approx(t2, rel=1e-9, abs=1e-12)
                assert np.sign(dn) == np.sign(den)
    assert n_hit > 200


def test_nearest_hit_is_minimum_over_all_triangles_and_axis_ray():
    w = dm.make_config(0)
    s = orc.OracleScene(w)
    tri, t, leaving = s.nearest_hit([0.3, 0.2, 250.0], [0, 0, -1.0])
    assert tri >= 0 and t == pytest.approx(250.0) and leaving == 0
    tri, t, leaving = s.nearest_hit([0.3, 0.2, -10.0], [0, 0, -1.0])
    assert t == pytest.approx(50.0) and leaving == 1
    rng = np.random.default_rng(5)
    for _ in range(200):
        o = rng.uniform(-40, 40, 3)
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        tri, t, _ = s.nearest_hit(o, d)
        ts = [s.ray_triangle(i, o, d) for i in range(w.mesh.n_tri)]
        cand = [(tt, i) for i, (h, tt, _) in enumerate(ts) if h and tt > 0]
        if not cand:
            assert tri == -1
        else:
            assert (t, tri) == min(cand)


# ------------------------------------------------------------------ P3 localisation
def test_parity_rule_equals_side_id_rule_and_no_leaks():
    w = dm.make_config(1)
    s = orc.OracleScene(w)
    rng = np.random.default_rng(3)
    n = 1500
    org, d = dm.configs.make_rays(n, 3, 45.0, -105.0, 10.0)
    seen = set()
    for i in range(n):
        a = s.locate_sideid(org[i].astype(np.float64), d[i].astype(np.float64))
        b = s.locate_parity(org[i].astype(np.float64), d[i].astype(np.float64))
        assert a == b
        seen.add(a)
    assert {dm.MAT["Ge_active"], dm.MAT["vacuum"], dm.MAT["Al"], dm.MAT["air"], dm.MAT["Cu"]} <= seen
    # from an interior point of a closed surface every direction hits (0 leaks)
    dirs = orc.sample_isotropic(9, 2000)
    for k in range(2000):
        tri, _, leaving = s.nearest_hit([1.0, 2.0, -40.0], dirs[k])
        assert tri >= 0 and leaving == 1


def test_material_at_known_points_config1():
    s = orc.OracleScene(dm.make_config(1))
    M = dm.MAT
    # generic (non-degenerate) rays: the Jordan count is only defined off the edges and vertices
    up = [0.0123, 0.0071, 0.9999]
    pts = {(20.0, 0.13, -30.0): M["Ge_active"], (34.6, 0.13, -30.0): M["Ge_dead"], (20.0, 0.13, -0.3): M["Ge_dead"],
           (0.5, 0.1, -40.0): M["vacuum"], (5.0001, 0.01, -40.0): M["Ge_dead"], (35.5, 0.13, -30.0): M["Cu"],
           (38.0, 0.13, -30.0): M["vacuum"], (41.5, 0.13, -30.0): M["Al"], (10.0, 0.13, 5.5): M["Al"],
           (100.0, 0.13, 0): M["air"], (10.0, 0.13, 2.0): M["vacuum"], (0.001, 0.0005, -14.99985): M["Ge_dead"]}
    for p, m in pts.items():
        for d in (up, [0.6, 0.0, -0.8], [-0.48, 0.64, 0.6]):
            assert s.locate_sideid(list(p), d) == m, (p, d)
            assert s.locate_parity(list(p), d) == m, (p, d)


# ------------------------------------------------------------------ helpers for custom scenes
def _cyl(R, z_top, z_bot, n_theta=32):
    return revolve(discretise([Line(0, z_top, R, z_top, 1), Line(R, z_top, R, z_bot, 1), Line(R, z_bot, 0, z_bot, 1)]),
                   n_theta)


def _scene(surfaces, mu, is_scoring, source):
    mesh = merge_surfaces(surfaces, 0)
    s = orc.OracleScene()
    s.set_materials(mu, is_scoring, dm.E_MIN_MEV, dm.E_MAX_MEV)
    s.load_mesh(mesh.vertices, mesh.triangles, mesh.tri_surface, mesh.surf_inside, mesh.surf_outside, 0)
    s.set_source(**source)
    return s


def _beam(e_kev, pos=(1.234, 0.567, 50.0)):
    return {"kind": SRC_BEAM, "pos": pos, "dir": (0, 0, -1), "line_mev": [e_kev * 1e-3], "line_intensity": [1.0]}


# ------------------------------------------------------------------ P4 free flight
def test_slab_pe_only_fepe_is_one_minus_exp():
    mu, sc, _ = dm.make_tables(coh_coeff=0.0)
    mu = mu.copy(); mu[:, 1:, :] = 0.0                       # photoelectric only
    x = 10.0
    v, t = _cyl(100.0, 0.0, -x)
    s = _scene([("slab", v, t, 1, 0)], mu, sc, _beam(120.0))
    n = 400_000
    _, em, pk, cnt = s.run(n, 4)
    p = 1 - math.exp(-s.mu(1, 0, 0.12) * x)
    assert 0.2 < p < 0.9
    assert abs(pk[0] / n - p) < 4 * math.sqrt(p * (1 - p) / n)
    assert cnt["n_filter_reject"] == 0 and cnt["n_leak"] == 0


def test_zero_event_fraction_with_tau_carry_over_across_layers():
    # five 2 mm Ge layers separated by vacuum gaps = 10 mm of Ge: P(no event) = exp(-mu_tot 10) = 0.693573
    w = dm.make_config(0)
    surfs = []
    for k in range(5):
        v, t = _cyl(100.0, -2.5 * k, -2.5 * k - 2.0)
        surfs.append((f"layer{k}", v, t, 1, 0))
    s = _scene(surfs, w.mu, w.is_scoring, _beam(661.7))
    n = 400_000
    edep, flags, other, esc, cnt = s.run_histories(0, n, 2, details=True)
    nev = flags >> 16
    p0 = (nev == 0).mean()
    assert abs(p0 - 0.693573) < 4 * math.sqrt(0.693573 * 0.306427 / n)
    assert cnt["n_crossings"] >= 10 * (nev == 0).sum()


# ------------------------------------------------------------------ P5 solid angle
def test_on_axis_solid_angle_of_ngon_cylinder():
    w = dm.make_config(0)
    mu = w.mu.copy(); mu[1, 0, :] = 1.0e3; mu[1, 1:, :] = 0.0      # "black" crystal: absorbed at the surface
    s = orc.OracleScene(w)
    s.set_materials(mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
    n = 4_000_000
    _, em, pk, _ = s.run(n, 1)
    N, R, h = 64, 30.0, 250.0
    frac = (2 * np.pi - 2 * N * np.arctan(np.tan(np.pi / N) * h / np.sqrt(h * h + R * R))) / (4 * np.pi)
    assert frac == pytest.approx(0.003555923, rel=1e-6)          # SURVEY.md P5 printed value
    assert abs(pk[0] / n - frac) < 4 * math.sqrt(frac / n)


# ------------------------------------------------------------------ P6 energy accounting
@pytest.mark.parametrize("cfg,n", [(1, 4000), (3, 600)])
def test_energy_accounting_per_history(cfg, n):
    w = dm.make_config(cfg)
    s = orc.OracleScene(w)
    edep, flags, other, esc, cnt = s.run_histories(0, n, 1, details=True)
    line = (flags >> 8) & 0xFF
    e0 = s.line_mev[line]
    peak = (flags & orc.F_PEAK) != 0
    dep_sc = np.where(peak, e0, edep)
    assert np.allclose(dep_sc + other + esc, e0, rtol=1e-12, atol=1e-13)
    assert (edep <= e0 * (1 + 1e-12)).all()
    assert cnt["n_leak"] == 0 and cnt["n_filter_reject"] == 0
    assert ((flags & orc.F_PEAK) == 0)[(flags & (orc.F_ESCAPED | orc.F_NONSCORING)) != 0].all()


# ------------------------------------------------------------------ P7 sampling laws
@pytest.mark.parametrize("e,printed", [(0.0595, (0.906997, 0.078007, 0.826200)), (0.6617, (0.618441, 0.318700, 0.432929)),
                                       (1.3325, (0.520877, 0.387824, 0.338794)), (3.0, (0.422677, 0.462002, 0.257963))])
def test_klein_nishina_sampling_moments(e, printed):
    _, m_eps, m_cos, m_eps2 = kn_quadrature(e / MEC2)
    assert (m_eps, m_cos, m_eps2) == pytest.approx(printed, abs=2e-6)   # SURVEY.md P7 printed values
    n = 400_000
    eps, cos = orc.sample_compton(e, 5, n)
    k = e / MEC2
    assert np.allclose(eps, 1.0 / (1.0 + k * (1.0 - cos)), rtol=1e-12)      # Compton kinematics
    assert (eps >= 1 / (1 + 2 * k) - 1e-15).all() and (eps <= 1).all()
    for got, ref in [(eps, m_eps), (cos, m_cos), (eps * eps, m_eps2)]:
        assert abs(got.mean() - ref) < 4 * got.std() / math.sqrt(n)
    # shape, not only moments: binned cos(theta) against the differential cross-section
    edges = np.linspace(-1, 1, 21)
    hist, _ = np.histogram(cos, edges)
    x, wq = np.polynomial.legendre.leggauss(40)
    exp = []
    for a, b in zip(edges[:-1], edges[1:]):
        xm = 0.5 * (b - a) * x + 0.5 * (a + b)
        exp.append(0.5 * (b - a) * (wq * kn_dsigma_domega(k, xm)).sum())
    exp = np.array(exp); exp *= n / exp.sum()
    chi2 = ((hist - exp) ** 2 / exp).sum()
    assert chi2 < 50      # 19 dof; P(chi2 > 50) ~ 1e-4


def test_thomson_and_isotropic_moments():
    n = 400_000
    c = orc.sample_thomson(3, n)
    assert abs(c.mean()) < 4 * c.std() / math.sqrt(n)
    assert abs((c * c).mean() - 0.4) < 4 * (c * c).std() / math.sqrt(n)
    assert (np.abs(c) <= 1 + 1e-12).all()
    # CDF (3 mu + mu^3 + 4)/8 is inverted exactly: F(c(u)) = u for the very draws used
    u = np.array([orc.u01(3, i, 0, 0) for i in range(200)])
    assert np.allclose((3 * c[:200] + c[:200] ** 3 + 4) / 8, u, atol=1e-12)
    d = orc.sample_isotropic(4, n)
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-12)
    assert (np.abs(d.mean(axis=0)) < 4 * 0.5774 / math.sqrt(n)).all()
    assert abs((d[:, 2] ** 2).mean() - 1 / 3) < 4 * 0.2981 / math.sqrt(n)


def test_rotation_preserves_polar_cosine_and_norm():
    rng = np.random.default_rng(8)
    for _ in range(300):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        c, phi = rng.uniform(-1, 1), rng.uniform(0, 2 * np.pi)
        r = orc.rotate(d, c, phi)
        assert np.linalg.norm(r) == pytest.approx(1.0, abs=1e-12)
        assert r @ d == pytest.approx(c, abs=1e-9)
    for w in (1.0, -1.0):
        r = orc.rotate([0, 0, w], 0.3, 1.1)
        assert r == pytest.approx([math.sqrt(1 - 0.09) * math.cos(1.1), math.sqrt(1 - 0.09) * math.sin(1.1), 0.3 * w])
    # azimuth convention: phi and phi + pi are mirror images about d
    d = np.array([0.6, 0.0, 0.8])
    a, b = orc.rotate(d, 0.5, 0.7), orc.rotate(d, 0.5, 0.7 + np.pi)
    assert (a + b) / 2 == pytest.approx(0.5 * d, abs=1e-12)


def test_channel_frequencies_follow_partial_mu():
    # infinite homogeneous medium, energy-independent mu: PE 0.01, coherent 0.03 /mm -> every interaction is
    # PE with p = 1/4; coherent events per history are geometric with mean 3, variance 12; all histories peak
    w = dm.make_config(1)
    mu = np.zeros_like(w.mu); mu[1, 0, :] = 0.01; mu[1, 2, :] = 0.03
    v, t = _cyl(1e5, 1e5, -1e5, 16)
    s = _scene([("block", v, t, 1, 0)], mu, w.is_scoring, _beam(1500.0, pos=(1.2, 0.5, 1.0)))
    n = 20000
    edep, flags, cnt = s.run_histories(0, n, 6)
    assert ((flags & orc.F_PEAK) != 0).all()
    assert cnt["n_pe"] == n and cnt["n_compton"] == 0 and cnt["n_pair"] == 0
    assert abs(cnt["n_coherent"] / n - 3.0) < 4 * math.sqrt(12.0 / n)
    assert np.array_equal(flags >> 16, (flags >> 16))
    assert (flags >> 16).sum() == cnt["n_pe"] + cnt["n_coherent"]


# ------------------------------------------------------------------ P8 PE-only FEPE vs deterministic quadrature
def test_pe_only_fepe_config0_vs_chord_quadrature():
    w = dm.make_config(0, n_theta=256)
    mu = np.zeros_like(w.mu); mu[1, 0, :] = 0.02                # 1/mm, constant, PE only
    s = orc.OracleScene(w)
    s.set_materials(mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
    n = 4_000_000
    _, em, pk, _ = s.run(n, 3)
    R, L, h = 30.0, 60.0, 250.0
    x, wq = np.polynomial.legendre.leggauss(2000)
    th_max = math.atan(R / h)
    th = 0.5 * th_max * (x + 1)
    chord = np.minimum((h + L) / np.cos(th), R / np.maximum(np.sin(th), 1e-300)) - h / np.cos(th)
    fepe = 0.5 * (0.5 * th_max * wq * (1 - np.exp(-0.02 * chord)) * np.sin(th)).sum()
    # polygonal (N=256) vs smooth cylinder: relative difference ~1e-4, far below the statistical error
    assert abs(pk[0] / n - fepe) < 4 * math.sqrt(fepe / n) + 2e-4 * fepe


# ------------------------------------------------------------------ P9 pair structure
def test_pair_escape_peaks_at_e_minus_511_and_1022():
    w = dm.make_config(1)
    v, t = _cyl(30.0, 0.0, -60.0, 32)
    s = _scene([("ge", v, t, 1, 0)], w.mu, w.is_scoring, _beam(2800.0))
    n, nb, emax = 60_000, 3000, 3.0
    spec, em, pk, cnt = s.run(n, 2, n_bins=nb, e_max_mev=emax)
    assert cnt["n_pair"] > 100
    # P6 with secondaries: the two 0.511 MeV photons are part of the balance
    edep, flags, other, esc, c2 = s.run_histories(0, 5000, 2, details=True)
    assert c2["n_pair"] > 10
    dep_sc = np.where((flags & orc.F_PEAK) != 0, s.line_mev[0], edep)
    assert np.allclose(dep_sc + other + esc, s.line_mev[0], rtol=1e-12)
    de = emax / nb
    b_se, b_de = int((2.8 - MEC2) / de), int((2.8 - 2 * MEC2) / de)
    for b in (b_se, b_de):
        neigh = np.concatenate([spec[b - 6:b - 1], spec[b + 2:b + 7]]).astype(float).mean()
        assert spec[b] > 5 * (neigh + 1)


# ------------------------------------------------------------------ P11 statistics
def test_two_seeds_agree_statistically():
    w = dm.make_config(0)
    s = orc.OracleScene(w)
    n = 2_000_000
    sa, _, pa, _ = s.run(n, 1)
    sb, _, pb, _ = s.run(n, 2)
    sig = math.sqrt(float(pa[0] + pb[0]))
    assert abs(float(pa[0]) - float(pb[0])) < 4 * sig
    # rebin to 64 coarse bins and compare
    a = sa[:4096].reshape(64, 64).sum(1).astype(float); b = sb[:4096].reshape(64, 64).sum(1).astype(float)
    m = (a + b) >= 20
    chi2 = ((a[m] - b[m]) ** 2 / (a[m] + b[m])).sum() / m.sum()
    assert chi2 < 1.8


# ------------------------------------------------------------------ NEXT-4: straight CSDA electron segments (R16)
def test_electron_range_katz_penfold_values():
    # R = 412 T^(1.265 - 0.0954 ln T) mg/cm^2: at 1 MeV the exponent does not matter (412 mg/cm^2), at 0.5 MeV the
    # textbook value is 0.164 g/cm^2 (aluminium range tables: 0.16 - 0.17), the range scales with 1/density
    assert orc.electron_range_mm(1.0, 1.0) == pytest.approx(4.12, rel=1e-12)            # 412 mg/cm^2 = 4.12 mm of water
    assert orc.electron_range_mm(1.0, 5.323) == pytest.approx(4.12 / 5.323, rel=1e-12)
    assert orc.electron_range_mm(0.5, 1.0) == pytest.approx(1.637, rel=2e-3)
    assert orc.electron_range_mm(0.1, 1.0) == pytest.approx(0.1350, rel=2e-3)
    assert orc.electron_range_mm(0.0, 1.0) == 0.0 and orc.electron_range_mm(1.0, 0.0) == 0.0
    r = [orc.electron_range_mm(t, 2.7) for t in np.geomspace(0.01, 2.5, 40)]
    assert (np.diff(r) > 0).all()                                                        # monotonic in the energy


def test_electron_split_below_a_plane_face_matches_closed_form():
    # A point at depth d below the flat top of the bare Ge cylinder (config 0; the range is far below its radius).
    # Isotropic straight segments of length R, uniform energy loss: a direction with cosine c towards the face keeps
    # the fraction min(1, a / c), a = d / R, inside; averaged over the sphere: 1/2 + a (1 - ln a) / 2 for a < 1.
    w = dm.make_config(0)
    s = orc.OracleScene(w)
    s.set_electron_mode(dm.DENSITY_G_CM3)
    t_kin = 1.0
    R = orc.electron_range_mm(t_kin, 5.323)
    n = 40_000
    for a in (0.1, 0.35, 0.8):
        f = s.electron_split([0.3, -0.2, -a * R], dm.MAT["Ge_active"], t_kin, 5, 0, n)
        assert (f >= 0).all() and (f <= 1 + 1e-12).all()
        exact = 0.5 + 0.5 * a * (1.0 - math.log(a))
        # variance of the kept fraction is below 1/4
        assert f.mean() == pytest.approx(exact, abs=4 * 0.5 / math.sqrt(n)), (a, f.mean(), exact)
        assert (f < 1 - 1e-9).mean() == pytest.approx(0.5 * (1 - a), abs=4 * 0.5 / math.sqrt(n))   # solid angle of c > a
    f = s.electron_split([0.0, 0.0, -30.0], dm.MAT["Ge_active"], t_kin, 5, 0, 2000)      # deep inside: nothing leaves
    assert (f == 1.0).all()
    s.set_electron_mode(None)
    f = s.electron_split([0.0, 0.0, -0.1 * R], dm.MAT["Ge_active"], t_kin, 5, 0, 2000)   # mode off: local deposit
    assert (f == 1.0).all()


def test_electron_mode_leaves_the_photons_alone_and_only_removes_energy():
    # The electrons draw from their own stream: same photon trajectories, so per history the flags other than
    # PEAK / NONSCORING, the event count and the escaped energy are unchanged, and with a single scoring volume in
    # vacuum the scored energy can only go down.
    w = dm.make_config(0)
    s = orc.OracleScene(w)
    n = 600_000
    e0, f0, o0, x0, c0 = s.run_histories(0, n, w.seed, details=True)
    s.set_electron_mode(dm.DENSITY_G_CM3)
    e1, f1, o1, x1, c1 = s.run_histories(0, n, w.seed, details=True)
    keep = ~np.uint32(orc.F_PEAK | orc.F_NONSCORING)
    assert np.array_equal(f0 & keep, f1 & keep) and np.array_equal(x0, x1)
    for k in ("n_pe", "n_compton", "n_coherent", "n_pair", "n_crossings", "n_escaped"):
        assert c0[k] == c1[k]
    line = w.source["line_mev"][0]
    d0 = np.where(f0 & orc.F_PEAK, line, e0)
    d1 = np.where(f1 & orc.F_PEAK, line, e1)
    assert (d1 <= d0 + 1e-12).all()
    lost = d0 - d1
    assert (lost > 1e-9).sum() >= 5                          # some electrons do reach the surface (R = 0.5 mm at 662 keV)
    assert np.allclose(d1 + o1 + x1, d0 + o0 + x0, atol=1e-9)    # energy is moved between tallies, not created
    assert ((f1 & orc.F_PEAK) != 0).sum() < ((f0 & orc.F_PEAK) != 0).sum()
