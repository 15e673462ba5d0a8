"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element on the same seeded inputs.

Tolerances (BASELINE.json north_star):
  geometry  nearest-hit facet index bit-exact except where the two candidates tie within 1e-6 relative;
            |t_gpu - t_oracle| <= 1e-5 t + 8 ulp32(largest coordinate) / |cos(ray, facet normal)| (float32 inputs bound
            the absolute accuracy of the hit point; a grazing ray amplifies it by 1/cos)
  histories same Philox streams on both sides: >= 99.9 % of histories agree in flags and deposit (float32 decisions
            flip rarely); FEPE within 3 combined sigma and 0.5 % relative at >= 1e7; chi^2/dof <= 1.2
"""
import json
import math
import os

import numpy as np
import pytest

import detmesh as dm
from detmesh.configs import make_rays

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2605_25963_b200 as p
    return p


@pytest.fixture(scope="module")
def orc():
    from oracle import gadep_oracle
    return gadep_oracle


_cache = {}


def _setup(pkg, orc, cfg, **kw):
    key = (cfg, tuple(sorted(kw.items())))
    if key not in _cache:
        w = dm.make_config(cfg, **kw)
        g = pkg.Gadep(0)
        g.load_workload(w)
        _cache[key] = (w, g, orc.OracleScene(w))
    return _cache[key]


def _ulp32(x):
    return float(np.spacing(np.float32(abs(x))))


# ------------------------------------------------------------------ RNG
def test_philox_device_vs_curand_and_oracle(pkg, orc):
    g = pkg.Gadep(0)
    rng = np.random.default_rng(0)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2),
             ([0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [0xA4093822, 0x299F31D0])]
    cases += [(list(rng.integers(0, 2 ** 32, 4)), list(rng.integers(0, 2 ** 32, 2))) for _ in range(20)]
    for ctr, key in cases:
        mine = g.philox_raw(ctr, key, 0)
        curand = g.philox_raw(ctr, key, 1)          # curand_Philox4x32_10 device routine
        assert np.array_equal(mine, curand)
        assert np.array_equal(mine, orc.philox(ctr, key))
    assert list(g.philox_raw([0, 0, 0, 0], [0, 0], 1)) == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]


# ------------------------------------------------------------------ geometry
def _check_rays(w, g, s, org, d, filter_mat=-2, t_min=0.0):
    tri, t = g.trace_rays(org, d, filter_mat, t_min)
    otri, ot = s.trace_rays(org, d, filter_mat, t_min)
    coord = float(np.abs(w.mesh.vertices).max())
    hit = otri >= 0
    # misses agree exactly, except grazing hits at the float32 resolution of an edge / silhouette
    miss_mismatch = np.nonzero((tri >= 0) != hit)[0]
    assert len(miss_mismatch) <= 2e-5 * len(tri) + 1, len(miss_mismatch)
    both = hit & (tri >= 0)
    # conditioning: a position error of a few ulp32(coordinate) moves t by that / |cos(angle to the facet normal)|
    v = w.mesh.vertices.astype(np.float64)
    f = w.mesh.triangles[otri[both]]
    nrm = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    cosang = np.maximum(np.abs(np.einsum("ij,ij->i", nrm, d[both].astype(np.float64))), 1e-7)
    tol = 1e-5 * np.abs(ot[both]) + 8 * _ulp32(coord) / cosang
    err = np.abs(t[both].astype(np.float64) - ot[both])
    assert (err <= tol).all(), (err / tol).max()
    diff = np.nonzero(both & (tri != otri))[0]
    for i in diff:      # allowed only for ties: the GPU's facet lies at the same distance in the oracle's arithmetic
        o64, d64 = org[i].astype(np.float64), d[i].astype(np.float64)
        p = v[w.mesh.triangles[tri[i]]]
        nn = np.cross(p[1] - p[0], p[2] - p[0])
        cs = max(abs(float(nn @ d64) / float(np.linalg.norm(nn))), 1e-7)
        floor = 8 * _ulp32(coord) / cs
        ok, tt, _ = s.ray_triangle(int(tri[i]), o64, d64)
        if not ok:      # the ray passes through a shared edge / vertex: the oracle's edge-inclusive test gives the
            # edge to the neighbour.  Accept if the GPU facet's plane is met at the same t and the hit point lies
            # within the float32 resolution of that facet.
            tt = float(nn @ (p[0] - o64)) / float(nn @ d64)
            q = o64 + tt * d64
            bary = [float(np.cross(p[(k + 1) % 3] - p[k], q - p[k]) @ nn) / float(nn @ nn) for k in range(3)]
            assert min(bary) >= -1e-5, (i, tri[i], otri[i], bary)
        assert abs(tt - ot[i]) <= 1e-6 * abs(ot[i]) + floor, (i, tri[i], otri[i], tt, ot[i])
    return len(diff), int(both.sum())


@pytest.mark.parametrize("cfg,n_rays,box", [(0, 1_000_000, (45.0, -80.0, 20.0)), (1, 200_000, (45.0, -105.0, 10.0)),
                                            (3, 60_000, (60.0, -235.0, 45.0))])
def test_nearest_hit_vs_brute_force(pkg, orc, cfg, n_rays, box):
    w, g, s = _setup(pkg, orc, cfg)
    org, d = make_rays(n_rays, 1, *box)
    n_tie, n_hit = _check_rays(w, g, s, org, d)
    assert n_hit > 0.5 * n_rays or cfg == 0
    assert n_tie <= 1e-4 * n_rays + 2
    c = g.get_counters()
    assert c["n_queries"] == n_rays and c["n_tri_tests"] > 0 and c["n_box_tests"] > 0


def test_nearest_hit_config4_instance_and_device_pointers(pkg, orc):
    import torch
    w, g, s = _setup(pkg, orc, 4, n_theta=512, total_bands=128)      # ~125 k facets, same recipe as configs[4]
    assert w.mesh.n_tri > 100_000
    r, z0, z1 = w.notes["ray_box"]
    org, d = make_rays(40_000, w.notes["ray_seed"], r, z0, z1)
    _check_rays(w, g, s, org, d)
    # device-resident inputs / outputs (torch is only memory here)
    o_t, d_t = torch.from_numpy(org).cuda(), torch.from_numpy(d).cuda()
    tri_t = torch.empty(len(org), dtype=torch.int32, device="cuda")
    t_t = torch.empty(len(org), dtype=torch.float32, device="cuda")
    g.trace_rays(o_t, d_t, tri_out=tri_t, t_out=t_t)
    tri_h, t_h = g.trace_rays(org, d)
    assert np.array_equal(tri_t.cpu().numpy(), tri_h) and np.array_equal(t_t.cpu().numpy(), t_h)


def test_cfg4_full_size_rays(pkg, orc):
    # BASELINE.json configs[4] at full size (2 M facets, BVH built from scratch): 1e6 seeded rays on the GPU, a sample
    # of them against the oracle's brute force over all facets; properties that hold at any size on the rest.
    w, g, s = _setup(pkg, orc, 4)
    assert w.mesh.n_tri > 2_000_000
    r, z0, z1 = w.notes["ray_box"]
    org, d = make_rays(1_000_000, w.notes["ray_seed"], r, z0, z1)
    tri, t = g.trace_rays(org, d)
    # every origin lies inside the closed world surface: every ray hits something, at a finite positive distance
    assert (tri >= 0).all() and (tri < w.mesh.n_tri).all() and np.isfinite(t).all() and (t > 0).all()
    k = 6_000
    _check_rays(w, g, s, org[:k], d[:k])


@pytest.mark.parametrize("cfg,n", [(1, 4000), (3, 2000)])
def test_localisation_side_id_and_parity_rules(pkg, orc, cfg, n):
    # the original side-id rule and the reworked parity rule (all-hits traversal) must name the same
    # material for every point, and both must agree with the oracle's brute-force versions of the two rules.
    w, g, s = _setup(pkg, orc, cfg)
    r, z0, z1 = (45.0, -105.0, 10.0) if cfg == 1 else (60.0, -235.0, 45.0)
    org, d = make_rays(n, 11, r, z0, z1)
    m_side = g.locate(org, d, 0)
    c0 = g.get_counters()
    m_par = g.locate(org, d, 1)
    c1 = g.get_counters()
    o_side = np.array([s.locate_sideid(org[i].astype(np.float64), d[i].astype(np.float64)) for i in range(n)])
    o_par = np.array([s.locate_parity(org[i].astype(np.float64), d[i].astype(np.float64)) for i in range(n)])
    assert (m_par != -3).all()                               # no ray met more facets than the hit list holds
    # a ray through an edge or vertex is counted twice by any edge-inclusive test: allow a handful of such rays
    for a, b in ((m_side, o_side), (m_par, o_par), (m_side, m_par)):
        assert (a != b).sum() <= 2 + 1e-3 * n, int((a != b).sum())
    assert set(np.unique(m_par)) <= set(range(len(w.is_scoring)))
    assert len(np.unique(m_par)) >= 5                        # the sample really visits the nested regions
    # the all-hits traversal visits more of the hierarchy than the nearest-hit one
    assert c1["n_box_tests"] >= c0["n_box_tests"] and c1["n_tri_tests"] >= c0["n_tri_tests"]


@pytest.mark.parametrize("cfg,n", [(1, 300_000), (3, 20_000)])
def test_transport_with_parity_localisation(pkg, orc, cfg, n):
    # GADEP_RUN_PARITY_LOCALISATION: the material after the start and after every crossing comes from the paper's parity
    # rule instead of the facet's side ids.  On a valid mesh the two rules name the same medium, so the
    # tallies must coincide except for the rare rays through an edge, which the counters report.
    from paper_2605_25963_b200.binding import RUN_HISTORY_PER_THREAD, RUN_PARITY_LOCALISATION
    w, g, s = _setup(pkg, orc, cfg)
    a = g.run(n, 3, w.n_bins, w.spectrum_e_max_mev, flags=RUN_HISTORY_PER_THREAD).copy()
    ca = g.get_counters()
    b = g.run(n, 3, w.n_bins, w.spectrum_e_max_mev, flags=RUN_PARITY_LOCALISATION).copy()
    cb = g.get_counters()
    assert cb["n_parity_queries"] >= n and cb["n_parity_mismatch"] <= 2e-5 * cb["n_parity_queries"] + 2
    assert ca["n_parity_queries"] == 0
    assert abs(int(a.sum()) - int(b.sum())) <= 5 * cb["n_parity_mismatch"] + 2
    assert np.abs(a.astype(np.int64) - b.astype(np.int64)).sum() <= 10 * cb["n_parity_mismatch"] + 4
    assert sum(cb["emitted"]) == n and cb["n_box_tests"] > ca["n_box_tests"]


def test_partial_cross_section_method_is_statistically_equivalent(pkg, orc):
    # GADEP_RUN_PARTIAL_XS: per-process optical-depth budgets instead of total-mu sampling + a selection
    # draw.  Different random streams, same distribution: 1e7 histories of config 1 against the stored oracle run
    # (total-mu method): FEPE per line within 3 combined standard errors, chi2/dof of the spectra <= 1.2.
    from paper_2605_25963_b200.binding import RUN_PARTIAL_XS
    path = os.path.join(GOLDEN, "cfg1_oracle_n10000000.json")
    if not os.path.exists(path):
        pytest.skip("stored oracle result not generated")
    gold = json.load(open(path))
    w, g, s = _setup(pkg, orc, 1)
    n = gold["n_histories"]
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"], flags=RUN_PARTIAL_XS)
    c = g.get_counters()
    assert sum(c["emitted"]) == n and c["emitted"] == gold["emitted"][:c["n_lines"]]      # the line draw is unchanged
    for l in range(c["n_lines"]):
        f, se = g.fepe(l, 0)
        fo = gold["peak"][l] / gold["emitted"][l]
        so = math.sqrt(max(fo * (1 - fo), 0) / gold["emitted"][l])
        assert abs(f - fo) <= 3 * math.sqrt(se * se + so * so) + 1e-12, (l, f, fo)
    chi2, dof = _chi2_dof(spec[:-1], n, np.array(gold["spectrum"][:-1]), n)
    assert dof > 10 and chi2 <= 1.2, (chi2, dof)
    # event mix within statistics of the oracle's
    oc = gold["counters"]
    for k in ("n_pe", "n_compton", "n_coherent"):
        assert abs(c[k] - oc[k]) <= 5 * math.sqrt(oc[k]) + 0.01 * oc[k], (k, c[k], oc[k])


def test_calibration_sweep_and_resolution_broadening(pkg, orc):
    # SURVEY.md 8(f) NEXT-3 (Table 3): 13 calibration energies from a point source 250 mm above a
    # parametric coaxial detector in one launch -> FEPE curve; Gaussian broadening against the numpy definition.
    from oracle.broaden import broaden
    w = dm.make_calibration(1, n_histories=2_000_000)
    g = pkg.Gadep(0)
    g.load_workload(w)
    spec = g.run(w.n_histories, w.seed, w.n_bins, w.spectrum_e_max_mev)
    c = g.get_counters()
    assert c["n_lines"] == 13 and sum(c["emitted"]) == w.n_histories and c["n_leak"] == 0
    fepe = np.array([g.fepe(l)[0] for l in range(13)])
    e = np.array(dm.TABLE3_KEV)
    # with the literal coherent constant of reading Q1 the curve is not the textbook one (low energies scatter away);
    # what must hold: every efficiency lies below the geometric solid-angle fraction of the crystal, the lowest
    # energies are the smallest, and the values are those of the oracle (below)
    p = w.notes["detector"]
    h = float(w.source["pos"][2])
    omega = 0.5 * (1.0 - h / math.hypot(h, p["R"]))
    assert (fepe >= 0).all() and (fepe < omega).all() and fepe[:2].max() < fepe[3:].min()
    assert len(e) == 13
    # same streams in the oracle on a sample: identical per-line peak counts up to float32 decision flips
    s = orc.OracleScene(w)
    n_s = 60_000
    oe, of, oc = s.run_histories(0, n_s, w.seed)
    ge, gf = g.run_histories(0, n_s, w.seed)
    assert ((gf == of) & (np.abs(ge - oe) <= 2e-6 + 1e-5 * oe)).mean() >= 0.999
    # broadening: total conserved, matches the float64 definition
    g.run(w.n_histories, w.seed, w.n_bins, w.spectrum_e_max_mev)
    a, b = (0.0012 / 1.0) ** 2, 2.0e-6          # FWHM 1.2 keV at 0, ~1.9 keV at 1.33 MeV
    got = g.broaden(a, b)
    want = broaden(spec, w.spectrum_e_max_mev, a, b)
    assert abs(got.sum() - float(spec.sum())) <= 1e-6 * spec.sum()
    assert np.abs(got - want).max() <= 1e-9 * spec.max() + 1e-9
    assert got[int(e[11] / 1e3 / (2.0 / 4096))] < spec[int(e[11] / 1e3 / (2.0 / 4096))]   # the 1332 keV peak is spread out


def test_filtered_trace_with_negative_window(pkg, orc):
    w, g, s = _setup(pkg, orc, 1)
    org, d = make_rays(60_000, 5, 36.0, -72.0, 1.0)
    for mat in (dm.MAT["Ge_active"], dm.MAT["Ge_dead"], dm.MAT["vacuum"]):
        _check_rays(w, g, s, org, d, filter_mat=mat, t_min=-1e-4)


@pytest.mark.parametrize("n_pellets", [6, 12, 300])
def test_material_entry_table_and_its_fallbacks(pkg, orc, n_pellets):
    # The clustered hierarchy starts a flight at the subtrees of the surfaces around its material.  6 pellets: every
    # material has an entry list (air: 7 surfaces).  12 pellets: air touches 13 surfaces, more than the table holds ->
    # root for air, entry lists for the pellet materials.  300 pellets: more surfaces than class bits -> plain order.
    # In every case filtered and unfiltered rays and whole histories must agree with the oracle.
    w = dm.make_pellet_stack(n_pellets)
    g = pkg.Gadep(0)
    g.load_workload(w)
    s = orc.OracleScene(w)
    assert dm.check_closed_oriented(w.mesh.triangles)["ok"]
    r, z0, z1 = w.notes["ray_box"]
    n_rays = 20_000 if n_pellets < 100 else 3_000
    org, d = make_rays(n_rays, 11, r, z0, z1)
    _check_rays(w, g, s, org, d)
    for mat in (dm.MAT["air"], dm.MAT["Ge_active"], dm.MAT["Cu"], dm.MAT["water"]):
        _check_rays(w, g, s, org, d, filter_mat=mat, t_min=-1e-4)
    n = 20_000 if n_pellets < 100 else 2_000
    edep, flags = g.run_histories(0, n, w.seed)
    oe, of, oc = s.run_histories(0, n, w.seed)
    same = (flags == of) & (np.abs(edep.astype(np.float64) - oe) <= 2e-6 + 1e-5 * oe)
    assert same.mean() >= 0.998, same.mean()
    c = g.get_counters()
    assert c["n_leak"] == 0 and oc["n_leak"] == 0
    for k in ("n_crossings", "n_pe", "n_compton", "n_coherent", "n_escaped"):
        assert abs(c[k] - oc[k]) <= 0.01 * oc[k] + 20, (k, c[k], oc[k])


# ------------------------------------------------------------------ histories, same random streams
@pytest.mark.parametrize("cfg,n", [(0, 400_000), (1, 40_000), (2, 6_000), (3, 6_000)])
def test_per_history_parity(pkg, orc, cfg, n):
    w, g, s = _setup(pkg, orc, cfg)
    edep, flags = g.run_histories(0, n, w.seed)
    c = g.get_counters()
    oe, of, oc = s.run_histories(0, n, w.seed)
    same = (flags == of) & (np.abs(edep.astype(np.float64) - oe) <= 2e-6 + 1e-5 * oe)
    # a float32 decision flips with probability ~1e-5 per event and the trajectory then diverges: 99.9 % for the
    # point-source set-ups (few events per history), 99.5 % for the volume sources (~150 events per history)
    assert same.mean() >= (0.999 if cfg < 2 else 0.995), same.mean()
    assert c["n_leak"] == 0 and oc["n_leak"] == 0
    assert (edep <= w.source["line_mev"][(flags >> 8) & 0xFF] * (1 + 1e-6)).all()      # deposit <= source energy
    # event totals track the oracle's to the fraction of diverged histories
    c = dict(c)
    # the first flight of every history is a query the oracle makes; the CUDA path answers it with the ray of the
    # start localisation
    c["n_queries"] += c["n_skipped_queries"] + n
    for k in ("n_queries", "n_crossings", "n_pe", "n_compton", "n_coherent", "n_escaped"):
        assert abs(c[k] - oc[k]) <= 0.01 * oc[k] + 50, (k, c[k], oc[k])
    assert c["n_pair"] == pytest.approx(oc["n_pair"], abs=3 + 0.05 * oc["n_pair"])
    # FEPE per line on this sample: identical counts up to the diverged histories
    line = (of >> 8) & 0xFF
    for l in range(len(w.source["line_mev"])):
        pg = int(((flags & 2) != 0)[((flags >> 8) & 0xFF) == l].sum())
        po = int(((of & 2) != 0)[line == l].sum())
        assert abs(pg - po) <= 3 + 0.01 * po


@pytest.mark.parametrize("scene,n", [("cfg0", 400_000), ("cfg1", 40_000), ("pellets", 40_000)])
def test_electron_range_mode_per_history_parity(pkg, orc, scene, n):
    # deposits as straight electron segments of the Katz-Penfold range.  The
    # electrons draw from their own Philox stream, so the photon side is the per-history parity above; here the split
    # of every deposit at the first facet must agree too (float32 range and hit distance against double).
    from paper_2605_25963_b200.binding import RUN_ELECTRON_RANGE
    w = dm.make_pellet_stack(9, n_histories=n) if scene == "pellets" else dm.make_config(int(scene[3]))
    g = pkg.Gadep(0)
    g.load_workload(w)
    s = orc.OracleScene(w)
    with pytest.raises(pkg.GadepError) as e:                      # densities first
        g.run_histories(0, 10, w.seed, flags=RUN_ELECTRON_RANGE)
    assert e.value.code == -2
    g.set_densities(dm.DENSITY_G_CM3)
    s.set_electron_mode(dm.DENSITY_G_CM3)
    edep0, flags0 = g.run_histories(0, n, w.seed)                 # local deposit, default kernel
    edep, flags = g.run_histories(0, n, w.seed, flags=RUN_ELECTRON_RANGE)
    c = g.get_counters()
    oe, of, oc = s.run_histories(0, n, w.seed)
    same = (flags == of) & (np.abs(edep.astype(np.float64) - oe) <= 2e-6 + 1e-5 * oe)
    assert same.mean() >= 0.999, same.mean()
    for k in ("n_queries", "n_crossings", "n_pe", "n_compton", "n_coherent", "n_escaped"):
        assert abs(c[k] + (n if k == "n_queries" else 0) - oc[k]) <= 0.01 * oc[k] + 50, (k, c[k], oc[k])
    # against the local-deposit run of the same histories: same photons (event count, line, escape bit) ...
    keep = ~np.uint32(2 | 8)
    assert np.array_equal(flags & keep, flags0 & keep)
    # ... and electrons that leave the scoring volume do show up
    changed = (np.abs(edep - edep0) > 1e-6) | ((flags ^ flags0) & 2 != 0)
    assert changed.sum() >= 3, changed.sum()
    if scene == "cfg0":                                           # one volume in vacuum: energy can only be lost
        line = w.source["line_mev"][(flags >> 8) & 0xFF]
        assert (edep <= edep0 + 1e-6).all() and (edep <= line * (1 + 1e-6)).all()
    # the spectrum of gadep_run in this mode is the histogram of the dump
    spec = g.run(n, w.seed, w.n_bins, w.spectrum_e_max_mev, flags=RUN_ELECTRON_RANGE)
    de = w.spectrum_e_max_mev / w.n_bins
    line, peak = (flags >> 8) & 0xFF, (flags & 2) != 0
    bins = np.minimum(np.floor(np.float32(edep) * np.float32(w.n_bins / w.spectrum_e_max_mev)).astype(np.int64), w.n_bins)
    lb = np.minimum(np.floor(w.source["line_mev"].astype(np.float64) / de).astype(np.int64), w.n_bins)
    bins[peak] = lb[line[peak]]
    ref = np.bincount(bins[edep.astype(np.float64) > 0], minlength=w.n_bins + 1)
    assert np.array_equal(ref.astype(np.uint64), spec)


def test_run_spectrum_equals_histogram_of_history_dump(pkg, orc):
    w, g, s = _setup(pkg, orc, 1)
    n = 200_000
    edep, flags = g.run_histories(0, n, 3)
    spec = g.run(n, 3, w.n_bins, w.spectrum_e_max_mev)
    c = g.get_counters()
    assert c["n_histories"] == n and sum(c["emitted"]) == n
    line = (flags >> 8) & 0xFF
    peak = (flags & 2) != 0
    for l in range(c["n_lines"]):
        assert c["emitted"][l] == int((line == l).sum()) and c["peak"][l] == int((peak & (line == l)).sum())
    de = w.spectrum_e_max_mev / w.n_bins
    e = edep.astype(np.float64)
    bins = np.minimum(np.floor(np.float32(edep) * np.float32(w.n_bins / w.spectrum_e_max_mev)).astype(np.int64), w.n_bins)
    lb = np.minimum(np.floor(w.source["line_mev"].astype(np.float64) / de).astype(np.int64), w.n_bins)
    bins[peak] = lb[line[peak]]
    ref = np.bincount(bins[(e > 0)], minlength=w.n_bins + 1)
    assert np.array_equal(ref.astype(np.uint64), spec)
    for l in range(c["n_lines"]):
        f, se = g.fepe(l, 0)
        assert f == pytest.approx(c["peak"][l] / c["emitted"][l])


def _chi2_dof(a, na, b, nb):
    a, b = a.astype(np.float64), b.astype(np.float64)
    m = (a + b) >= 20
    num = (a[m] / na - b[m] / nb) ** 2
    den = a[m] / na ** 2 + b[m] / nb ** 2
    return float((num / den).sum() / m.sum()), int(m.sum())


@pytest.mark.parametrize("cfg", [0, 1])
def test_full_size_fepe_and_spectrum_vs_stored_oracle(pkg, orc, cfg):
    path = os.path.join(GOLDEN, f"cfg{cfg}_oracle_n10000000.json")
    if not os.path.exists(path):
        pytest.skip("stored oracle result not generated")
    gold = json.load(open(path))
    w, g, s = _setup(pkg, orc, cfg)
    n = gold["n_histories"]
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"])
    c = g.get_counters()
    assert c["emitted"] == gold["emitted"][:c["n_lines"]] or sum(abs(a - b) for a, b in zip(c["emitted"], gold["emitted"])) <= 4
    for l in range(c["n_lines"]):
        f, se = g.fepe(l, 0)
        fo = gold["peak"][l] / gold["emitted"][l]
        so = math.sqrt(max(fo * (1 - fo), 0) / gold["emitted"][l])
        assert abs(f - fo) <= 3 * math.sqrt(se * se + so * so) + 1e-12
        if fo > 0:
            assert abs(f - fo) <= 0.005 * fo + 2.0 / gold["emitted"][l]
    chi2, dof = _chi2_dof(spec[:-1], n, np.array(gold["spectrum"][:-1]), n)
    assert dof > 10 and chi2 <= 1.2, (chi2, dof)


@pytest.mark.parametrize("cfg", [2, 3])
def test_headline_size_volume_sources_vs_stored_oracle(pkg, orc, cfg):
    # BASELINE.json configs[2], [3]: 1e8 histories on the GPU (the launch bench.py times) against the stored oracle run
    # of the same workload at the size the oracle can afford (independent sample sizes, same seed): FEPE per line
    # within 3 combined standard errors, chi2/dof of the normalised spectra <= 1.2, and the exact invariants.
    import glob
    files = sorted(glob.glob(os.path.join(GOLDEN, f"cfg{cfg}_oracle_n*.json")))
    if not files:
        pytest.skip("stored oracle result not generated")
    gold = max((json.load(open(f)) for f in files), key=lambda d: d["n_histories"])
    w, g, s = _setup(pkg, orc, cfg)
    n = w.n_histories
    assert n == 100_000_000
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"])
    c = g.get_counters()
    assert sum(c["emitted"]) == n == c["n_histories"]
    assert c["n_leak"] <= 20        # float32 corner cases that needed a second localisation: ~1e-8 per history
    assert int(spec.sum()) <= n and all(p <= e for p, e in zip(c["peak"], c["emitted"]))
    z = []
    for l in range(c["n_lines"]):
        f, se = g.fepe(l, 0)
        fo = gold["peak"][l] / gold["emitted"][l]
        so = math.sqrt(max(fo * (1 - fo), 1.0 / gold["emitted"][l]) / gold["emitted"][l])
        z.append((f - fo) / math.sqrt(se * se + so * so))
        # the emission frequencies follow the line intensities
        assert abs(c["emitted"][l] / n - gold["emitted"][l] / gold["n_histories"]) <= 4 * math.sqrt(0.25 / gold["n_histories"])
    # north_star: FEPE per line within 3 combined standard errors.  The two samples are independent here, so with L
    # lines a correct implementation leaves the 3-sigma band on some line with probability 0.0027 L (11 % for the 40
    # lines of config 3): the family of lines is held to "at most one line of >= 20 beyond 3 sigma, none beyond 4, and
    # the mean z^2 within 3 standard deviations of its expectation 1".  The same stored run is
    # compared history by history, far below its statistical error, in test_gpu_acceptance.py.
    z = np.array(z)
    L = len(z)
    assert int((np.abs(z) > 3.0).sum()) <= (1 if L >= 20 else 0), z
    assert np.abs(z).max() <= 4.0, z
    assert float((z * z).mean()) <= 1.0 + 3.0 * math.sqrt(2.0 / L), (float((z * z).mean()), z)
    # sample sizes differ by 500-1000x: the per-bin variance comes from the pooled rate, not from the sparse bin itself
    # (and the spectrum is re-binned 32:1 so that the oracle's few thousand scoring histories populate the bins)
    a = spec[:-1].astype(np.float64).reshape(-1, 32).sum(axis=1)
    b = np.array(gold["spectrum"][:-1], dtype=np.float64).reshape(-1, 32).sum(axis=1)
    na, nb = float(n), float(gold["n_histories"])
    m = (a + b) * nb / (na + nb) >= 5.0                 # expected oracle count of the bin >= 5
    p = (a[m] + b[m]) / (na + nb)
    chi2 = float((((a[m] / na - b[m] / nb) ** 2) / (p * (1 / na + 1 / nb))).sum() / m.sum())
    assert m.sum() > 10 and chi2 <= 1.2, (chi2, int(m.sum()))


def test_headline_size_config4_vs_coarser_tessellation_oracle(pkg, orc):
    # BASELINE.json configs[4] (2 M facets, 1e8 histories).  The oracle's brute force cannot afford that mesh, so the
    # stored oracle run uses the same geometry recipe at 512 x 128 segments (125 k facets): the two tessellations
    # inscribe the same surfaces to 2e-5 relative in radius, far below the statistical error of the oracle sample.
    import glob
    files = sorted(glob.glob(os.path.join(GOLDEN, "cfg4_oracle_n*_nt512_b128.json")))
    if not files:
        pytest.skip("stored oracle result not generated")
    gold = max((json.load(open(f)) for f in files), key=lambda d: d["n_histories"])
    w, g, s = _setup(pkg, orc, 4)
    n = w.n_histories
    assert n == 100_000_000 and w.mesh.n_tri > 2_000_000
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"])
    c = g.get_counters()
    assert sum(c["emitted"]) == n == c["n_histories"] and c["n_leak"] <= 20
    f, se = g.fepe(0, 0)
    fo = gold["peak"][0] / gold["emitted"][0]
    so = math.sqrt(fo * (1 - fo) / gold["emitted"][0])
    assert abs(f - fo) <= 3 * math.sqrt(se * se + so * so) + 1e-3 * fo, (f, fo, so)
    a = spec[:-1].astype(np.float64).reshape(-1, 32).sum(axis=1)
    b = np.array(gold["spectrum"][:-1], dtype=np.float64).reshape(-1, 32).sum(axis=1)
    na, nb = float(n), float(gold["n_histories"])
    m = (a + b) * nb / (na + nb) >= 5.0
    p = (a[m] + b[m]) / (na + nb)
    chi2 = float((((a[m] / na - b[m] / nb) ** 2) / (p * (1 / na + 1 / nb))).sum() / m.sum())
    assert m.sum() > 10 and chi2 <= 1.2, (chi2, int(m.sum()))


# ------------------------------------------------------------------ invariants at any size / launch shape
def test_results_do_not_depend_on_partitioning_and_are_deterministic(pkg, orc):
    w, g, s = _setup(pkg, orc, 1)
    n = 300_000
    a = g.run(n, 9, w.n_bins, w.spectrum_e_max_mev).copy()
    b = g.run(n, 9, w.n_bins, w.spectrum_e_max_mev).copy()
    assert np.array_equal(a, b)
    p1 = g.run(100_000, 9, w.n_bins, w.spectrum_e_max_mev, first_history=0).copy()
    p2 = g.run(200_000, 9, w.n_bins, w.spectrum_e_max_mev, first_history=100_000, flags=pkg.binding.RUN_ACCUMULATE).copy()
    assert np.array_equal(a, p2) and not np.array_equal(a, p1)


def test_all_kernel_variants_give_identical_tallies(pkg, orc):
    # warp-resident wavefront (default) vs persistent lanes vs plain history-per-thread: same streams, integer
    # tallies -> bit-identical spectra and event counts.  The wavefront kernel uses an FMA slab test with its own
    # conservative padding, so only its box / triangle test counts may differ.
    from paper_2605_25963_b200.binding import RUN_BVH8, RUN_HISTORY_PER_THREAD, RUN_PERSISTENT_LANES
    for cfg, n in ((1, 400_000), (3, 20_000)):
        w, g, s = _setup(pkg, orc, cfg)
        a = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev).copy()
        ca = g.get_counters()
        b = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev, flags=RUN_HISTORY_PER_THREAD).copy()
        cb = g.get_counters()
        c = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev, flags=RUN_PERSISTENT_LANES).copy()
        cc = g.get_counters()
        d = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev, flags=RUN_BVH8).copy()      # compressed 8-wide nodes
        cd = g.get_counters()
        assert np.array_equal(a, d)
        g.set_bvh_width(5)                                                          # compressed 4-wide nodes (64 bytes)
        e = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev).copy()
        ce = g.get_counters()
        g.set_bvh_width(4)
        assert np.array_equal(a, e)
        for k in ("n_histories", "n_queries", "n_skipped_queries", "n_crossings", "n_pe", "n_compton", "n_coherent",
                  "n_pair", "n_escaped", "n_leak", "n_cutoff", "emitted", "peak"):
            assert ca[k] == ce[k], k
        for k in ("n_histories", "n_queries", "n_crossings", "n_pe", "n_compton", "n_coherent",
                  "n_pair", "n_escaped", "n_leak", "n_cutoff", "emitted", "peak"):
            assert ca[k] == cd[k], k
        assert ca["n_stack_overflow"] == 0
        assert np.array_equal(a, b) and np.array_equal(a, c)
        for k in ("n_histories", "n_crossings", "n_pe", "n_compton", "n_coherent",
                  "n_pair", "n_escaped", "n_leak", "n_cutoff", "emitted", "peak"):
            assert ca[k] == cb[k] == cc[k], k
        for k in ("n_queries", "n_box_tests", "n_tri_tests"):
            assert cb[k] == cc[k], k
        assert ca["n_queries"] + ca["n_skipped_queries"] == cb["n_queries"]
        assert ca["n_box_tests"] <= 1.25 * cb["n_box_tests"] and ca["n_tri_tests"] <= 1.25 * cb["n_tri_tests"]
        assert ca["n_histories"] == n


def test_clearance_grid_plane_lists_change_no_result(pkg, orc, monkeypatch):
    # The plane lists of the clearance grid only decide *which* flights are answered without a BVH query: tallies, event
    # counts and the number of flights are those of a run without lists (and of the grid-free kernels, test above).
    # Build flags: lists with the build, never, or (0) by the size of the first run.
    from paper_2605_25963_b200.binding import BUILD_NO_PLANE_LISTS, BUILD_PLANE_LISTS
    for cfg, n in ((2, 60_000), (3, 30_000)):
        w = dm.make_config(cfg)
        res = {}
        for name, flags in (("lists", BUILD_PLANE_LISTS), ("none", BUILD_NO_PLANE_LISTS)):
            g = pkg.Gadep(0)
            g.load_workload(w, build_flags=flags)
            c0 = g.get_counters()
            assert (c0["n_grid_lists"] > 0) == (name == "lists")
            spec = g.run(n, 11, w.n_bins, w.spectrum_e_max_mev).copy()
            res[name] = (spec, g.get_counters())
        (sa, ca), (sb, cb) = res["lists"], res["none"]
        assert cb["n_grid_lists"] == 0 and ca["n_grid_lists"] <= ca["n_grid_list_cells"]
        assert np.array_equal(sa, sb)
        for k in ("n_histories", "n_crossings", "n_pe", "n_compton", "n_coherent", "n_pair", "n_escaped", "n_leak",
                  "n_cutoff", "emitted", "peak"):
            assert ca[k] == cb[k], k
        assert ca["n_queries"] + ca["n_skipped_queries"] == cb["n_queries"] + cb["n_skipped_queries"]
        assert ca["n_queries"] < 0.8 * cb["n_queries"]            # the lists answer the tiny steps beside walls
    # flags 0: a small run makes no lists, a run of at least the threshold does (threshold lowered for the test)
    w = dm.make_config(2)
    monkeypatch.setenv("GADEP_LIST_MIN_HISTORIES", "50000")
    g = pkg.Gadep(0)
    g.load_workload(w)
    g.run(20_000, 11, w.n_bins, w.spectrum_e_max_mev)
    assert g.get_counters()["n_grid_lists"] == 0
    g.run(50_000, 11, w.n_bins, w.spectrum_e_max_mev)
    assert g.get_counters()["n_grid_lists"] > 0
    g.build_bvh()                                                 # a new build starts without lists again
    assert g.get_counters()["n_grid_lists"] == 0


def test_many_warp_instance_gives_identical_tallies(pkg, orc, monkeypatch):
    # the 28-warp x 72-register instance of the wavefront kernel (chosen for hierarchies far larger than the L2; forced
    # here on a small one) against the 12-warp default: same streams, integer tallies
    w = dm.make_config(3)
    res = []
    for threads in ("384", "896"):
        monkeypatch.setenv("GADEP_WAVE_THREADS", threads)
        g = pkg.Gadep(0)
        g.load_workload(w)
        res.append((g.run(40_000, 9, w.n_bins, w.spectrum_e_max_mev).copy(), g.get_counters()))
    (sa, ca), (sb, cb) = res
    assert np.array_equal(sa, sb)
    for k in ("n_histories", "n_queries", "n_skipped_queries", "n_crossings", "n_pe", "n_compton", "n_coherent", "n_pair",
              "n_escaped", "n_leak", "n_cutoff", "emitted", "peak", "n_box_tests", "n_tri_tests"):
        assert ca[k] == cb[k], k


def test_slab_transmission_on_gpu(pkg, orc):
    # closed form directly on the CUDA path: P(no event) = exp(-mu_tot x) through 10 mm Ge at 661.7 keV = 0.693573
    from detmesh.geometry import Line, discretise, merge_surfaces, revolve
    w0 = dm.make_config(0)
    v, t = revolve(discretise([Line(0, 0, 100, 0, 1), Line(100, 0, 100, -10, 1), Line(100, -10, 0, -10, 1)]), 32)
    mesh = merge_surfaces([("slab", v, t, 1, 0)], 0)
    g = pkg.Gadep(0)
    g.set_materials(w0.mu, w0.is_scoring, w0.e_min_mev, w0.e_max_mev)
    g.load_mesh(mesh.vertices, mesh.triangles, mesh.tri_surface, mesh.surf_inside, mesh.surf_outside, 0)
    g.build_bvh()
    g.set_source(2, pos=(1.234, 0.567, 50.0), dir=(0, 0, -1), line_mev=[0.6617], line_intensity=[1.0])
    n = 1_000_000
    edep, flags = g.run_histories(0, n, 2)
    p0 = ((flags >> 16) == 0).mean()
    assert abs(p0 - 0.693573) < 4 * math.sqrt(0.693573 * 0.306427 / n)


# ------------------------------------------------------------------ edge cases and errors
def test_edge_cases_and_error_codes(pkg, orc):
    w = dm.make_config(0)
    g = pkg.Gadep(0)
    with pytest.raises(pkg.GadepError) as e:
        g.run(10, 1)
    assert e.value.code == -2                                   # GADEP_E_ORDER
    g.set_materials(w.mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
    m = w.mesh
    with pytest.raises(pkg.GadepError) as e:                    # open surface
        g.load_mesh(m.vertices, m.triangles[:-1], m.tri_surface[:-1], m.surf_inside, m.surf_outside, 0)
    assert e.value.code == -7
    flipped = m.triangles.copy(); flipped[5] = flipped[5][[0, 2, 1]]
    with pytest.raises(pkg.GadepError) as e:                    # inconsistent orientation
        g.load_mesh(m.vertices, flipped, m.tri_surface, m.surf_inside, m.surf_outside, 0)
    assert e.value.code == -7
    bad = m.triangles.copy(); bad[0, 0] = 10 ** 6
    with pytest.raises(pkg.GadepError) as e:
        g.load_mesh(m.vertices, bad, m.tri_surface, m.surf_inside, m.surf_outside, 0)
    assert e.value.code == -5
    vbad = m.vertices.copy(); vbad[3, 1] = np.nan
    with pytest.raises(pkg.GadepError) as e:
        g.load_mesh(vbad, m.triangles, m.tri_surface, m.surf_inside, m.surf_outside, 0)
    assert e.value.code == -4
    deg = m.triangles.copy(); deg[7] = [deg[7][0], deg[7][0], deg[7][2]]
    with pytest.raises(pkg.GadepError) as e:
        g.load_mesh(m.vertices, deg, m.tri_surface, m.surf_inside, m.surf_outside, 0)
    assert e.value.code == -6
    g.load_mesh(m.vertices, m.triangles, m.tri_surface, m.surf_inside, m.surf_outside, 0)
    with pytest.raises(pkg.GadepError) as e:                    # trace before build
        g.trace_rays(np.zeros((1, 3), np.float32), np.array([[0, 0, 1]], np.float32))
    assert e.value.code == -2
    g.build_bvh()
    with pytest.raises(pkg.GadepError) as e:                    # line outside the table range
        g.set_source(0, pos=(0, 0, 250), line_mev=[5.0], line_intensity=[1.0])
    assert e.value.code == -3
    with pytest.raises(pkg.GadepError):
        g.set_source(0, pos=(0, 0, 250), line_mev=[0.5], line_intensity=[-1.0])
    g.set_source(**w.source)
    spec = g.run(0, 1)                                          # empty run: zeros
    assert spec.sum() == 0 and g.get_counters()["n_histories"] == 0
    spec = g.run(1, 1)                                          # a single history (ragged tail of one)
    assert g.get_counters()["n_histories"] == 1
    spec = g.run(1000, 1, n_bins=16, e_max_mev=0.5)             # line above the spectrum top -> overflow slot
    assert spec.shape == (17,)
    edep, flags = g.run_histories(12345, 777, 1)                # ragged size, offset start
    oe, of, _ = orc.OracleScene(w).run_histories(12345, 777, 1)
    assert (flags == of).mean() > 0.995
