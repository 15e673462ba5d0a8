"""-m gpu: acceptance at the sizes BASELINE.json states, against the stored oracle runs under tests/golden/ (written
by tests/golden/make_golden.py, which calls only detmesh/ and oracle/).

Common random numbers: the GPU transports the *same* histories the stored oracle run holds -- same
seed, same history indices, same Philox streams -- so the two runs are almost perfectly correlated and the north_star's
"0.5 % relative" on the FEPE can be checked far below the statistical error of either run:
  emitted[l]    identical (line selection is an integer decision on identical uniforms; a float32 / double tie on the
                cumulative intensities may move a handful of histories)
  peak[l]       |gpu - oracle| <= 3 + 0.005 * oracle  per line
  spectrum      sum |gpu - oracle| <= 2 * (histories that took a different course)
  per history   (where the golden holds the dump) flags and deposit agree except for the diverged fraction, which is
                printed, bounded, and checked for bias
and the independent-sample criteria (3 combined standard errors, chi^2/dof <= 1.2) on top.
The config-4 geometry bar: nearest facet of the first 1e6 seeded rays on the full 2.0 M-facet mesh against the stored
brute-force result, index bit-exact except ties within 1e-6 relative, distance within 1e-5 relative (R12).
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


def _gold(name):
    path = os.path.join(GOLDEN, name)
    if not os.path.exists(path):
        pytest.skip(f"{name} not generated")
    return json.load(open(path))


def _context(pkg, gold):
    kw = {}
    if gold.get("tessellation"):
        kw.update(n_theta=gold["tessellation"]["n_theta"], total_bands=gold["tessellation"]["total_bands"])
    if gold.get("coh_coeff") is not None:
        kw.update(coh_coeff=gold["coh_coeff"])
    w = dm.make_config(gold["config"], **kw)
    assert w.mesh.n_tri == gold["n_tri"] and w.seed == gold["seed"]
    g = pkg.Gadep(0)
    g.load_workload(w)
    return w, g


def _chi2_dof(a, na, b, nb):
    a, b = a.astype(np.float64), b.astype(np.float64)
    m = (a + b) >= 20
    num = (a[m] / na - b[m] / nb) ** 2
    den = a[m] / na ** 2 + b[m] / nb ** 2
    return float((num / den).sum() / max(m.sum(), 1)), int(m.sum())


def _counts_agree(c, gold, n_div_bound, report):
    """Common-random-number criteria on the integer tallies."""
    L = c["n_lines"]
    d_em = sum(abs(a - b) for a, b in zip(c["emitted"], gold["emitted"]))
    assert d_em <= 4, (c["emitted"], gold["emitted"])          # identical up to ties of the line-selection draw
    for l in range(L):
        po, pg = gold["peak"][l], c["peak"][l]
        assert abs(pg - po) <= 3 + 0.005 * po, (l, pg, po)
        # FEPE: both criteria of the north_star, on the correlated runs
        fo, fg = po / gold["emitted"][l], pg / c["emitted"][l]
        so = math.sqrt(max(fo * (1 - fo), 0.0) / gold["emitted"][l])
        sg = math.sqrt(max(fg * (1 - fg), 0.0) / c["emitted"][l])
        assert abs(fg - fo) <= 3 * math.sqrt(so * so + sg * sg) + 1e-12
        assert abs(fg - fo) <= 0.005 * fo + 3.0 / gold["emitted"][l]
    report["peak_abs_diff_per_line"] = [abs(c["peak"][l] - gold["peak"][l]) for l in range(L)]
    report["emitted_abs_diff"] = d_em
    return report


# ------------------------------------------------------------------ per-history CRN parity at golden size (<= 2e6)
@pytest.mark.parametrize("name,div_max", [("cfg2_oracle_n1000000.json", 0.005), ("cfg3_oracle_n1000000.json", 0.005),
                                          ("cfg4_oracle_n1000000_nt512_b128.json", 0.002)])
def test_common_random_number_parity_per_history(pkg, orc, name, div_max):
    gold = _gold(name)
    dump = np.load(os.path.join(GOLDEN, gold["per_history"]))
    of, oe = dump["flags"], dump["edep"].astype(np.float64)
    n = gold["n_histories"]
    w, g = _context(pkg, gold)
    # the GPU on the same histories: one accumulated run for the tallies, chunked dumps for the per-history comparison
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"], first_history=gold["first_history"]).copy()
    c = g.get_counters()
    assert c["n_histories"] == n and sum(c["emitted"]) == n and c["n_leak"] <= 2 and c["n_stack_overflow"] == 0
    gf = np.empty(n, dtype=np.uint32)
    ge = np.empty(n, dtype=np.float64)
    for first in range(0, n, 250_000):
        m = min(250_000, n - first)
        e, f = g.run_histories(first, m, gold["seed"])
        gf[first:first + m] = f
        ge[first:first + m] = e
    same = (gf == of) & (np.abs(ge - oe) <= 2e-6 + 1e-5 * oe)
    n_div = int((~same).sum())
    report = {"golden": name, "n": n, "diverged": n_div, "diverged_fraction": n_div / n}
    assert n_div <= div_max * n, report
    # what a diverged history does is unbiased: its chance to be a full-absorption event is the same on both sides
    pk_g, pk_o = int(((gf[~same] & 2) != 0).sum()), int(((of[~same] & 2) != 0).sum())
    assert abs(pk_g - pk_o) <= 4 * math.sqrt(pk_g + pk_o + 1), (pk_g, pk_o)
    report["diverged_peaks_gpu_oracle"] = (pk_g, pk_o)
    # the line of a history is decided before any float32 arithmetic differs
    assert int((((gf >> 8) & 0xFF) != ((of >> 8) & 0xFF)).sum()) <= 4
    _counts_agree(c, gold, n_div, report)
    d_spec = int(np.abs(spec.astype(np.int64) - np.array(gold["spectrum"], dtype=np.int64)).sum())
    assert d_spec <= 2 * n_div + 4, (d_spec, n_div)
    report["spectrum_l1_diff"] = d_spec
    chi2, dof = _chi2_dof(spec[:-1], n, np.array(gold["spectrum"][:-1]), n)
    assert chi2 <= 1.2, (chi2, dof)
    # event totals track the oracle's to the diverged fraction (the first flight of a history shares the ray of its
    # start localisation on the GPU; flights answered by the clearance grid are queries the oracle makes)
    oc = gold["counters"]
    assert abs(c["n_queries"] + c["n_skipped_queries"] + n - oc["n_queries"]) <= 0.01 * oc["n_queries"]
    for k in ("n_crossings", "n_pe", "n_compton", "n_coherent", "n_escaped"):
        assert abs(c[k] - oc[k]) <= 0.01 * oc[k] + 50, (k, c[k], oc[k])
    print("\nCRN parity", json.dumps(report))


# ------------------------------------------------------------------ CRN parity of the tallies at 1e7 (point sources)
@pytest.mark.parametrize("name", ["cfg0_oracle_n10000000.json", "cfg1_oracle_n10000000.json",
                                  "cfg1_coh7.0e-30_oracle_n10000000.json"])
def test_common_random_number_parity_tallies_1e7(pkg, orc, name):
    gold = _gold(name)
    n = gold["n_histories"]
    w, g = _context(pkg, gold)
    spec = g.run(n, gold["seed"], gold["n_bins"], gold["e_max_mev"], first_history=gold.get("first_history", 0)).copy()
    c = g.get_counters()
    assert c["n_histories"] == n and sum(c["emitted"]) == n and c["n_leak"] == 0
    d_spec = int(np.abs(spec.astype(np.int64) - np.array(gold["spectrum"], dtype=np.int64)).sum())
    report = {"golden": name, "n": n, "spectrum_l1_diff": d_spec,
              "scoring_histories": int(np.array(gold["spectrum"]).sum())}
    # every diverged history moves at most two bins; 99.9 % of the histories agree
    assert d_spec <= 2 * 0.001 * n, report
    _counts_agree(c, gold, d_spec, report)
    chi2, dof = _chi2_dof(spec[:-1], n, np.array(gold["spectrum"][:-1]), n)
    assert dof > 10 and chi2 <= 1.2, (chi2, dof)
    print("\nCRN parity", json.dumps(report))


# ------------------------------------------------------------------ FEPE read from the spectrum (mode 1)
def test_fepe_mode1_matches_its_definition(pkg, orc):
    w = dm.make_config(1)
    g = pkg.Gadep(0)
    g.load_workload(w)
    n = 2_000_000
    spec = g.run(n, 5, w.n_bins, w.spectrum_e_max_mev)
    c = g.get_counters()
    for l in range(c["n_lines"]):
        f1, se1 = g.fepe(l, 1)
        fo, so = orc.fepe(spec, c["emitted"], c["peak"], w.source["line_mev"], l, 1, w.spectrum_e_max_mev)
        assert f1 == pytest.approx(fo, rel=1e-12, abs=1e-15) and se1 == pytest.approx(so, rel=1e-9, abs=1e-15)
        f0, _ = g.fepe(l, 0)
        assert f0 == pytest.approx(orc.fepe(spec, c["emitted"], c["peak"], w.source["line_mev"], l, 0)[0], rel=1e-12)
    # single line, clean peak: both modes agree to the continuum under the peak bin
    w0 = dm.make_config(0)
    g0 = pkg.Gadep(0)
    g0.load_workload(w0)
    g0.run(1_000_000, 1, w0.n_bins, w0.spectrum_e_max_mev)
    assert abs(g0.fepe(0, 1)[0] - g0.fepe(0, 0)[0]) <= 0.01 * g0.fepe(0, 0)[0]


# ------------------------------------------------------------------ sharded run: two contexts + one exchange
def test_two_contexts_sharded_run_equals_one_context(pkg, orc):
    from paper_2605_25963_b200.sharding import history_range
    w = dm.make_config(2)
    n, seed = 300_001, 11
    one = pkg.Gadep(0)
    one.load_workload(w)
    one.run(n, seed, w.n_bins, w.spectrum_e_max_mev)
    ref = one.get_tallies()
    assert len(ref) == one.tally_size() == w.n_bins + 1 + 128
    parts = []
    ctxs = []
    for r in range(2):
        first, cnt = history_range(n, r, 2)
        g = pkg.Gadep(0)
        g.load_workload(w)
        g.run(cnt, seed, w.n_bins, w.spectrum_e_max_mev, first_history=first)
        parts.append(g.get_tallies())
        ctxs.append(g)
    total = parts[0] + parts[1]                 # what the all-reduce does (integer sum)
    assert np.array_equal(total, ref)
    assert not np.array_equal(parts[0], ref)
    # the reduced block goes back into a context: FEPE and counters now describe the whole job
    ctxs[0].set_tallies(total)
    c0, cr = ctxs[0].get_counters(), one.get_counters()
    assert c0["emitted"] == cr["emitted"] and c0["peak"] == cr["peak"]
    for l in range(cr["n_lines"]):
        assert ctxs[0].fepe(l, 0) == one.fepe(l, 0) and ctxs[0].fepe(l, 1) == one.fepe(l, 1)
    # device-resident exchange buffers (torch is only memory here)
    import torch
    d = torch.zeros(len(ref), dtype=torch.int64, device="cuda")
    ctxs[1].get_tallies(d)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy().astype(np.uint64), parts[1])


# ------------------------------------------------------------------ run-time checks of the ABI (call orders it allows)
def test_material_ids_and_line_energies_are_checked_against_the_tables_in_use(pkg, orc):
    w = dm.make_config(1)
    g = pkg.Gadep(0)
    m = w.mesh
    # mesh first, with ids that only a larger material set covers: accepted (nothing to check against yet) ...
    g.load_mesh(m.vertices, m.triangles, m.tri_surface, m.surf_inside, m.surf_outside, m.world_material)
    g.build_bvh()
    # ... but the run refuses tables that do not cover them
    g.set_materials(w.mu[:3], w.is_scoring[:3], w.e_min_mev, w.e_max_mev)
    g.set_source(**w.source)
    with pytest.raises(pkg.GadepError) as ei:
        g.run(1000, 1)
    assert ei.value.code == -5                  # GADEP_E_INDEX
    g.set_materials(w.mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
    g.run(1000, 1)
    # tables re-set with a narrower energy range after the source: the 59.5 keV line no longer fits
    g.set_materials(w.mu, w.is_scoring, 0.1, w.e_max_mev)
    with pytest.raises(pkg.GadepError) as ei:
        g.run(1000, 1)
    assert ei.value.code == -3                  # GADEP_E_ARG
    # kernel-selecting run flags exclude one another
    g.set_materials(w.mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
    with pytest.raises(pkg.GadepError):
        g.run(1000, 1, flags=pkg.binding.RUN_PARTIAL_XS | pkg.binding.RUN_PARITY_LOCALISATION)


# ------------------------------------------------------------------ the two traversals hold the same facets
@pytest.mark.parametrize("cfg,n_rays,box", [(1, 1_000_000, (45.0, -105.0, 10.0)), (3, 1_000_000, (60.0, -235.0, 45.0))])
def test_compressed_wide_nodes_give_the_same_hits(pkg, orc, cfg, n_rays, box):
    w = dm.make_config(cfg)
    g = pkg.Gadep(0)
    g.load_workload(w)
    org, d = make_rays(n_rays, 2, *box)
    res = {}
    for width in (4, 5, 8):                    # 5 = 4-wide with 8-bit quantised boxes (64-byte nodes)
        g.set_bvh_width(width)
        for filt, tmin in ((-2, 0.0), (dm.MAT["Ge_active"], -1.0e-4)):
            tri, t = g.trace_rays(org, d, filt, tmin)
            res[(width, filt)] = (tri.copy(), t.copy())
            assert g.get_counters()["n_stack_overflow"] == 0
    for filt in (-2, dm.MAT["Ge_active"]):
        for width in (5, 8):
            assert np.array_equal(res[(4, filt)][0], res[(width, filt)][0])
            assert np.array_equal(res[(4, filt)][1], res[(width, filt)][1])
    with pytest.raises(pkg.GadepError):
        g.set_bvh_width(6)


# ------------------------------------------------------------------ config 4: 1e6 seeded rays, full mesh, brute force
def test_cfg4_full_mesh_1e6_rays_vs_stored_brute_force(pkg, orc):
    path = os.path.join(GOLDEN, "cfg4_rays_n1000000.npz")
    if not os.path.exists(path):
        pytest.skip("stored brute-force rays not generated")
    gold = np.load(path)
    otri, ot = gold["tri"], gold["t"]
    n = len(otri)
    w = dm.make_config(4)
    assert w.mesh.n_tri == int(gold["n_tri"]) and w.notes["ray_seed"] == int(gold["ray_seed"])
    g = pkg.Gadep(0)
    g.load_workload(w)
    R, z0, z1 = w.notes["ray_box"]
    org, d = make_rays(n, w.notes["ray_seed"], R, z0, z1)
    report = {"n_rays": n}
    tri_auto, t_auto = g.trace_rays(org, d)          # no width set: the 64-byte nodes on a hierarchy of this size
    for width in (4, 5, 8):
        g.set_bvh_width(width)
        tri, t = g.trace_rays(org, d)
        assert np.array_equal(tri, tri_auto) and np.array_equal(t, t_auto)
        assert g.get_counters()["n_stack_overflow"] == 0
        hit = otri >= 0
        assert hit.all()                             # origins lie inside the world surface: every ray meets a facet
        miss = np.nonzero(tri < 0)[0]
        assert len(miss) == 0, len(miss)
        coord = float(np.abs(w.mesh.vertices).max())
        ulp = float(np.spacing(np.float32(coord)))
        v = w.mesh.vertices.astype(np.float64)
        f = w.mesh.triangles[otri]
        nrm = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
        nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
        cosang = np.maximum(np.abs(np.einsum("ij,ij->i", nrm, d.astype(np.float64))), 1e-7)
        floor = 8 * ulp / cosang                     # DESIGN.md R12: float32 inputs bound the hit point, 1/cos amplifies
        err = np.abs(t.astype(np.float64) - ot)
        same_idx = tri == otri
        assert (err[same_idx] <= 1e-5 * np.abs(ot[same_idx]) + floor[same_idx]).all(), \
            float((err[same_idx] / (1e-5 * np.abs(ot[same_idx]) + floor[same_idx])).max())
        n_rel_only = int((err <= 1e-5 * np.abs(ot)).sum())
        diff = np.nonzero(~same_idx)[0]
        # index mismatches: ties only -- the GPU's facet, in the oracle's double arithmetic, lies at the same distance as
        # the oracle's facet; or the ray starts on a facet (the oracle sees it a few nm behind the origin, float32 a few nm
        # ahead: a tie at the edge of the window t > 0)
        s = None
        n_edge = n_origin = 0
        for i in diff:
            if s is None:
                s = orc.OracleScene(w)
            o64, d64 = org[i].astype(np.float64), d[i].astype(np.float64)
            ok, tt, _ = s.ray_triangle(int(tri[i]), o64, d64)
            p = v[w.mesh.triangles[tri[i]]]
            nn = np.cross(p[1] - p[0], p[2] - p[0])
            cs = max(abs(float(nn @ d64) / float(np.linalg.norm(nn))), 1e-7)
            if not ok:                               # through a shared edge: the oracle's inclusive test gave it to the neighbour
                n_edge += 1
                tt = float(nn @ (p[0] - o64)) / float(nn @ d64)
                q = o64 + tt * d64
                # signed in-plane distance of the hit point to each edge line (positive inside): the GPU's facet must hold
                # the point within the float32 resolution of the hit point (a relative barycentric bound would be
                # meaningless on the 0.05 mm slivers of this mesh)
                nl = float(np.linalg.norm(nn))
                dist = [float(np.cross(p[(k + 1) % 3] - p[k], q - p[k]) @ nn) / (nl * float(np.linalg.norm(p[(k + 1) % 3] - p[k]))) for k in range(3)]
                assert min(dist) >= -8 * ulp / cs, (i, dist)
            if tt <= 0.0 and abs(tt) <= 8 * ulp / cs and abs(float(t[i]) - tt) <= 8 * ulp / cs:
                n_origin += 1                        # origin on the facet within float32 resolution
                continue
            assert abs(tt - ot[i]) <= 1e-6 * abs(ot[i]) + 8 * ulp / cs, (i, tri[i], otri[i], tt, ot[i])
            assert abs(float(t[i]) - ot[i]) <= 1e-5 * abs(ot[i]) + 8 * ulp / cs
        assert n_origin <= 5
        assert len(diff) <= 1e-4 * n + 2
        report[f"width{width}"] = {"index_identical": n - len(diff), "ties": len(diff), "of_which_through_an_edge": n_edge, "origin_on_a_facet": n_origin,
                                   "t_within_1e-5_relative_alone": n_rel_only}
    print("\nconfig-4 rays", json.dumps(report))


# ------------------------------------------------------------------ NEXT-3: several detectors in one scene, one launch
def test_batched_detectors_one_launch_vs_oracle_and_vs_separate_launches(pkg, orc):
    dets = (0, 1, 2)
    wb = dm.make_calibration_batch(dets, n_histories=3_000_000)
    g = pkg.Gadep(0)
    g.load_workload(wb)                         # applies notes["source_copies"] through gadep_set_source_copies
    # per-history parity with the oracle on the batched scene (same streams)
    n = 30_000
    s = orc.OracleScene(wb)
    edep, flags = g.run_histories(0, n, wb.seed)
    oe, of, oc = s.run_histories(0, n, wb.seed)
    same = (flags == of) & (np.abs(edep.astype(np.float64) - oe) <= 2e-6 + 1e-5 * oe)
    assert same.mean() >= 0.999, same.mean()
    assert np.array_equal((flags >> 8) & 0xFF, (of >> 8) & 0xFF)          # copy * 13 + line on both sides
    # one launch = three FEPE curves; each equals the curve of that detector run on its own (same histories: history h
    # of the batch is history h of the single-detector run for h = k mod 3 -- the other two thirds of the single run are
    # different histories, so the comparison is statistical, 4 sigma)
    nb = wb.n_histories
    g.run(nb, wb.seed, wb.n_bins, wb.spectrum_e_max_mev)
    cb = g.get_counters()
    assert cb["n_lines"] == 39 and cb["n_leak"] == 0
    em = np.array(cb["emitted"]).reshape(3, 13)
    assert em.sum(axis=1).tolist() == [nb // 3] * 3                      # round robin
    for k, d in enumerate(dets):
        w1 = dm.make_calibration(d, n_histories=nb // 3)
        g1 = pkg.Gadep(0)
        g1.load_workload(w1)
        g1.run(nb // 3, w1.seed + 1, w1.n_bins, w1.spectrum_e_max_mev)       # an independent sample of the same detector
        for l in range(13):
            fb, sb_ = g.fepe(13 * k + l, 0)
            f1, s1_ = g1.fepe(l, 0)
            assert abs(fb - f1) <= 4 * math.sqrt(sb_ * sb_ + s1_ * s1_) + 1e-9, (k, l, fb, f1)
    # the replicated source is reset by a new gadep_set_source and refuses too many lines
    with pytest.raises(pkg.GadepError):
        g.set_source_copies(np.zeros((5, 3), dtype=np.float32))           # 5 x 13 > 64 lines
    g.set_source_copies(None)
    assert g.get_counters()["n_lines"] == 13
