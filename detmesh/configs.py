"""The five synthetic detector / source set-ups of BASELINE.json `configs`.

Frame: z = 0 at the crystal front face, crystal toward -z, source toward +z, units mm / MeV.
These stand in for the paper's ORTEC detectors and point-source runs,
whose housing parameters d1-d10 are not printed.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

from .geometry import Line, Arc, discretise, revolve, merge_surfaces, allocate_bands, Mesh
from .materials import MAT, MAT_KILL, make_tables, E_MIN_MEV, E_MAX_MEV

SRC_POINT, SRC_VOLUME, SRC_BEAM = 0, 1, 2
DELTA = 1.0e-3  # separation of coincident back faces, from the inside outward


@dataclass
class Workload:
    name: str
    mesh: Mesh
    mu: np.ndarray            # f32 [M,4,G] 1/mm
    is_scoring: np.ndarray    # u8 [M]
    e_min_mev: float
    e_max_mev: float
    source: dict
    n_histories: int
    seed: int
    n_bins: int = 4096
    spectrum_e_max_mev: float = 2.0
    notes: dict = field(default_factory=dict)


def philox_u01_host(key0: int, key1: int, ctr, n: int) -> np.ndarray:
    """n uniforms ((w>>9)+0.5)*2^-23 from Philox4x32-10 words, counter (c0, c1, block, c3), block = 0,1,...
    Input-generator use only (BASELINE.json configs[2] intensities)."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
    out = []
    blk = 0
    while len(out) < n:
        c = [ctr[0] & 0xFFFFFFFF, ctr[1] & 0xFFFFFFFF, blk & 0xFFFFFFFF, ctr[3] & 0xFFFFFFFF]
        k0, k1 = key0 & 0xFFFFFFFF, key1 & 0xFFFFFFFF
        for _ in range(10):
            p0, p1 = M0 * c[0], M1 * c[2]
            c = [((p1 >> 32) ^ c[1] ^ k0) & 0xFFFFFFFF, p1 & 0xFFFFFFFF,
                 ((p0 >> 32) ^ c[3] ^ k1) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
            k0, k1 = (k0 + W0) & 0xFFFFFFFF, (k1 + W1) & 0xFFFFFFFF
        out.extend(c)
        blk += 1
    w = np.array(out[:n], dtype=np.uint64)
    return ((w >> np.uint64(9)).astype(np.float64) + 0.5) * 2.0 ** -23


def _surface(name, segments, n_theta, mat_in, mat_out, band_counts=None):
    v, t = revolve(discretise(segments, band_counts), n_theta)
    return (name, v, t, mat_in, mat_out)


def _cyl_segments(R, z_top, z_bot, side_bands):
    return [Line(0.0, z_top, R, z_top, 1), Line(R, z_top, R, z_bot, side_bands), Line(R, z_bot, 0.0, z_bot, 1)]


def _rounded_cyl_segments(R, z_front, z_back, r_ch, n_phi, side_bands):
    # Eq. 3-4 in the build frame: rho_j = (R-r) + r cos(phi_j),
    # z_j = z_front - r (1 - sin(phi_j)); traversed from phi = pi/2 (front face) to phi = 0 (side).
    return [Line(0.0, z_front, R - r_ch, z_front, 1),
            Arc(R - r_ch, z_front - r_ch, r_ch, 0.5 * np.pi, 0.0, n_phi),
            Line(R, z_front - r_ch, R, z_back, side_bands),
            Line(R, z_back, 0.0, z_back, 1)]


def _bore_segments(r, z_apex, z_back, n_phi, side_bands):
    # hemispherical front end, radius = bore radius, apex at z_apex
    return [Arc(0.0, z_apex - r, r, 0.5 * np.pi, 0.0, n_phi),
            Line(r, z_apex - r, r, z_back, side_bands),
            Line(r, z_back, 0.0, z_back, 1)]


def _cup_segments(R_in, R_out, z_rim, z_in_bot, z_out_bot, side_bands):
    return [Line(0.0, z_in_bot, R_in, z_in_bot, 1), Line(R_in, z_in_bot, R_in, z_rim, side_bands),
            Line(R_in, z_rim, R_out, z_rim, 1), Line(R_out, z_rim, R_out, z_out_bot, side_bands),
            Line(R_out, z_out_bot, 0.0, z_out_bot, 1)]


def _beaker_segments(R_well, z_well_top, R_out, z_top, z_bot, side_bands):
    return [Line(0.0, z_top, R_out, z_top, 1), Line(R_out, z_top, R_out, z_bot, side_bands),
            Line(R_out, z_bot, R_well, z_bot, 1), Line(R_well, z_bot, R_well, z_well_top, side_bands),
            Line(R_well, z_well_top, 0.0, z_well_top, 1)]


def _detector_segment_lists(n_phi, side_bands, world_z=(-300.0, 400.0)):
    """Coaxial p-type HPGe of BASELINE.json configs[1]; surfaces S0..S7 of SURVEY.md 8(d)."""
    d = DELTA
    G_A, G_D, AL, CU, AIR, VAC = (MAT["Ge_active"], MAT["Ge_dead"], MAT["Al"], MAT["Cu"], MAT["air"],
                                  MAT["vacuum"])
    return [
        ("S0_crystal_outer", _rounded_cyl_segments(35.0, 0.0, -70.0, 8.0, n_phi, side_bands), G_D, VAC),
        # Eq. 6: R_active = D2 - D4, L_active = D1 - D4; rounding 8 - 0.7
        ("S1_active", _rounded_cyl_segments(34.3, -0.7, -70.0 + d, 7.3, n_phi, side_bands), G_A, G_D),
        ("S2_bore_shell", _bore_segments(5.0003, -15.0 + 0.0003, -70.0 + 2 * d, n_phi, side_bands), G_D, G_A),
        ("S3_bore", _bore_segments(5.0, -15.0, -70.0 + 3 * d, n_phi, side_bands), VAC, G_D),
        ("S4_cu_cup", _cup_segments(35.1, 35.9, 0.0, -70.1, -70.9, side_bands), CU, VAC),
        ("S5_endcap_outer", _cyl_segments(41.9, 6.0, -101.9, side_bands), AL, AIR),
        ("S6_endcap_cavity", _cyl_segments(40.9, 5.0, -100.9, side_bands), VAC, AL),
        ("S7_world", _cyl_segments(300.0, world_z[1], world_z[0], side_bands), AIR, MAT_KILL),
    ]


def _build(seglists, n_theta, world_material, total_bands=None):
    if total_bands is None:
        surfs = [_surface(n, s, n_theta, mi, mo) for (n, s, mi, mo) in seglists]
    else:  # configs[4]: bands distributed over all segments of all surfaces by arc length
        flat = [seg for (_, s, _, _) in seglists for seg in s]
        counts = allocate_bands(flat, total_bands)
        surfs, k = [], 0
        for (n, s, mi, mo) in seglists:
            surfs.append(_surface(n, s, n_theta, mi, mo, counts[k:k + len(s)]))
            k += len(s)
    return merge_surfaces(surfs, world_material)


def _source(kind, pos=(0, 0, 0), direction=(0, 0, -1), cyl=(0, 0, 0), ex=(0, 0, 0), lines_kev=(), intens=None):
    lines = np.asarray(lines_kev, dtype=np.float64) * 1e-3
    if intens is None:
        intens = np.ones_like(lines)
    return {"kind": kind, "pos": np.asarray(pos, dtype=np.float32), "dir": np.asarray(direction, dtype=np.float32),
            "cyl_r": float(cyl[0]), "cyl_z0": float(cyl[1]), "cyl_z1": float(cyl[2]),
            "ex_r": float(ex[0]), "ex_z0": float(ex[1]), "ex_z1": float(ex[2]),
            "line_mev": np.ascontiguousarray(lines, dtype=np.float32),
            "line_intensity": np.ascontiguousarray(intens, dtype=np.float32)}


def make_config(i: int, n_theta: int | None = None, total_bands: int | None = None,
                coh_coeff: float | None = None) -> Workload:
    """Workload i of BASELINE.json `configs`.  `n_theta` / `total_bands` override the tessellation
    (used by tests to make small instances of config 4); `coh_coeff` overrides SURVEY.md Q1."""
    if i == 0:
        nt = 64 if n_theta is None else n_theta
        mesh = _build([("S0_crystal", _cyl_segments(30.0, 0.0, -60.0, 1), MAT["Ge_active"], MAT["vacuum"])],
                      nt, MAT["vacuum"])
        mu, sc, _ = make_tables(coh_coeff=0.0 if coh_coeff is None else coh_coeff)
        src = _source(SRC_POINT, pos=(0, 0, 250.0), lines_kev=[661.7])
        return Workload("cfg0_bare_ge_point_661keV", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, 1_000_000, 1)

    mu, sc, _ = make_tables(coh_coeff=7.0e-27 if coh_coeff is None else coh_coeff)
    nt = (4096 if i == 4 else 256) if n_theta is None else n_theta
    n_phi, side = 8, 4
    if i == 1:
        mesh = _build(_detector_segment_lists(n_phi, side), nt, MAT["air"])
        src = _source(SRC_POINT, pos=(0, 0, 106.0), lines_kev=[59.5, 122.1, 661.7, 1173.2, 1332.5])
        return Workload("cfg1_coax_hpge_point_5lines", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, 10_000_000, 1)
    if i in (2, 4):
        segl = _detector_segment_lists(n_phi, side)
        segl.insert(7, ("S8_container", _cyl_segments(36.0, 48.01, 6.01, side), MAT["polypropylene"], MAT["air"]))
        segl.insert(8, ("S9_water", _cyl_segments(35.0, 47.01, 7.01, side), MAT["water"], MAT["polypropylene"]))
        # keep the world as the last surface
        if i == 2:
            mesh = _build(segl, nt, MAT["air"])
            u = philox_u01_host(7, 0, (0, 0, 0, 0xFFFFFFFF), 8)
            src = _source(SRC_VOLUME, cyl=(35.0, 7.01, 47.01),
                          lines_kev=[46.5, 88.0, 122.1, 661.7, 898.0, 1173.2, 1332.5, 1836.1], intens=0.5 + 0.5 * u)
            return Workload("cfg2_coax_hpge_water_volume_8lines", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src,
                            100_000_000, 1)
        tb = 256 if total_bands is None else total_bands
        mesh = _build(segl, nt, MAT["air"], total_bands=tb)
        src = _source(SRC_POINT, pos=(0, 0, 31.0), lines_kev=[1332.5])
        return Workload("cfg4_mesh_stress_point_1332keV", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, 100_000_000, 1,
                        notes={"ray_box": (41.9, -101.9, 6.0), "ray_seed": 1, "n_rays": 100_000_000})
    if i == 3:
        segl = _detector_segment_lists(n_phi, side, world_z=(-400.0, 400.0))
        segl.insert(7, ("S8_beaker", _beaker_segments(42.4, 6.5, 55.4, 39.5, -229.85, side),
                        MAT["polypropylene"], MAT["air"]))
        segl.insert(8, ("S9_matrix", _beaker_segments(43.9, 8.0, 53.9, 38.0, -228.35, side),
                        MAT["SiO2"], MAT["polypropylene"]))
        mesh = _build(segl, nt, MAT["air"])
        lines = 40.0 * 75.0 ** (np.arange(40) / 39.0)
        src = _source(SRC_VOLUME, cyl=(53.9, -228.35, 38.0), ex=(43.9, -228.35, 8.0), lines_kev=lines)
        return Workload("cfg3_marinelli_sio2_40lines", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, 100_000_000, 1)
    raise ValueError(f"no config {i}")


def make_pellet_stack(n_pellets: int, n_theta: int = 24, n_histories: int = 20_000) -> Workload:
    """Test scene for the per-material BVH entries: `n_pellets` disjoint cylinders (r = 6 mm, 4 mm tall, 2 mm apart)
    stacked on the axis in air, materials cycling Ge_active / Cu / water, point source above the stack.  Air touches
    every pellet and the world (n_pellets + 1 surfaces), each pellet material n_pellets / 3 of them."""
    mats = [MAT["Ge_active"], MAT["Cu"], MAT["water"]]
    segl = []
    for k in range(n_pellets):
        z_top = -6.0 * k
        segl.append((f"P{k}", _cyl_segments(6.0, z_top, z_top - 4.0, 1), mats[k % 3], MAT["air"]))
    depth = 6.0 * n_pellets
    segl.append(("world", _cyl_segments(40.0, 30.0, -depth - 30.0, 2), MAT["air"], -1))
    mesh = _build(segl, n_theta, MAT["air"])
    mu, sc, _ = make_tables(coh_coeff=7.0e-27)
    src = _source(SRC_POINT, pos=(0, 0, 12.0), lines_kev=[122.1, 661.7])
    return Workload(f"pellet_stack_{n_pellets}", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, n_histories, 3,
                    notes={"ray_box": (8.0, -depth - 2.0, 2.0)})


def make_rays(n: int, seed: int, cyl_r: float, z0: float, z1: float):
    """Seeded isotropic rays from uniform points in a z-axis cylinder (BASELINE.json configs[4] ray test).
    Returns (org f32[n,3], dir f32[n,3]); directions are unit in float32 to 1 ulp."""
    rng = np.random.default_rng(seed)
    u = rng.random((n, 5))
    r = cyl_r * np.sqrt(u[:, 0])
    ph = 2 * np.pi * u[:, 1]
    org = np.stack([r * np.cos(ph), r * np.sin(ph), z0 + (z1 - z0) * u[:, 2]], axis=1)
    w = 1 - 2 * u[:, 3]
    s = np.sqrt(np.maximum(0.0, 1 - w * w))
    ps = 2 * np.pi * u[:, 4]
    d = np.stack([s * np.cos(ps), s * np.sin(ps), w], axis=1)
    return np.ascontiguousarray(org, dtype=np.float32), np.ascontiguousarray(d, dtype=np.float32)


# ---------------------------------------------------------------------------------------------------------------------
# Calibration sweep (Table 3, Fig. 11): 13 calibration energies from a point
# source 250 mm above the endcap, one FEPE curve per detector.  The paper's six ORTEC detectors are not specified in
# print (parameters d1-d10), so three synthetic coaxial p-type detectors span the same range of sizes.
TABLE3_KEV = (59.54, 81.00, 121.78, 244.70, 344.28, 356.02, 411.13, 443.97, 778.90, 964.06, 1112.09, 1332.49, 1408.02)

CALIBRATION_DETECTORS = (
    # crystal radius / length / front rounding, bore radius / depth of its apex, outer dead layer, endcap gap
    dict(name="cal_d60", R=30.0, L=60.0, r_ch=6.0, bore_r=4.5, bore_apex=-14.0, dead=0.5, gap=4.0),
    dict(name="cal_d70", R=35.0, L=70.0, r_ch=8.0, bore_r=5.0, bore_apex=-15.0, dead=0.7, gap=5.0),
    dict(name="cal_d85", R=42.5, L=80.0, r_ch=8.0, bore_r=5.5, bore_apex=-18.0, dead=1.0, gap=5.0),
)


def _param_detector_segment_lists(p, n_phi, side_bands):
    """Coaxial p-type HPGe from a parameter set: same surface recipe as configs[1] (Eq. 1-6)."""
    d = DELTA
    G_A, G_D, AL, CU, AIR, VAC = (MAT["Ge_active"], MAT["Ge_dead"], MAT["Al"], MAT["Cu"], MAT["air"], MAT["vacuum"])
    R, L, r, dl = p["R"], p["L"], p["r_ch"], p["dead"]
    shell = 0.0003                                   # inner bore dead layer, 0.3 um
    cup_in, cup_out = R + 0.1, R + 0.9               # 0.1 mm clearance, 0.8 mm Cu
    cav_r = cup_out + 5.0                            # cup outer + 5 mm
    cav_top, cav_bot = p["gap"], -(L + 0.9) - 30.0   # front gap; 30 mm rear vacuum
    return [
        ("S0_crystal_outer", _rounded_cyl_segments(R, 0.0, -L, r, n_phi, side_bands), G_D, VAC),
        ("S1_active", _rounded_cyl_segments(R - dl, -dl, -L + d, r - dl, n_phi, side_bands), G_A, G_D),
        ("S2_bore_shell", _bore_segments(p["bore_r"] + shell, p["bore_apex"] + shell, -L + 2 * d, n_phi, side_bands), G_D, G_A),
        ("S3_bore", _bore_segments(p["bore_r"], p["bore_apex"], -L + 3 * d, n_phi, side_bands), VAC, G_D),
        ("S4_cu_cup", _cup_segments(cup_in, cup_out, 0.0, -L - 0.1, -L - 0.9, side_bands), CU, VAC),
        ("S5_endcap_outer", _cyl_segments(cav_r + 1.0, cav_top + 1.0, cav_bot - 1.0, side_bands), AL, AIR),
        ("S6_endcap_cavity", _cyl_segments(cav_r, cav_top, cav_bot, side_bands), VAC, AL),
        ("S7_world", _cyl_segments(300.0, 400.0, -300.0, side_bands), AIR, MAT_KILL),
    ]


def make_calibration(detector: int, n_histories: int = 10_000_000, n_theta: int = 256) -> Workload:
    """Point source 250 mm above the endcap of CALIBRATION_DETECTORS[detector], the 13 energies of PAPER.md Table 3
    at equal intensity, 1e7 histories (Fig. 11)."""
    p = CALIBRATION_DETECTORS[detector]
    mu, sc, _ = make_tables(coh_coeff=7.0e-27)
    mesh = _build(_param_detector_segment_lists(p, 8, 4), n_theta, MAT["air"])
    src = _source(SRC_POINT, pos=(0, 0, p["gap"] + 1.0 + 250.0), lines_kev=TABLE3_KEV)
    return Workload(p["name"] + "_point250_13lines", mesh, mu, sc, E_MIN_MEV, E_MAX_MEV, src, n_histories, 1,
                    notes={"detector": dict(p)})


def make_calibration_batch(detectors=(0, 1, 2), n_histories: int = 30_000_000, n_theta: int = 256, pitch_mm: float = 768.0) -> Workload:
    """Several detector parameter sets in ONE scene and one launch (the paper's calibration
    use-case: six detectors x 13 energies).  Detector k of `detectors` is the CALIBRATION_DETECTORS
    geometry translated by k * pitch_mm along x inside its own world cylinder (air inside, KILL outside; the cylinders
    are disjoint), the point source 250 mm above each endcap is one source replicated at the matching translations
    (`notes["source_copies"]`): history h belongs to detector h mod K, and its line is counted under k * 13 + l, so one
    run returns K FEPE curves.  Materials and tables are shared."""
    surfs, offs = [], []
    z0 = None
    for k, d in enumerate(detectors):
        p = CALIBRATION_DETECTORS[d]
        zs = p["gap"] + 1.0 + 250.0
        if z0 is None:
            z0 = zs
        shift = np.array([k * pitch_mm, 0.0, 0.0])
        for (name, segs, mi, mo) in _param_detector_segment_lists(p, 8, 4):
            v, t = revolve(discretise(segs), n_theta)
            surfs.append((f"{p['name']}_{name}", v + shift, t, mi, mo))
        offs.append([k * pitch_mm, 0.0, zs - z0])
    mesh = merge_surfaces(surfs, MAT["air"])
    mu, sc, _ = make_tables(coh_coeff=7.0e-27)
    src = _source(SRC_POINT, pos=(0, 0, z0), lines_kev=TABLE3_KEV)
    return Workload("calibration_batch_" + "_".join(CALIBRATION_DETECTORS[d]["name"] for d in detectors), mesh, mu, sc,
                    E_MIN_MEV, E_MAX_MEV, src, n_histories, 1,
                    notes={"source_copies": np.asarray(offs, dtype=np.float32), "detectors": [dict(CALIBRATION_DETECTORS[d]) for d in detectors]})
