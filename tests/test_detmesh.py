"""P1 -- generator / mesh pins: closed, oriented, Euler, closed-form volume and area,
Eq. 1-4 vertex positions, Eq. 6 shrink."""
import numpy as np
import pytest

import detmesh as dm
from detmesh.geometry import Arc, Line, discretise, revolve


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_surfaces_closed_oriented_positive_volume(cfg):
    m = dm.make_config(cfg).mesh
    for s in range(m.n_surf):
        tri = m.triangles[m.tri_surface == s]
        c = dm.check_closed_oriented(tri)
        assert c["ok"], (m.surface_names[s], c)
        assert c["euler"] == 2
        assert dm.mesh_signed_volume(m.vertices, tri) > 0


def test_pellet_stack_scene_is_closed_disjoint_and_of_known_volume():
    # the test scene of the per-material BVH entries: n disjoint cylinders r = 6, h = 4 on the axis, 2 mm apart
    m = dm.make_pellet_stack(12, n_theta=96).mesh
    assert m.n_surf == 13
    for s in range(12):
        tri = m.triangles[m.tri_surface == s]
        c = dm.check_closed_oriented(tri)
        assert c["ok"] and c["euler"] == 2
        vol = dm.mesh_signed_volume(m.vertices, tri)
        prism = 0.5 * 96 * 36.0 * np.sin(2 * np.pi / 96) * 4.0      # regular 96-gon prism
        assert vol == pytest.approx(prism, rel=1e-5)
        z = m.vertices[np.unique(tri)][:, 2]
        assert z.max() == pytest.approx(-6.0 * s) and z.min() == pytest.approx(-6.0 * s - 4.0)
    assert (m.surf_outside[:12] == dm.MAT["air"]).all() and m.surf_outside[12] == -1


def test_triangle_counts():
    assert dm.make_config(0).mesh.n_tri == 256           # BASELINE.json configs[0]: "~256 triangles"
    assert dm.make_config(1).mesh.n_tri == 38400
    assert dm.make_config(2).mesh.n_tri == 43520
    assert dm.make_config(3).mesh.n_tri == 48640


def test_config4_small_instance_and_band_allocation():
    w = dm.make_config(4, n_theta=64, total_bands=64)
    m = w.mesh
    for s in range(m.n_surf):
        assert dm.check_closed_oriented(m.triangles[m.tri_surface == s])["ok"]
    # 2 * n_theta * bands minus one n_theta per fan (2 fans per surface)
    assert m.n_tri == 64 * (2 * 64 - 2 * m.n_surf)


def test_prism_closed_forms():
    # inscribed N-gon prism: V = (N/2) R^2 sin(2pi/N) L ; area = 2 (N/2) R^2 sin(2pi/N) + 2 N R sin(pi/N) L
    N, R, L = 64, 30.0, 60.0
    m = dm.make_config(0).mesh
    V = 0.5 * N * R * R * np.sin(2 * np.pi / N) * L
    A = N * R * R * np.sin(2 * np.pi / N) + 2 * N * R * np.sin(np.pi / N) * L
    assert abs(V - 169373.618) < 1e-2 and abs(A - 16950.979) < 1e-2     # SURVEY.md P1 printed values
    assert dm.mesh_signed_volume(m.vertices, m.triangles) == pytest.approx(V, rel=1e-6)
    assert dm.mesh_area(m.vertices, m.triangles) == pytest.approx(A, rel=1e-6)


def test_eq1_to_eq4_vertices():
    R, r, n_phi, n_theta = 35.0, 8.0, 8, 256
    arc = Arc(R - r, -r, r, 0.5 * np.pi, 0.0, n_phi)
    p = arc.points()
    j = np.arange(n_phi + 1)[::-1]                      # traversed from phi = pi/2 down to 0
    phi = 0.5 * np.pi * j / n_phi                       # Eq. 3
    assert np.allclose(p[:, 0], (R - r) + r * np.cos(phi), atol=1e-12)      # Eq. 4 rho_j
    assert np.allclose(p[:, 1], 0.0 - r * (1 - np.sin(phi)), atol=1e-12)    # Eq. 4 z_j in the build frame (Q7)
    assert p[0] == pytest.approx([R - r, 0.0]) and p[-1] == pytest.approx([R, -r])
    prof = discretise([Line(0, 0, R - r, 0, 1), arc, Line(R, -r, R, -70, 4), Line(R, -70, 0, -70, 1)])
    v, t = revolve(prof, n_theta)
    ring = v[1:1 + n_theta]                             # first ring after the axis vertex: rho = R - r
    th = 2 * np.pi * np.arange(n_theta) / n_theta       # Eq. 1
    assert np.allclose(ring[:, 0], (R - r) * np.cos(th)) and np.allclose(ring[:, 1], (R - r) * np.sin(th))  # Eq. 2
    assert np.allclose(np.hypot(v[:, 0], v[:, 1]).max(), R)


def test_eq6_active_volume_nested_in_crystal():
    m = dm.make_config(1).mesh
    v = m.vertices.astype(np.float64)
    s0 = np.unique(m.triangles[m.tri_surface == 0])
    s1 = np.unique(m.triangles[m.tri_surface == 1])
    r0, r1 = np.hypot(v[s0, 0], v[s0, 1]).max(), np.hypot(v[s1, 0], v[s1, 1]).max()
    assert r0 == pytest.approx(35.0) and r1 == pytest.approx(35.0 - 0.7)       # R_active = D2 - D4
    assert v[s0, 2].max() == pytest.approx(0.0) and v[s1, 2].max() == pytest.approx(-0.7, abs=1e-6)
    # L_active = D1 - D4: back faces coincide up to the inside-outward separation delta
    assert v[s1, 2].min() - v[s0, 2].min() == pytest.approx(1e-3, abs=2e-5)
    # dead-layer volume ~ shell of 0.7 mm on front + side
    vol0 = dm.mesh_signed_volume(m.vertices, m.triangles[m.tri_surface == 0])
    vol1 = dm.mesh_signed_volume(m.vertices, m.triangles[m.tri_surface == 1])
    assert 0.04 < (vol0 - vol1) / vol0 < 0.06


def test_normals_outward_eq5():
    m = dm.make_config(0).mesh
    v = m.vertices.astype(np.float64)
    t = m.triangles
    n = np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]])      # Eq. 5 (un-normalised)
    c = (v[t[:, 0]] + v[t[:, 1]] + v[t[:, 2]]) / 3 - np.array([0, 0, -30.0])
    assert (np.einsum("ij,ij->i", n, c) > 0).all()


def test_marinelli_matrix_is_one_litre():
    m = dm.make_config(3).mesh
    s = m.surface_names.index("S9_matrix")
    vol = dm.mesh_signed_volume(m.vertices, m.triangles[m.tri_surface == s])
    assert vol == pytest.approx(1.0e6, rel=2e-4)       # BASELINE.json configs[3]: 1.0 L (polygonal, N=256)


def test_intensities_seed7_in_range():
    src = dm.make_config(2).source
    assert src["line_intensity"].shape == (8,)
    assert (src["line_intensity"] >= 0.5).all() and (src["line_intensity"] < 1.0).all()
