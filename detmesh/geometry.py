"""Triangulated surfaces of revolution (DetMesh `Geometry` layer).

A surface is the revolution about the z-axis of a meridian *profile*: a chain of
`Line` / `Arc` segments that starts and ends on the axis (rho = 0), so that the
revolved surface is closed (genus 0).  Rings are sampled angularly equidistantly,
theta_i = 2*pi*i/N_theta (Eq. 1-2); arcs are sampled at equal
polar-angle steps (Eq. 3-4).  A band that touches the axis is a
fan of N_theta triangles, any other band is 2*N_theta triangles.  Facets are
wound so that the Eq. 5 normal points out of the enclosed volume.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np


@dataclass(frozen=True)
class Line:
    """Straight meridian segment from (rho0, z0) to (rho1, z1), split into `bands` bands."""
    rho0: float
    z0: float
    rho1: float
    z1: float
    bands: int = 1

    def length(self) -> float:
        return float(np.hypot(self.rho1 - self.rho0, self.z1 - self.z0))

    def points(self, bands: int | None = None) -> np.ndarray:
        n = self.bands if bands is None else bands
        t = np.arange(n + 1, dtype=np.float64) / n
        return np.stack([self.rho0 + (self.rho1 - self.rho0) * t,
                         self.z0 + (self.z1 - self.z0) * t], axis=1)


@dataclass(frozen=True)
class Arc:
    """Circular meridian arc: rho = c_rho + r*cos(phi), z = c_z + r*sin(phi), phi0 -> phi1.

    Eq. 3-4 is the instance c_rho = R_out - R_chamfer, r = R_chamfer,
    equal steps in phi (angularly equidistant sampling of the rounding)."""
    c_rho: float
    c_z: float
    r: float
    phi0: float
    phi1: float
    bands: int = 8

    def length(self) -> float:
        return float(abs(self.phi1 - self.phi0) * self.r)

    def points(self, bands: int | None = None) -> np.ndarray:
        n = self.bands if bands is None else bands
        phi = self.phi0 + (self.phi1 - self.phi0) * (np.arange(n + 1, dtype=np.float64) / n)
        rho = self.c_rho + self.r * np.cos(phi)
        z = self.c_z + self.r * np.sin(phi)
        # snap exact end values (cos(pi/2) is 6e-17, not 0)
        rho[np.abs(rho) < 1e-12 * max(1.0, self.r + abs(self.c_rho))] = 0.0
        return np.stack([rho, z], axis=1)


def discretise(segments, band_counts=None) -> np.ndarray:
    """Chain segments into one meridian polyline [(rho, z)], dropping duplicated joints."""
    pts = []
    for k, seg in enumerate(segments):
        p = seg.points(None if band_counts is None else int(band_counts[k]))
        if pts:
            if not np.allclose(pts[-1], p[0], atol=1e-9):
                raise ValueError(f"profile segments {k-1} and {k} do not join: {pts[-1]} vs {p[0]}")
            p = p[1:]
        pts.extend(list(p))
    pts = np.asarray(pts, dtype=np.float64)
    if abs(pts[0, 0]) > 1e-12 or abs(pts[-1, 0]) > 1e-12:
        raise ValueError("profile must start and end on the axis (rho = 0)")
    pts[0, 0] = 0.0
    pts[-1, 0] = 0.0
    return pts


def allocate_bands(segments, total_bands: int) -> list[int]:
    """Distribute `total_bands` over segments in proportion to arc length, >= 1 each
    (largest-remainder rounding; SURVEY.md Q17 reading of BASELINE.json configs[4])."""
    lengths = np.array([s.length() for s in segments], dtype=np.float64)
    n = len(segments)
    if total_bands < n:
        raise ValueError("fewer bands than segments")
    share = lengths / lengths.sum() * (total_bands - n)
    base = np.floor(share).astype(int)
    rem = total_bands - n - int(base.sum())
    order = np.argsort(-(share - base), kind="stable")
    base[order[:rem]] += 1
    return [int(b) + 1 for b in base]


def revolve(profile: np.ndarray, n_theta: int):
    """Revolve a meridian polyline about z.  Returns (vertices f64[V,3], triangles i32[T,3]),
    wound so that the enclosed signed volume is positive (normals of Eq. 5 point outward)."""
    profile = np.asarray(profile, dtype=np.float64)
    theta = 2.0 * np.pi * np.arange(n_theta, dtype=np.float64) / n_theta  # Eq. 1
    cos_t, sin_t = np.cos(theta), np.sin(theta)
    verts = []
    ring_start = []  # index of first vertex of each profile point; axis points have 1 vertex
    on_axis = []
    nv = 0
    for rho, z in profile:
        ring_start.append(nv)
        if rho == 0.0:
            verts.append(np.array([[0.0, 0.0, z]]))
            on_axis.append(True)
            nv += 1
        else:
            verts.append(np.stack([rho * cos_t, rho * sin_t, np.full(n_theta, z)], axis=1))  # Eq. 2
            on_axis.append(False)
            nv += n_theta
    verts = np.concatenate(verts, axis=0)
    i = np.arange(n_theta, dtype=np.int64)
    ip = (i + 1) % n_theta
    tris = []
    for k in range(len(profile) - 1):
        a, b = ring_start[k], ring_start[k + 1]
        if on_axis[k] and on_axis[k + 1]:
            raise ValueError("two consecutive axis points in profile")
        if on_axis[k]:
            tris.append(np.stack([np.full(n_theta, a), b + i, b + ip], axis=1))
        elif on_axis[k + 1]:
            tris.append(np.stack([a + i, np.full(n_theta, b), a + ip], axis=1))
        else:
            tris.append(np.stack([a + i, b + i, b + ip], axis=1))
            tris.append(np.stack([a + i, b + ip, a + ip], axis=1))
    tris = np.concatenate(tris, axis=0).astype(np.int32)
    if _signed_volume(verts, tris) < 0.0:
        tris = tris[:, [0, 2, 1]].copy()
    return verts, tris


def _signed_volume(v: np.ndarray, t: np.ndarray) -> float:
    a, b, c = v[t[:, 0]], v[t[:, 1]], v[t[:, 2]]
    return float(np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0)


@dataclass
class Mesh:
    """In-memory hand-off DetMesh -> Gadep: shared vertex array, indexed
    facets, per-facet surface index, per-surface inside / outside material ids."""
    vertices: np.ndarray        # f32 [V,3], mm
    triangles: np.ndarray       # i32 [T,3]
    tri_surface: np.ndarray     # i32 [T]
    surf_inside: np.ndarray     # i32 [S]
    surf_outside: np.ndarray    # i32 [S]
    world_material: int
    surface_names: list = field(default_factory=list)

    @property
    def n_tri(self) -> int:
        return int(self.triangles.shape[0])

    @property
    def n_surf(self) -> int:
        return int(self.surf_inside.shape[0])


def merge_surfaces(surfaces, world_material: int) -> Mesh:
    """surfaces: list of (name, vertices f64[V,3], triangles i32[T,3], inside_id, outside_id)."""
    vs, ts, sid, s_in, s_out, names = [], [], [], [], [], []
    off = 0
    for s, (name, v, t, mi, mo) in enumerate(surfaces):
        vs.append(v)
        ts.append(t.astype(np.int64) + off)
        sid.append(np.full(t.shape[0], s, dtype=np.int32))
        s_in.append(mi)
        s_out.append(mo)
        names.append(name)
        off += v.shape[0]
    return Mesh(vertices=np.ascontiguousarray(np.concatenate(vs), dtype=np.float32),
                triangles=np.ascontiguousarray(np.concatenate(ts), dtype=np.int32),
                tri_surface=np.ascontiguousarray(np.concatenate(sid), dtype=np.int32),
                surf_inside=np.asarray(s_in, dtype=np.int32),
                surf_outside=np.asarray(s_out, dtype=np.int32),
                world_material=int(world_material), surface_names=names)


def mesh_signed_volume(vertices, triangles) -> float:
    return _signed_volume(np.asarray(vertices, dtype=np.float64), np.asarray(triangles))


def mesh_area(vertices, triangles) -> float:
    v = np.asarray(vertices, dtype=np.float64)
    t = np.asarray(triangles)
    n = np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]])
    return float(0.5 * np.linalg.norm(n, axis=1).sum())


def check_closed_oriented(triangles, n_vertices_hint: int | None = None) -> dict:
    """Edge-manifold / orientation / Euler check of one surface: every directed
    edge appears once and its reverse appears once.  Returns counts; `ok` is the verdict."""
    t = np.asarray(triangles, dtype=np.int64)
    e = np.concatenate([t[:, [0, 1]], t[:, [1, 2]], t[:, [2, 0]]], axis=0)
    nv = int(t.max()) + 1
    key = e[:, 0] * nv + e[:, 1]
    rkey = e[:, 1] * nv + e[:, 0]
    uk, cnt = np.unique(key, return_counts=True)
    dup = int((cnt != 1).sum())
    unmatched = int((~np.isin(rkey, uk)).sum())
    used = np.unique(t)
    V, E, F = int(used.size), int(uk.size // 2), int(t.shape[0])
    return {"ok": dup == 0 and unmatched == 0 and uk.size % 2 == 0,
            "duplicate_directed_edges": dup, "unmatched_edges": unmatched,
            "V": V, "E": E, "F": F, "euler": V - E + F}
