"""ctypes front-end of the CPU oracle (oracle/gadep_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It never imports, links or calls anything of the CUDA path (paper_2605_25963_b200).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gadep_oracle.c")
_LIB = os.path.join(_HERE, "libgadep_oracle.so")

F_ESCAPED, F_PEAK, F_LEAK, F_NONSCORING = 1, 2, 4, 8
COUNTER_NAMES = ("n_queries", "n_crossings", "n_pe", "n_compton", "n_coherent", "n_pair", "n_escaped", "n_leak",
                 "n_cutoff", "n_filter_reject")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP threads over histories)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        vp, dbl, i32, u64, u32, ll = C.c_void_p, C.c_double, C.c_int, C.c_uint64, C.c_uint32, C.c_longlong
        L.orc_create.restype = vp
        L.orc_destroy.argtypes = [vp]
        L.orc_set_materials.argtypes = [vp, i32, i32, dbl, dbl, vp, vp]
        L.orc_load_mesh.argtypes = [vp, vp, i32, vp, vp, i32, vp, vp, i32, i32]
        L.orc_set_source.argtypes = [vp, i32, vp, vp, dbl, dbl, dbl, dbl, dbl, dbl, i32, vp, vp]
        L.orc_philox.argtypes = [vp, vp, vp]
        L.orc_u01.argtypes = [u64, u64, u32, u32]
        L.orc_u01.restype = dbl
        L.orc_mu.argtypes = [vp, i32, i32, dbl]
        L.orc_mu.restype = dbl
        L.orc_ray_triangle.argtypes = [vp, i32, vp, vp, vp, vp]
        L.orc_nearest_hit.argtypes = [vp, vp, vp, i32, dbl, vp, vp]
        L.orc_trace_rays.argtypes = [vp, vp, vp, ll, i32, dbl, vp, vp]
        L.orc_trace_rays.restype = None
        L.orc_locate_sideid.argtypes = [vp, vp, vp]
        L.orc_locate_parity.argtypes = [vp, vp, vp]
        L.orc_test_compton.argtypes = [dbl, u64, ll, vp, vp]
        L.orc_test_compton.restype = None
        L.orc_test_thomson.argtypes = [u64, ll, vp]
        L.orc_test_thomson.restype = None
        L.orc_test_isotropic.argtypes = [u64, ll, vp]
        L.orc_test_isotropic.restype = None
        L.orc_test_rotate.argtypes = [vp, dbl, dbl, vp]
        L.orc_test_rotate.restype = None
        L.orc_set_source_copies.argtypes = [vp, i32, vp]
        L.orc_test_source.argtypes = [vp, u64, u64, ll, vp, vp, vp, vp]
        L.orc_test_source.restype = None
        L.orc_run_histories.argtypes = [vp, u64, ll, u64, vp, vp, vp, vp, vp]
        L.orc_run.argtypes = [vp, u64, ll, u64, i32, dbl, vp, vp, vp, vp]
        L.orc_num_threads.restype = i32
        L.orc_set_electron_mode.argtypes = [vp, vp, i32]
        L.orc_electron_range_mm.argtypes = [dbl, dbl]
        L.orc_electron_range_mm.restype = dbl
        L.orc_test_electron_split.argtypes = [vp, vp, i32, dbl, u64, u64, ll, vp]
        L.orc_test_electron_split.restype = None
    return _lib


def electron_range_mm(t_mev: float, rho_g_cm3: float) -> float:
    """Katz-Penfold range of an electron of kinetic energy t_mev in a material of that density (R16)."""
    return float(lib().orc_electron_range_mm(float(t_mev), float(rho_g_cm3)))


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(_p(c), _p(k), _p(out))
    return out


def u01(seed, history, stream, draw) -> float:
    return lib().orc_u01(seed, history, stream, draw)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def sample_compton(e_mev: float, seed: int, n: int):
    eps = np.empty(n)
    cos = np.empty(n)
    lib().orc_test_compton(e_mev, seed, n, _p(eps), _p(cos))
    return eps, cos


def sample_thomson(seed: int, n: int):
    cos = np.empty(n)
    lib().orc_test_thomson(seed, n, _p(cos))
    return cos


def sample_isotropic(seed: int, n: int):
    d = np.empty((n, 3))
    lib().orc_test_isotropic(seed, n, _p(d))
    return d


def rotate(d, c, phi):
    d = np.ascontiguousarray(d, dtype=np.float64)
    out = np.empty(3)
    lib().orc_test_rotate(_p(d), c, phi, _p(out))
    return out


class OracleScene:
    """Scene handle; takes the same arrays as the C-ABI of include/gadep.h."""

    def __init__(self, workload=None):
        self.L = lib()
        self.h = C.c_void_p(self.L.orc_create())
        self.n_lines = 0
        if workload is not None:
            w = workload
            self.set_materials(w.mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
            m = w.mesh
            self.load_mesh(m.vertices, m.triangles, m.tri_surface, m.surf_inside, m.surf_outside, m.world_material)
            self.set_source(**w.source)
            if getattr(w, "notes", None) and w.notes.get("source_copies") is not None:
                self.set_source_copies(w.notes["source_copies"])

    def __del__(self):
        try:
            self.L.orc_destroy(self.h)
        except Exception:
            pass

    def set_materials(self, mu, is_scoring, e_min, e_max):
        mu = np.ascontiguousarray(mu, dtype=np.float32)
        sc = np.ascontiguousarray(is_scoring, dtype=np.uint8)
        rc = self.L.orc_set_materials(self.h, mu.shape[0], mu.shape[2], e_min, e_max, _p(mu), _p(sc))
        assert rc == 0, rc

    def load_mesh(self, vertices, triangles, tri_surface, surf_inside, surf_outside, world_material):
        v = np.ascontiguousarray(vertices, dtype=np.float32)
        t = np.ascontiguousarray(triangles, dtype=np.int32)
        ts = np.ascontiguousarray(tri_surface, dtype=np.int32)
        si = np.ascontiguousarray(surf_inside, dtype=np.int32)
        so = np.ascontiguousarray(surf_outside, dtype=np.int32)
        rc = self.L.orc_load_mesh(self.h, _p(v), v.shape[0], _p(t), _p(ts), t.shape[0], _p(si), _p(so), si.shape[0],
                                  int(world_material))
        assert rc == 0, rc
        self.n_tri = t.shape[0]

    def set_source(self, kind, pos, dir, cyl_r=0.0, cyl_z0=0.0, cyl_z1=0.0, ex_r=0.0, ex_z0=0.0, ex_z1=0.0,
                   line_mev=None, line_intensity=None):
        pos = np.ascontiguousarray(pos, dtype=np.float32).astype(np.float64)
        d = np.ascontiguousarray(dir, dtype=np.float32).astype(np.float64)
        le = np.ascontiguousarray(line_mev, dtype=np.float32)
        li = np.ascontiguousarray(line_intensity, dtype=np.float32)
        f32 = lambda x: float(np.float32(x))
        rc = self.L.orc_set_source(self.h, int(kind), _p(pos), _p(d), f32(cyl_r), f32(cyl_z0), f32(cyl_z1), f32(ex_r),
                                   f32(ex_z0), f32(ex_z1), le.shape[0], _p(le), _p(li))
        assert rc == 0, rc
        self.n_lines = le.shape[0]
        self.line_mev = le.astype(np.float64)
        self.line_mev_base = self.line_mev.copy()
        self.L.orc_set_source_copies(self.h, 1, None)

    def set_source_copies(self, offsets):
        """NEXT-3 batched scenes: replicate the source at these translations (float32 values, [n][3]); history h is emitted
        from copy h mod n and counted under line copy * n_lines + l.  None = the plain source."""
        if offsets is None:
            assert self.L.orc_set_source_copies(self.h, 1, None) == 0
            self.n_lines = len(self.line_mev_base)
        else:
            off = np.ascontiguousarray(np.asarray(offsets, dtype=np.float32).astype(np.float64))
            assert off.ndim == 2 and off.shape[1] == 3
            assert self.L.orc_set_source_copies(self.h, off.shape[0], _p(off)) == 0
            self.n_lines = len(self.line_mev_base) * off.shape[0]
        self.line_mev = np.tile(self.line_mev_base, self.n_lines // len(self.line_mev_base))

    def mu(self, m, ch, e):
        return self.L.orc_mu(self.h, m, ch, e)

    def ray_triangle(self, tri, o, d):
        o = np.ascontiguousarray(o, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        t = C.c_double()
        dn = C.c_double()
        hit = self.L.orc_ray_triangle(self.h, int(tri), _p(o), _p(d), C.byref(t), C.byref(dn))
        return (bool(hit), t.value, dn.value)

    def nearest_hit(self, o, d, filter_mat=-2, t_min=0.0):
        o = np.ascontiguousarray(o, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        t = C.c_double()
        lv = C.c_int()
        tri = self.L.orc_nearest_hit(self.h, _p(o), _p(d), filter_mat, t_min, C.byref(t), C.byref(lv))
        return tri, t.value, lv.value

    def trace_rays(self, org, dir, filter_mat=-2, t_min=0.0):
        org = np.ascontiguousarray(org, dtype=np.float32)
        dir = np.ascontiguousarray(dir, dtype=np.float32)
        n = org.shape[0]
        tri = np.empty(n, dtype=np.int32)
        t = np.empty(n, dtype=np.float64)
        self.L.orc_trace_rays(self.h, _p(org), _p(dir), n, filter_mat, t_min, _p(tri), _p(t))
        return tri, t

    def locate_sideid(self, o, d):
        o = np.ascontiguousarray(o, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        return self.L.orc_locate_sideid(self.h, _p(o), _p(d))

    def locate_parity(self, o, d):
        o = np.ascontiguousarray(o, dtype=np.float64)
        d = np.ascontiguousarray(d, dtype=np.float64)
        return self.L.orc_locate_parity(self.h, _p(o), _p(d))

    def set_electron_mode(self, rho):
        """NEXT-4: straight CSDA electron segments instead of local deposit; rho = g/cm^3 per material, None = off."""
        if rho is None:
            assert self.L.orc_set_electron_mode(self.h, None, 0) == 0
        else:
            r = np.ascontiguousarray(rho, dtype=np.float64)
            assert self.L.orc_set_electron_mode(self.h, _p(r), len(r)) == 0

    def electron_split(self, pos, m, t_kin, seed, first, n):
        """Fraction of t_kin that stays in material m for electron 0 of histories first .. first+n-1 (test hook)."""
        out = np.empty(n)
        p = np.ascontiguousarray(pos, dtype=np.float64)
        self.L.orc_test_electron_split(self.h, _p(p), int(m), float(t_kin), seed, first, n, _p(out))
        return out

    def sample_source(self, seed, first, n):
        """O4 test hook: (line i32[n], pos f64[n,3], dir f64[n,3], draw u32[n]) of histories first .. first+n-1;
        draw = index of the first stream-0 draw after the source sampling."""
        line = np.empty(n, dtype=np.int32)
        pos = np.empty((n, 3))
        d = np.empty((n, 3))
        draw = np.empty(n, dtype=np.uint32)
        self.L.orc_test_source(self.h, seed, first, n, _p(line), _p(pos), _p(d), _p(draw))
        return line, pos, d, draw

    def run_histories(self, first, n, seed, details=False):
        edep = np.empty(n)
        flags = np.empty(n, dtype=np.uint32)
        other = np.empty(n) if details else None
        esc = np.empty(n) if details else None
        cnt = np.zeros(len(COUNTER_NAMES), dtype=np.uint64)
        rc = self.L.orc_run_histories(self.h, first, n, seed, _p(edep), _p(flags), _p(other), _p(esc), _p(cnt))
        assert rc == 0, rc
        counters = dict(zip(COUNTER_NAMES, (int(x) for x in cnt)))
        if details:
            return edep, flags, other, esc, counters
        return edep, flags, counters

    def run(self, n, seed, n_bins=4096, e_max_mev=2.0, first=0):
        spec = np.zeros(n_bins + 1, dtype=np.uint64)
        emitted = np.zeros(self.n_lines, dtype=np.uint64)
        peak = np.zeros(self.n_lines, dtype=np.uint64)
        cnt = np.zeros(len(COUNTER_NAMES), dtype=np.uint64)
        rc = self.L.orc_run(self.h, first, n, seed, n_bins, e_max_mev, _p(spec), _p(emitted), _p(peak), _p(cnt))
        assert rc == 0, rc
        return spec, emitted, peak, dict(zip(COUNTER_NAMES, (int(x) for x in cnt)))


def fepe(spectrum, emitted, peak, line_mev, line, mode=0, e_max_mev=2.0):
    """O14: full-energy-peak efficiency of one line and its binomial standard error.
    mode 0: exact counters, peak[l] / emitted[l].  mode 1: read from the spectrum, the line's bin b_l = floor(E_l / dE)
    (computed in double) minus the mean of its two neighbours, over emitted[l]."""
    em = float(emitted[line])
    if em <= 0:
        return 0.0, 0.0
    if mode == 0:
        p = float(peak[line]) / em
    else:
        n_bins = len(spectrum) - 1
        b = int(np.floor(float(line_mev[line]) / (e_max_mev / n_bins)))
        assert 1 <= b < n_bins - 1
        p = (float(spectrum[b]) - 0.5 * (float(spectrum[b - 1]) + float(spectrum[b + 1]))) / em
    return p, float(np.sqrt(max(p * (1.0 - p), 0.0) / em))


def tally(edep, flags, line_mev, n_bins=4096, e_max_mev=2.0):
    """O14 on a per-history dump (what orc_run does inside C, restated for dumps that were produced in chunks):
    emitted[l] counts every history of line l, peak[l] the full-absorption ones; a history with E_dep > 0 goes to bin
    floor(E_dep / dE), the last slot takes E_dep >= e_max.  `edep` is the dump's value: E_line for a peak history."""
    edep = np.asarray(edep, dtype=np.float64)
    flags = np.asarray(flags, dtype=np.uint32)
    n_lines = len(line_mev)
    line = ((flags >> 8) & 0xFF).astype(np.int64)
    emitted = np.bincount(line, minlength=n_lines).astype(np.uint64)
    peak = np.bincount(line[(flags & F_PEAK) != 0], minlength=n_lines).astype(np.uint64)
    pos = edep > 0.0
    b = np.floor(edep[pos] / (e_max_mev / n_bins))
    b = np.where(b >= n_bins, n_bins, b).astype(np.int64)
    spectrum = np.bincount(b, minlength=n_bins + 1).astype(np.uint64)
    return spectrum, emitted, peak
