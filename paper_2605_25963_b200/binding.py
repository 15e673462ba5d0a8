"""ctypes binding of include/gadep.h -- same names, argument marshalling only.

PyTorch is used by callers for device memory and streams (`tensor.data_ptr()`,
`torch.cuda.current_stream().cuda_stream`); this module itself needs only numpy and ctypes.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB, build_library

F_ESCAPED, F_PEAK, F_LEAK, F_NONSCORING = 1, 2, 4, 8
FILTER_NONE = -2
STATIC_MAX_RAYS = 1 << 18      # GADEP_STATIC_MAX_RAYS of include/gadep.h
MAT_KILL = -1
MAX_LINES = 64
RUN_ASYNC, RUN_ACCUMULATE, RUN_HISTORY_PER_THREAD, RUN_PERSISTENT_LANES, RUN_PARITY_LOCALISATION = 1, 2, 4, 8, 16
RUN_PARTIAL_XS = 32
RUN_WARP_SPECIALISED = 64
RUN_BVH8 = 256
RUN_ELECTRON_RANGE = 128
BUILD_PLANE_LISTS, BUILD_NO_PLANE_LISTS = 1, 2

EXPORTED_SYMBOLS = ("gadep_create", "gadep_destroy", "gadep_last_error", "gadep_set_materials", "gadep_load_mesh",
                    "gadep_build_bvh", "gadep_set_source", "gadep_run", "gadep_fepe", "gadep_trace_rays",
                    "gadep_run_histories", "gadep_get_counters", "gadep_philox_raw", "gadep_locate", "gadep_broaden",
                    "gadep_set_densities", "gadep_run_histories_ex", "gadep_set_bvh_width", "gadep_tally_size",
                    "gadep_get_tallies", "gadep_set_tallies", "gadep_set_source_copies", "gadep_trace_rays_static")


class GadepError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"gadep error {code}: {text}")
        self.code = code


class GadepSource(C.Structure):
    _fields_ = [("kind", C.c_int), ("pos", C.c_float * 3), ("dir", C.c_float * 3),
                ("cyl_r", C.c_float), ("cyl_z0", C.c_float), ("cyl_z1", C.c_float),
                ("ex_r", C.c_float), ("ex_z0", C.c_float), ("ex_z1", C.c_float),
                ("n_lines", C.c_int), ("line_mev", C.c_void_p), ("line_intensity", C.c_void_p)]


class GadepRunOpts(C.Structure):
    _fields_ = [("n_bins", C.c_int), ("e_max_mev", C.c_float), ("first_history", C.c_ulonglong), ("flags", C.c_int)]


class GadepCounters(C.Structure):
    _fields_ = [(n, C.c_ulonglong) for n in ("n_histories", "n_queries", "n_box_tests", "n_tri_tests", "n_crossings",
                                             "n_pe", "n_compton", "n_coherent", "n_pair", "n_escaped", "n_leak",
                                             "n_cutoff")] + \
               [("emitted", C.c_ulonglong * MAX_LINES), ("peak", C.c_ulonglong * MAX_LINES), ("n_lines", C.c_int),
                ("n_bvh_nodes", C.c_int), ("bvh_max_depth", C.c_int), ("last_run_ms", C.c_float),
                ("last_build_ms", C.c_float), ("last_run_launches", C.c_int), ("last_build_launches", C.c_int),
                ("n_skipped_queries", C.c_ulonglong), ("n_stack_overflow", C.c_ulonglong),
                ("n_parity_queries", C.c_ulonglong), ("n_parity_mismatch", C.c_ulonglong),
                ("n_grid_list_cells", C.c_uint), ("n_grid_lists", C.c_uint)]

    def as_dict(self):
        d = {n: int(getattr(self, n)) for n, _ in self._fields_[:12]}
        nl = int(self.n_lines)
        d.update(emitted=[int(x) for x in self.emitted[:nl]], peak=[int(x) for x in self.peak[:nl]], n_lines=nl,
                 n_bvh_nodes=int(self.n_bvh_nodes), bvh_max_depth=int(self.bvh_max_depth),
                 last_run_ms=float(self.last_run_ms), last_build_ms=float(self.last_build_ms),
                 last_run_launches=int(self.last_run_launches), last_build_launches=int(self.last_build_launches),
                 n_skipped_queries=int(self.n_skipped_queries), n_stack_overflow=int(self.n_stack_overflow),
                 n_parity_queries=int(self.n_parity_queries), n_parity_mismatch=int(self.n_parity_mismatch),
                 n_grid_list_cells=int(self.n_grid_list_cells), n_grid_lists=int(self.n_grid_lists))
        return d


_lib = None


def library_path() -> str:
    return LIB


def load_library(build_if_missing: bool = True):
    """Loads libgadep.so (building it with nvcc if it is missing or stale).  Fails loudly otherwise."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        try:
            build_library()
        except Exception as e:  # nvcc missing on a deployment box: the shipped .so must then exist
            if not os.path.exists(LIB):
                raise RuntimeError(f"libgadep.so is missing and could not be built: {e}") from e
    if not os.path.exists(LIB):
        raise RuntimeError("libgadep.so is missing: run `python -m paper_2605_25963_b200.build` (there is no CPU fallback)")
    L = C.CDLL(LIB)
    vp, i32, f32, dbl, ull, ll = C.c_void_p, C.c_int, C.c_float, C.c_double, C.c_ulonglong, C.c_longlong
    L.gadep_create.argtypes = [C.POINTER(vp), i32, vp]
    L.gadep_destroy.argtypes = [vp]
    L.gadep_destroy.restype = None
    L.gadep_last_error.argtypes = [vp]
    L.gadep_last_error.restype = C.c_char_p
    L.gadep_set_materials.argtypes = [vp, i32, i32, dbl, dbl, vp, vp]
    L.gadep_load_mesh.argtypes = [vp, vp, i32, vp, vp, i32, vp, vp, i32, i32]
    L.gadep_build_bvh.argtypes = [vp, i32]
    L.gadep_set_source.argtypes = [vp, C.POINTER(GadepSource)]
    L.gadep_run.argtypes = [vp, ull, ull, C.POINTER(GadepRunOpts), vp]
    L.gadep_fepe.argtypes = [vp, i32, i32, C.POINTER(dbl), C.POINTER(dbl)]
    L.gadep_trace_rays.argtypes = [vp, vp, vp, ll, i32, f32, vp, vp]
    L.gadep_trace_rays_static.argtypes = [vp, vp, vp, ll, i32, f32, vp, vp]
    L.gadep_run_histories.argtypes = [vp, ull, ll, ull, vp, vp]
    L.gadep_run_histories_ex.argtypes = [vp, ull, ll, ull, C.c_int, vp, vp]
    L.gadep_set_densities.argtypes = [vp, C.c_int, vp]
    L.gadep_get_counters.argtypes = [vp, C.POINTER(GadepCounters)]
    L.gadep_philox_raw.argtypes = [vp, vp, vp, i32, vp]
    L.gadep_locate.argtypes = [vp, vp, vp, ll, i32, vp]
    L.gadep_broaden.argtypes = [vp, dbl, dbl, dbl, vp]
    L.gadep_set_bvh_width.argtypes = [vp, i32]
    L.gadep_set_source_copies.argtypes = [vp, i32, vp]
    L.gadep_tally_size.argtypes = [vp]
    L.gadep_get_tallies.argtypes = [vp, vp]
    L.gadep_set_tallies.argtypes = [vp, vp]
    _lib = L
    return L


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _ptr(x):
    """numpy array -> host pointer; object with data_ptr() (torch tensor) -> its pointer; int -> as is."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        return x.ctypes.data_as(C.c_void_p)
    if hasattr(x, "data_ptr"):
        return C.c_void_p(x.data_ptr())
    return C.c_void_p(int(x))


class Gadep:
    """One context = one device + one stream.  Method names mirror the C entry points."""

    def __init__(self, device: int = 0, stream: int = 0):
        self.L = load_library()
        self.h = C.c_void_p()
        rc = self.L.gadep_create(C.byref(self.h), int(device), C.c_void_p(int(stream)))
        if rc != 0:
            raise GadepError(rc, "gadep_create failed (no CUDA device? there is no CPU fallback)")
        self._keep = []

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.gadep_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise GadepError(rc, self.L.gadep_last_error(self.h).decode())

    # ---- set-up
    def set_materials(self, mu, is_scoring, e_min_mev, e_max_mev):
        mu = np.ascontiguousarray(mu, dtype=np.float32)
        sc = np.ascontiguousarray(is_scoring, dtype=np.uint8)
        self._check(self.L.gadep_set_materials(self.h, mu.shape[0], mu.shape[2], e_min_mev, e_max_mev, _np_ptr(mu),
                                               _np_ptr(sc)))

    def load_mesh(self, vertices, triangles, tri_surface, surf_inside, surf_outside, world_material):
        v = np.ascontiguousarray(vertices, dtype=np.float32)
        t = np.ascontiguousarray(triangles, dtype=np.int32)
        ts = np.ascontiguousarray(tri_surface, dtype=np.int32)
        si = np.ascontiguousarray(surf_inside, dtype=np.int32)
        so = np.ascontiguousarray(surf_outside, dtype=np.int32)
        self._check(self.L.gadep_load_mesh(self.h, _np_ptr(v), v.shape[0], _np_ptr(t), _np_ptr(ts), t.shape[0],
                                           _np_ptr(si), _np_ptr(so), si.shape[0], int(world_material)))

    def build_bvh(self, flags: int = 0):
        self._check(self.L.gadep_build_bvh(self.h, flags))

    def set_source(self, kind, pos=(0, 0, 0), dir=(0, 0, -1), cyl_r=0.0, cyl_z0=0.0, cyl_z1=0.0, ex_r=0.0, ex_z0=0.0,
                   ex_z1=0.0, line_mev=None, line_intensity=None):
        le = np.ascontiguousarray(line_mev, dtype=np.float32)
        li = np.ascontiguousarray(line_intensity, dtype=np.float32)
        s = GadepSource()
        s.kind = int(kind)
        s.pos = (C.c_float * 3)(*[float(x) for x in pos])
        s.dir = (C.c_float * 3)(*[float(x) for x in dir])
        s.cyl_r, s.cyl_z0, s.cyl_z1 = float(cyl_r), float(cyl_z0), float(cyl_z1)
        s.ex_r, s.ex_z0, s.ex_z1 = float(ex_r), float(ex_z0), float(ex_z1)
        s.n_lines = le.shape[0]
        s.line_mev = le.ctypes.data
        s.line_intensity = li.ctypes.data
        self._check(self.L.gadep_set_source(self.h, C.byref(s)))
        self.n_lines = le.shape[0]

    def load_workload(self, w, build=True, build_flags=0):
        """Convenience: all set-up calls for a detmesh.Workload-like object."""
        self.set_materials(w.mu, w.is_scoring, w.e_min_mev, w.e_max_mev)
        m = w.mesh
        self.load_mesh(m.vertices, m.triangles, m.tri_surface, m.surf_inside, m.surf_outside, m.world_material)
        if build:
            self.build_bvh(build_flags)
        self.set_source(**w.source)
        if getattr(w, "notes", None) and w.notes.get("source_copies") is not None:
            self.set_source_copies(w.notes["source_copies"])

    def set_source_copies(self, offsets):
        """Replicate the source at these translations ([n][3]); None = the plain source."""
        if offsets is None:
            self._check(self.L.gadep_set_source_copies(self.h, 1, None))
            return
        off = np.ascontiguousarray(offsets, dtype=np.float32)
        self._check(self.L.gadep_set_source_copies(self.h, int(off.shape[0]), _np_ptr(off)))

    # ---- hot path
    def run(self, n_histories, seed, n_bins=4096, e_max_mev=2.0, first_history=0, flags=0, spectrum=None):
        """spectrum: None -> a new host uint64 array is returned; numpy array or device tensor/pointer -> filled."""
        opts = GadepRunOpts(int(n_bins), float(e_max_mev), int(first_history), int(flags))
        self._last_bins = int(n_bins)
        out = spectrum
        if out is None and not (int(flags) & RUN_ASYNC):
            out = np.zeros(n_bins + 1, dtype=np.uint64)
        # RUN_ASYNC without a device spectrum: nothing is copied out, the tallies stay in the context
        self._check(self.L.gadep_run(self.h, int(n_histories), int(seed), C.byref(opts), _ptr(out)))
        return out

    def fepe(self, line, mode=0):
        f, s = C.c_double(), C.c_double()
        self._check(self.L.gadep_fepe(self.h, int(line), int(mode), C.byref(f), C.byref(s)))
        return f.value, s.value

    def trace_rays(self, org, dir, filter_material=FILTER_NONE, t_min=0.0, tri_out=None, t_out=None):
        if isinstance(org, np.ndarray):
            org = np.ascontiguousarray(org, dtype=np.float32)
            dir = np.ascontiguousarray(dir, dtype=np.float32)
            n = org.shape[0]
            tri_out = np.empty(n, dtype=np.int32) if tri_out is None else tri_out
            t_out = np.empty(n, dtype=np.float32) if t_out is None else t_out
        else:
            n = org.shape[0]
            if tri_out is None or t_out is None:
                raise ValueError("device inputs need device outputs")
        self._check(self.L.gadep_trace_rays(self.h, _ptr(org), _ptr(dir), n, int(filter_material), float(t_min),
                                            _ptr(tri_out), _ptr(t_out)))
        return tri_out, t_out

    def trace_rays_static(self, org, dir, filter_material=FILTER_NONE, t_min=0.0, tri_out=None, t_out=None):
        """gadep_trace_rays_static: the same query without any device allocation (scratch in a static device array of
        the library, at most STATIC_MAX_RAYS rays per call; calls on one device must not overlap).  With numpy inputs
        and no outputs given, the two HOST result arrays are made here, by the caller's side."""
        if isinstance(org, np.ndarray):
            org = np.ascontiguousarray(org, dtype=np.float32)
            dir = np.ascontiguousarray(dir, dtype=np.float32)
            n = org.shape[0]
            tri_out = np.empty(n, dtype=np.int32) if tri_out is None else tri_out
            t_out = np.empty(n, dtype=np.float32) if t_out is None else t_out
        else:
            n = org.shape[0]
            if tri_out is None or t_out is None:
                raise ValueError("device inputs need device outputs")
        self._check(self.L.gadep_trace_rays_static(self.h, _ptr(org), _ptr(dir), n, int(filter_material), float(t_min),
                                                   _ptr(tri_out), _ptr(t_out)))
        return tri_out, t_out

    def broaden(self, fwhm_a, fwhm_b=0.0, fwhm_c=0.0, out=None):
        """Spectrum of the last run with Gaussian resolution FWHM(E)^2 = a + b E + c E^2 (MeV); float64[n_bins+1]."""
        if out is None:
            out = np.empty(self._last_bins + 1, dtype=np.float64)
        self._check(self.L.gadep_broaden(self.h, float(fwhm_a), float(fwhm_b), float(fwhm_c), _ptr(out)))
        return out

    def locate(self, org, dir, mode=0, material_out=None):
        """Material containing each point (mode 0 side-id rule, 1 parity rule)."""
        if isinstance(org, np.ndarray):
            org = np.ascontiguousarray(org, dtype=np.float32)
            dir = np.ascontiguousarray(dir, dtype=np.float32)
            material_out = np.empty(org.shape[0], dtype=np.int32) if material_out is None else material_out
        elif material_out is None:
            raise ValueError("device inputs need a device output")
        self._check(self.L.gadep_locate(self.h, _ptr(org), _ptr(dir), org.shape[0], int(mode), _ptr(material_out)))
        return material_out

    def set_bvh_width(self, width: int):
        self._check(self.L.gadep_set_bvh_width(self.h, int(width)))

    def tally_size(self) -> int:
        return int(self.L.gadep_tally_size(self.h))

    def get_tallies(self, out=None):
        """spectrum[n_bins + 1] + emitted[64] + peak[64] of the context; out: None -> new host array, else filled."""
        if out is None:
            out = np.zeros(self.tally_size(), dtype=np.uint64)
        self._check(self.L.gadep_get_tallies(self.h, _ptr(out)))
        return out

    def set_tallies(self, tallies):
        self._check(self.L.gadep_set_tallies(self.h, _ptr(tallies)))

    def set_densities(self, rho_g_cm3):
        rho = np.ascontiguousarray(rho_g_cm3, dtype=np.float32)
        self._check(self.L.gadep_set_densities(self.h, int(len(rho)), _np_ptr(rho)))

    def run_histories(self, first, n, seed, flags=0):
        edep = np.empty(n, dtype=np.float32)
        run_flags = int(flags)
        flags = np.empty(n, dtype=np.uint32)
        self._check(self.L.gadep_run_histories_ex(self.h, int(first), int(n), int(seed), run_flags, _np_ptr(edep),
                                                  _np_ptr(flags)))
        return edep, flags

    def get_counters(self) -> dict:
        c = GadepCounters()
        self._check(self.L.gadep_get_counters(self.h, C.byref(c)))
        return c.as_dict()

    def philox_raw(self, ctr4, key2, which=0):
        c = np.ascontiguousarray(ctr4, dtype=np.uint32)
        k = np.ascontiguousarray(key2, dtype=np.uint32)
        out = np.zeros(4, dtype=np.uint32)
        self._check(self.L.gadep_philox_raw(self.h, _np_ptr(c), _np_ptr(k), int(which), _np_ptr(out)))
        return out
