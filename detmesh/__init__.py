"""DetMesh-style host-side input generators (outside the hot path).

Seeded, synthetic inputs shared by the CUDA path and by the CPU oracle:
closed triangulated detector surfaces (Eq. 1-6), per-material
attenuation tables (BASELINE.json configs[0..1]) and the five source/detector
set-ups of BASELINE.json.  Nothing in here performs transport arithmetic.
"""
from .geometry import (Line, Arc, discretise, revolve, Mesh, merge_surfaces,
                       mesh_signed_volume, mesh_area, check_closed_oriented)
from .materials import (ELEMENTS, MATERIALS, MAT, DENSITY_G_CM3, energy_grid, sigma_kn_total,
                        make_tables, N_GRID, E_MIN_MEV, E_MAX_MEV)
from .configs import make_config, make_calibration, make_calibration_batch, make_pellet_stack, Workload, philox_u01_host, TABLE3_KEV, CALIBRATION_DETECTORS

__all__ = [
    "Line", "Arc", "discretise", "revolve", "Mesh", "merge_surfaces",
    "mesh_signed_volume", "mesh_area", "check_closed_oriented",
    "ELEMENTS", "MATERIALS", "MAT", "DENSITY_G_CM3", "energy_grid", "sigma_kn_total", "make_tables",
    "N_GRID", "E_MIN_MEV", "E_MAX_MEV", "make_config", "make_calibration", "make_calibration_batch", "make_pellet_stack", "Workload", "philox_u01_host",
    "TABLE3_KEV", "CALIBRATION_DETECTORS",
]
