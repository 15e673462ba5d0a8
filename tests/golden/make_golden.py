"""Writes the stored oracle results under tests/golden/ (calls only detmesh/ and oracle/, never the CUDA path).

    python tests/golden/make_golden.py <config> <n_histories> [--nt N_THETA --bands TOTAL_BANDS] [--coh COEFF]
    python tests/golden/make_golden.py rays <n_rays>

Histories: tests/golden/cfg<config>[_coh<coeff>]_oracle_n<n>[_nt.._b..].json -- spectrum[4097], emitted[L], peak[L] and
the event counters of histories [0, n) of the BASELINE.json workload under seed `w.seed`, run through
`OracleScene.run_histories` in chunks and tallied with `oracle.tally` (O14).  For n <= 2e6 the per-history dump
(flags u32, deposit f32) goes to a .npz beside it, so that a GPU run of the same histories (common random numbers,
SURVEY.md Q14) can be compared history by history.
Rays: tests/golden/cfg4_rays_n<n>.npz -- brute-force nearest facet (index, distance) of the first n seeded rays of
BASELINE.json configs[4] on the full 2.0 M-facet mesh (`detmesh.configs.make_rays` with the workload's ray seed).
No value in these files comes from the paper (it prints no numeric FEPE or spectrum): they are oracle outputs, used by
the -m gpu parity tests at sizes the oracle cannot finish inside a test.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import detmesh as dm                       # noqa: E402
from oracle import gadep_oracle as orc    # noqa: E402

CHUNK = 50_000


def golden_tag(cfg, n, n_theta=None, bands=None, coh=None):
    tag = f"cfg{cfg}" + (f"_coh{coh:.1e}" if coh is not None else "") + f"_oracle_n{n}"
    return tag + (f"_nt{n_theta}_b{bands}" if n_theta else "")


def histories(cfg, n, n_theta, bands, coh):
    kw = {}
    if n_theta:
        kw.update(n_theta=n_theta, total_bands=bands)
    if coh is not None:
        kw.update(coh_coeff=coh)
    w = dm.make_config(cfg, **kw)
    s = orc.OracleScene(w)
    t0 = time.time()
    edep = np.empty(n, dtype=np.float64)
    flags = np.empty(n, dtype=np.uint32)
    counters = {}
    for first in range(0, n, CHUNK):
        m = min(CHUNK, n - first)
        e, f, c = s.run_histories(first, m, w.seed)
        edep[first:first + m] = e
        flags[first:first + m] = f
        for k, v in c.items():
            counters[k] = counters.get(k, 0) + v
        print(f"  {first + m}/{n}  {time.time() - t0:.0f} s", flush=True)
    spec, emitted, peak = orc.tally(edep, flags, w.source["line_mev"], w.n_bins, w.spectrum_e_max_mev)
    dt = time.time() - t0
    tag = golden_tag(cfg, n, n_theta, bands, coh)
    out = {"config": cfg, "workload": w.name, "n_histories": n, "seed": w.seed, "first_history": 0, "n_tri": w.mesh.n_tri,
           "tessellation": {"n_theta": n_theta, "total_bands": bands} if n_theta else {},
           "coh_coeff": coh, "n_bins": w.n_bins, "e_max_mev": w.spectrum_e_max_mev,
           "oracle_seconds": round(dt, 2), "oracle_threads": orc.num_threads(),
           "line_mev": [float(x) for x in w.source["line_mev"]],
           "emitted": [int(x) for x in emitted], "peak": [int(x) for x in peak], "counters": counters,
           "spectrum": [int(x) for x in spec], "per_history": None}
    if n <= 2_000_000:
        out["per_history"] = tag + "_hist.npz"
        np.savez_compressed(os.path.join(HERE, out["per_history"]), flags=flags, edep=edep.astype(np.float32))
    with open(os.path.join(HERE, tag + ".json"), "w") as f:
        json.dump(out, f, separators=(",", ":"))
        f.write("\n")
    print(tag, dt)


def rays(n):
    w = dm.make_config(4)
    s = orc.OracleScene(w)
    R, z0, z1 = w.notes["ray_box"]
    org, d = dm.configs.make_rays(n, w.notes["ray_seed"], R, z0, z1)
    tri = np.empty(n, dtype=np.int32)
    t = np.empty(n, dtype=np.float64)
    t0 = time.time()
    for first in range(0, n, CHUNK):
        m = min(CHUNK, n - first)
        tri[first:first + m], t[first:first + m] = s.trace_rays(org[first:first + m], d[first:first + m])
        print(f"  {first + m}/{n}  {time.time() - t0:.0f} s", flush=True)
    np.savez_compressed(os.path.join(HERE, f"cfg4_rays_n{n}.npz"), tri=tri, t=t, n_tri=np.int64(w.mesh.n_tri),
                        ray_seed=np.int64(w.notes["ray_seed"]), oracle_seconds=np.float64(time.time() - t0))
    print("rays", n, time.time() - t0)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("what")
    ap.add_argument("n", type=float)
    ap.add_argument("--nt", type=int, default=None)
    ap.add_argument("--bands", type=int, default=None)
    ap.add_argument("--coh", type=float, default=None)
    a = ap.parse_args()
    if a.what == "rays":
        rays(int(a.n))
    else:
        histories(int(a.what), int(a.n), a.nt, a.bands, a.coh)


if __name__ == "__main__":
    main()
