"""Writes the stored oracle results under tests/golden/ (calls only detmesh/ and oracle/, never the CUDA path).

    python tests/golden/make_golden.py <config> <n_histories> [n_theta total_bands]

Output: tests/golden/cfg<config>_oracle_n<n>.json -- spectrum[4097], emitted[L], peak[L], event counters of
`OracleScene.run(n, seed=1)` on the BASELINE.json workload.  No value in these files comes from the
paper (it prints no numeric FEPE or spectrum): they are oracle outputs, used by the -m gpu parity tests at sizes the
oracle cannot finish inside a test.
"""
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import detmesh as dm                       # noqa: E402
from oracle import gadep_oracle as orc    # noqa: E402


def main():
    cfg, n = int(sys.argv[1]), int(float(sys.argv[2]))
    kw = {}
    if len(sys.argv) > 4:
        kw = {"n_theta": int(sys.argv[3]), "total_bands": int(sys.argv[4])}
    w = dm.make_config(cfg, **kw)
    s = orc.OracleScene(w)
    t0 = time.time()
    spec, emitted, peak, cnt = s.run(n, w.seed, w.n_bins, w.spectrum_e_max_mev)
    dt = time.time() - t0
    out = {"config": cfg, "workload": w.name, "n_histories": n, "seed": w.seed, "n_tri": w.mesh.n_tri,
           "tessellation": kw, "n_bins": w.n_bins, "e_max_mev": w.spectrum_e_max_mev,
           "oracle_seconds": round(dt, 2), "oracle_threads": orc.num_threads(),
           "line_mev": [float(x) for x in w.source["line_mev"]],
           "emitted": [int(x) for x in emitted], "peak": [int(x) for x in peak], "counters": cnt,
           "spectrum": [int(x) for x in spec]}
    tag = f"cfg{cfg}_oracle_n{n}" + (f"_nt{kw['n_theta']}_b{kw['total_bands']}" if kw else "")
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), tag + ".json")
    with open(path, "w") as f:
        json.dump(out, f, separators=(",", ":"))
        f.write("\n")
    print(path, dt)


if __name__ == "__main__":
    main()
