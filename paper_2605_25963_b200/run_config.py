"""Runs one of the BASELINE.json set-ups once and prints time and counters -- the smallest command to put under a
profiler (the ncu captures under profiles/ name it).

    python -m paper_2605_25963_b200.run_config <config 0..4> <n_histories> [--coh COEFF] [--bvh-width 4|5|8] [--flags N]
                                               [--build-flags 0|1|2]     (1 = plane lists with the build, 2 = never)
    python -m paper_2605_25963_b200.run_config <config> --rays <n_rays> [--bvh-width 4|5|8]

Histories: gadep_load_mesh / gadep_build_bvh / gadep_set_source, then ONE gadep_run of n_histories (no warm-up launch, so
the transport kernel of interest is the first `gd_k_transport_wave` launch of the process).  Rays: ONE gadep_trace_rays
of n seeded isotropic rays from the endcap's bounding cylinder (the config-4 ray benchmark's recipe) on the config's mesh.
"""
import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", type=int)
    ap.add_argument("n_histories", type=float, nargs="?", default=0)
    ap.add_argument("--coh", type=float, default=None)
    ap.add_argument("--bvh-width", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0)
    ap.add_argument("--rays", type=float, default=0)
    ap.add_argument("--build-flags", type=int, default=0)
    a = ap.parse_args()
    import torch
    import detmesh as dm
    import paper_2605_25963_b200 as pkg
    w = dm.make_config(a.config) if a.coh is None else dm.make_config(a.config, coh_coeff=a.coh)
    g = pkg.Gadep(0, torch.cuda.current_stream().cuda_stream)
    g.load_workload(w, build_flags=a.build_flags)
    if a.bvh_width:
        g.set_bvh_width(a.bvh_width)
    if a.rays:
        n = int(a.rays)
        org, d = dm.configs.make_rays(n, 1, 41.9, -101.9, 6.0)
        to, td = torch.from_numpy(org).cuda(), torch.from_numpy(d).cuda()
        tri = torch.empty(n, dtype=torch.int32, device="cuda")
        t = torch.empty(n, dtype=torch.float32, device="cuda")
        g.trace_rays(to, td, tri_out=tri, t_out=t)
        c = g.get_counters()
        print(json.dumps({"workload": w.name, "n_rays": n, "bvh_width": a.bvh_width or 4, "kernel_ms": c["last_run_ms"],
                          "box_tests_per_ray": c["n_box_tests"] / n, "tri_tests_per_ray": c["n_tri_tests"] / n}))
        return
    n = int(a.n_histories) if a.n_histories else w.n_histories
    g.run(n, w.seed, w.n_bins, w.spectrum_e_max_mev, flags=a.flags)
    c = g.get_counters()
    keep = ("n_histories", "n_queries", "n_skipped_queries", "n_box_tests", "n_tri_tests", "n_crossings", "n_pe", "n_compton",
            "n_coherent", "n_pair", "n_escaped", "n_leak", "last_run_ms", "last_build_ms", "n_grid_lists")
    print(json.dumps({"workload": w.name, **{k: c[k] for k in keep}, "fepe": [g.fepe(l)[0] for l in range(c["n_lines"])]}))


if __name__ == "__main__":
    main()
