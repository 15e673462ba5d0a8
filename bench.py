#!/usr/bin/env python
"""bench.py -- photon histories/s of the Gadep hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--histories 1e7] [--impl reference]

A step = one pass of the whole hot path over one batch: gadep_build_bvh + gadep_run of
`histories` photon histories (a1-a13) on the workload of BASELINE.json configs[config] (default configs[1], the
coaxial HPGe with 5 lines and 1e7 histories).  Inputs (mesh, tables) are resident in HBM for `value`; `e2e` repeats
the step through the C ABI from HOST buffers (tables + mesh uploaded, spectrum read back) with wall-clock timing.
For N > 1 (torchrun) every rank transports its own range of the global history index and the integer tallies are
summed with one NCCL all-reduce inside the timed region (weak scaling).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "photon histories/s"
UNIT = "histories/s"
# SURVEY.md 8(d) per-unit algorithmic work, FP32 lane-instructions
INSTR_BOX, INSTR_TRI, INSTR_EVENT, INSTR_QUERY = 15, 36, 250, 60


def load_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) > 8 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) > 8 and r[2].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) > 8:
                for k, nm in enumerate(names):
                    if r[5 + k].lower().startswith("active"):
                        reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(w, n_sample, first=0):
    """The oracle as it stands on the host cores: histories/s on a bounded sample of the same workload."""
    from oracle import gadep_oracle as orc
    s = orc.OracleScene(w)
    s.run(min(2000, n_sample), w.seed, w.n_bins, w.spectrum_e_max_mev)      # page in
    t0 = time.perf_counter()
    s.run(n_sample, w.seed, w.n_bins, w.spectrum_e_max_mev, first=first)
    dt = time.perf_counter() - t0
    return n_sample / dt, dt, orc.num_threads()


def run_reference(args, w, rank):
    """--impl reference: the CPU oracle, as it stands, on this box's host cores; rank 0 only."""
    if rank != 0:
        return
    n_sample = int(args.ref_sample)
    rates = []
    for _ in range(args.warmup):
        oracle_rate(w, max(n_sample // 10, 1000))
    t_all = 0.0
    for k in range(args.steps):
        r, dt, cores = oracle_rate(w, n_sample, first=k * n_sample)
        rates.append(r)
        t_all += dt
    value = n_sample * args.steps / t_all
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_all / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "histories_per_step": n_sample, "n_triangles": w.mesh.n_tri},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{n_sample} histories per step of {w.name}, brute-force double precision"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ray_bench(args, dm):
    """BASELINE.json configs[4]: seeded isotropic rays from random points inside the endcap's bounding cylinder through
    the 2 M-facet BVH (device arrays, CUDA events), the check of a sample against brute force is tests/test_gpu_parity.py::test_cfg4_full_size_rays."""
    import torch
    import paper_2605_25963_b200 as pkg
    w = dm.make_config(4)
    g = pkg.Gadep(0, torch.cuda.current_stream().cuda_stream)
    g.load_workload(w)
    n, chunk = int(args.ray_bench), 20_000_000
    t_ms, boxes, tris, done = 0.0, 0, 0, 0
    while done < n:
        m = min(chunk, n - done)
        org, d = dm.configs.make_rays(m, 1 + done // chunk, 41.9, -101.9, 6.0)
        to, td = torch.from_numpy(org).cuda(), torch.from_numpy(d).cuda()
        tri = torch.empty(m, dtype=torch.int32, device="cuda")
        t = torch.empty(m, dtype=torch.float32, device="cuda")
        if done == 0:
            g.trace_rays(to[:100000], td[:100000], tri_out=tri[:100000], t_out=t[:100000])      # warm-up
        g.trace_rays(to, td, tri_out=tri, t_out=t)
        c = g.get_counters()
        t_ms += c["last_run_ms"]; boxes += c["n_box_tests"]; tris += c["n_tri_tests"]
        done += m
    line = {"metric": "BVH nearest-hit rays/s", "value": n / (t_ms * 1e-3), "unit": "rays/s", "n_rays": n,
            "workload": w.name, "n_triangles": w.mesh.n_tri, "kernel_ms": t_ms, "box_tests_per_s": boxes / (t_ms * 1e-3),
            "tri_tests_per_s": tris / (t_ms * 1e-3), "bvh_build_ms": g.get_counters()["last_build_ms"]}
    print(json.dumps(line), flush=True)


def run_calibration(args, dm):
    """the paper's calibration use-case (Table 3, Fig. 11): one launch of 1e7
    histories per detector gives the full-energy-peak efficiency at the 13 calibration energies."""
    import torch
    import paper_2605_25963_b200 as pkg
    out = {"metric": "FEPE curves (13 energies per launch)", "energies_kev": list(dm.TABLE3_KEV), "detectors": []}
    for k in range(len(dm.CALIBRATION_DETECTORS)):
        w = dm.make_calibration(k, n_histories=int(args.histories) if args.histories else 10_000_000)
        g = pkg.Gadep(0, torch.cuda.current_stream().cuda_stream)
        g.load_workload(w)
        g.run(200_000, w.seed, w.n_bins, w.spectrum_e_max_mev)
        g.run(w.n_histories, w.seed, w.n_bins, w.spectrum_e_max_mev)
        c = g.get_counters()
        fe = [g.fepe(l) for l in range(13)]
        out["detectors"].append({"name": w.name, "n_triangles": w.mesh.n_tri, "histories": w.n_histories,
                                 "kernel_ms": c["last_run_ms"], "bvh_build_ms": c["last_build_ms"],
                                 "histories_per_s": w.n_histories / (c["last_run_ms"] * 1e-3),
                                 "fepe": [f for f, _ in fe], "fepe_std_err": [s_ for _, s_ in fe]})
    print(json.dumps(out), flush=True)


def run_locate_bench(args, dm):
    """cost of the paper's reworked localisation (parity counting over all facets hit, an
    all-hits BVH traversal) against its original side-id rule (nearest facet), on the config-1 detector at the
    standard tessellation and at 3x the angular segments (the paper's facet-count sensitivity experiment)."""
    import torch
    import paper_2605_25963_b200 as pkg
    n = int(args.locate_bench)
    out = {"metric": "localisation queries/s", "unit": "queries/s", "n_points": n, "cases": []}
    for nt in (256, 768):
        w = dm.make_config(1, n_theta=nt)
        g = pkg.Gadep(0, torch.cuda.current_stream().cuda_stream)
        g.load_workload(w)
        org, d = dm.configs.make_rays(n, 3, 45.0, -105.0, 10.0)
        to, td = torch.from_numpy(org).cuda(), torch.from_numpy(d).cuda()
        mat = torch.empty(n, dtype=torch.int32, device="cuda")
        case = {"n_theta": nt, "n_triangles": w.mesh.n_tri}
        res = {}
        for mode, name in ((0, "side_id"), (1, "parity")):
            g.locate(to[:10000], td[:10000], mode, material_out=mat[:10000])
            g.locate(to, td, mode, material_out=mat)
            c = g.get_counters()
            res[name] = mat.cpu().numpy().copy()
            case[name] = {"queries_per_s": n / (c["last_run_ms"] * 1e-3), "kernel_ms": c["last_run_ms"],
                          "box_tests_per_query": c["n_box_tests"] / n, "tri_tests_per_query": c["n_tri_tests"] / n}
        case["parity_over_side_id_time"] = case["parity"]["kernel_ms"] / case["side_id"]["kernel_ms"]
        case["rules_disagree"] = int((res["side_id"] != res["parity"]).sum())
        out["cases"].append(case)
    a, b = out["cases"]
    out["facets_x3_time_increase"] = {k: b[k]["kernel_ms"] / a[k]["kernel_ms"] - 1.0 for k in ("side_id", "parity")}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--histories", type=float, default=0, help="per GPU per step; 0 = the config's own count")
    ap.add_argument("--impl", default="gadep")
    ap.add_argument("--ref-sample", type=float, default=60000)
    ap.add_argument("--cpu-sample", type=float, default=0, help="oracle histories; 0 = sized for ~15 s from a pilot run")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--calibration", action="store_true", help="FEPE curves: 13 Table-3 energies x 3 parametric detectors")
    ap.add_argument("--locate-bench", type=float, default=0, help="localisation benchmark: side-id vs parity rule (PAPER.md:191-193)")
    ap.add_argument("--ray-bench", type=float, default=0, help="config-4 ray benchmark: this many seeded rays through gadep_trace_rays")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    import detmesh as dm
    w = dm.make_config(args.config)
    if args.impl == "reference":
        run_reference(args, w, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2605_25963_b200 as pkg
    from paper_2605_25963_b200.sharding import allreduce_tallies

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if args.ray_bench:
        run_ray_bench(args, dm)
        return
    if args.locate_bench:
        run_locate_bench(args, dm)
        return
    if args.calibration:
        run_calibration(args, dm)
        return
    n_hist = int(args.histories) if args.histories else w.n_histories
    stream = torch.cuda.current_stream()
    g = pkg.Gadep(local_rank, stream.cuda_stream)
    g.load_workload(w)                                           # inputs resident in HBM from here on
    n_tally = w.n_bins + 1
    d_spec = torch.zeros(n_tally, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    first = rank * n_hist                                        # weak scaling: every rank its own histories

    def step(k):
        g.build_bvh()                                            # a0
        g.run(n_hist, w.seed, w.n_bins, w.spectrum_e_max_mev, first_history=first + k * world * n_hist,
              spectrum=d_spec)                                   # a1-a13, spectrum stays on the device
        if world > 1:
            allreduce_tallies(d_spec)

    for k in range(args.warmup):
        step(k)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms, build_ms, launches = [], [], 0
    agg = {}
    torch.cuda.synchronize()
    for k in range(args.steps):
        flush.fill_(k & 0xFF)                                    # L2 flush between timed iterations (untimed)
        ev[k][0].record(stream)
        step(args.warmup + k)
        ev[k][1].record(stream)
        c = g.get_counters()
        kern_ms.append(c["last_run_ms"]); build_ms.append(c["last_build_ms"])
        launches += c["last_run_launches"] + c["last_build_launches"]
        for key in ("n_queries", "n_box_tests", "n_tri_tests", "n_pe", "n_compton", "n_coherent", "n_pair", "n_crossings"):
            agg[key] = agg.get(key, 0) + c[key]
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    t = torch.tensor([t_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    t_ms = float(t.item())
    value = world * n_hist * args.steps / (t_ms * 1e-3)

    # ---- e2e: same step through the C ABI from HOST buffers (tables + mesh up, spectrum down), wall clock
    m = w.mesh
    h2d = int(w.mu.nbytes + w.is_scoring.nbytes + m.vertices.nbytes + m.triangles.nbytes + m.tri_surface.nbytes
              + m.surf_inside.nbytes + m.surf_outside.nbytes + w.source["line_mev"].nbytes * 2)
    d2h = int(8 * n_tally)
    g2 = pkg.Gadep(local_rank, stream.cuda_stream)
    e2e_steps = 3                                                # median of three: one wall-clock hiccup does not count
    g2.load_workload(w); g2.run(min(n_hist, 100000), w.seed)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    e2e_times = []
    for k in range(e2e_steps):
        t0 = time.perf_counter()
        g2.load_workload(w)                                      # host arrays -> device, validation, BVH build
        h_spec = g2.run(n_hist, w.seed, w.n_bins, w.spectrum_e_max_mev, first_history=first)   # host spectrum out
        fepe = [g2.fepe(l)[0] for l in range(len(w.source["line_mev"]))]
        torch.cuda.synchronize()
        e2e_times.append(time.perf_counter() - t0)
    # wall clock on a shared host: the median step, times the number of steps, guards against a single hiccup
    e2e_t = torch.tensor([float(np.median(e2e_times)) * e2e_steps], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    e2e_value = world * n_hist * e2e_steps / float(e2e_t.item())

    if rank == 0:
        peaks, peak_src = load_peaks()
        n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
        alu_peak = n_sm * 128 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12         # T lane-instr/s
        events = agg["n_pe"] + agg["n_compton"] + agg["n_coherent"] + agg["n_pair"]
        work = (agg["n_box_tests"] * INSTR_BOX + agg["n_tri_tests"] * INSTR_TRI + events * INSTR_EVENT
                + agg["n_queries"] * INSTR_QUERY)
        k_s = sum(kern_ms) * 1e-3
        achieved = work / k_s / 1e12
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "histories_per_step_per_gpu": n_hist, "n_triangles": m.n_tri,
                           "seed": w.seed, "l2": "flushed between timed steps (256 MiB write)",
                           "step": "gadep_build_bvh + gadep_run", "parallelism": f"history-sharded x{world}"},
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "steps": e2e_steps, "fepe": fepe},
                "gpu_launches": launches,
                "clocks": clocks,
                "roofline": {"bound": "alu", "kernel": "gd_k_transport_wave", "achieved": achieved, "peak": alu_peak,
                             "unit": "Tinstr/s (FP32 lane-instructions)", "frac": achieved / alu_peak,
                             "traffic": 14633984 if args.config == 1 and n_hist == 10_000_000 else None,
                             "traffic_source": "profiles/r01k_wave_kernel.md (ncu dram bytes of one launch)",
                             "limiter": "L1 data pipe: l1tex__throughput 84 % of peak in the stand-alone traversal kernel, "
                                        "51 % over a whole 1e7-history launch (ncu, profiles/r01f_trace_kernel.md, r01h)",
                             "peak_source": f"{n_sm} SMs x 128 lanes x sm_max_mhz ({peak_src})",
                             "kernel_ms_per_step": sum(kern_ms) / args.steps,
                             "bvh_build_ms_per_step": sum(build_ms) / args.steps,
                             "kernel_share_of_step": sum(kern_ms) / t_ms,
                             "box_tests_per_s": agg["n_box_tests"] / k_s, "tri_tests_per_s": agg["n_tri_tests"] / k_s,
                             "queries_per_s": agg["n_queries"] / k_s, "events_per_s": events / k_s},
                "paper_context": "RTX 4090: 1e8 particles in 66.08 s = 1.51e6 /s (PAPER.md:270), other physics"}
        if not args.no_cpu_baseline and world == 1:
            n_s = int(args.cpu_sample)
            if n_s <= 0:                                         # pilot -> about 15 s of CPU work
                r0, dt0, _ = oracle_rate(w, 20000)
                n_s = int(min(max(15.0 * r0, 20000), 5e7))
            r, dt, cores = oracle_rate(w, n_s)
            line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"first {n_s} histories of {w.name} ({dt:.1f} s)"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
