"""bench.py -- throughput of the SOP Langevin hot path (BASELINE.json metric: bead-steps/s, us per Langevin step,
fraction of the HBM roofline) on synthetic inputs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4] [--block B]

One bench "step" is one pass of the whole hot path over the workload: B Langevin steps (default 1000 = 10 pair-list
rebuilds a1+a2, 100 neighbor-list filters a3, 1000 fused force+noise+update steps a4..a9) plus one energy
reduction a10.  The default workload is config 3 of BASELINE.json (the 30,000-bead shell, the configuration the
north star's roofline target is quoted on); the other four configs are measured by the same routine, shorter, and
reported under "workloads" in the same JSON line (rank 0, N = 1 only).

Multi-GPU: the path shards across independent trajectories only, with
no collective on the data path.  With --gpus N the job is a batch of N x T trajectories of the workload; rank r
owns trajectories [r T, (r+1) T) through the Philox trajectory offset -> weak scaling.

--impl reference times the fp64 CPU oracle (oracle/), as it stands, on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "bead-steps/s"
NOMINAL_HBM_GBS = 8000.0          # the north star's figure; context only
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


# ---------------------------------------------------------------------------------------------- distributed glue
def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def max_over_ranks(x: float) -> float:
    import torch
    d = _dist()
    if d is None:
        return float(x)
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    import torch
    d = _dist()
    if d is None:
        return float(x)
    dev = "cuda" if d.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return float(t.item())


def barrier():
    d = _dist()
    if d is not None:
        d.barrier()


# ---------------------------------------------------------------------------------------------- helpers
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:  # noqa: BLE001
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def __enter__(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:  # noqa: BLE001
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:  # noqa: BLE001
                self.proc.kill()

    def summary(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.path or not os.path.exists(self.path):
            return out
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            f = [v.strip() for v in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower() == "active":
                    reasons.add(nme)
        os.unlink(self.path)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def list_stats(w, s):
    """Mean partners per bead (symmetric rows) of trajectory 0 at the current state -> algorithmic bytes."""
    N = w.n_beads
    nb = float(s.get_lists(2, 0, counts_only=True)[0].mean())
    pl = float(s.get_lists(1, 0, counts_only=True)[0].mean())
    return {"n_b": 2.0 * len(w.bonds) / N, "n_nat": 2.0 * len(w.native) / N, "n_nb": nb, "n_pl": pl}


def algorithmic_bytes(st, T, compensated, static_l1, p):
    """per bead-step of the fused step kernel, per bead of one L2
    filter, per bead of one L1 build.  Static tables are shared by the T trajectories of a batch."""
    b_fi = 16 + 16 + (32 if compensated else 0) + 4 * st["n_nb"] + (8 * st["n_nat"] + 8 * st["n_b"]) / T
    b_filter = 16 + 4 * st["n_pl"] / (T if static_l1 else 1) + 4 * st["n_nb"]
    b_l1 = 0.0 if static_l1 else 16 + 8 + 4 * st["n_pl"]
    per_step = b_fi + b_filter / p["nb_interval"] + b_l1 / p["pl_interval"]
    return {"B_fi": b_fi, "B_filter": b_filter, "B_l1": b_l1, "B_step": per_step}


def roofline_block(res, w, T, peak, peak_src):
    """The roofline record of one measured workload: algorithmic bytes / CUDA-event time of the step kernel /
    measured HBM copy peak, with every term it is made of, and the DRAM traffic of the committed ncu capture beside it."""
    sk = res.get("step_kernel")
    if not sk:
        return None
    ab, nbi = res["bytes"], w.params["nb_interval"]
    inside = sk["includes_l2_filter"]
    per_bead_step = ab["B_fi"] + (ab["B_filter"] / nbi if inside else 0.0)
    out = {"bound": "hbm",
           "kernel": "fused force+noise+update step kernel" + (" (persistent; L2 filter inside)" if inside else ""),
           "achieved": sk["achieved_gbs"], "peak": peak, "unit": "GB/s", "frac": sk["achieved_gbs"] / peak, "peak_source": peak_src,
           "frac_is": "ALGORITHMIC bytes / time / measured HBM copy peak (the working set is SM/L2 resident: see dram_frac and limited_by)",
           "frac_of_nominal_8TBs": sk["achieved_gbs"] / NOMINAL_HBM_GBS, "us_per_langevin_step": sk["us_per_langevin_step"],
           "bytes_per_bead_step": per_bead_step, "B_fi": ab["B_fi"], "B_filter_per_step": ab["B_filter"] / nbi if inside else 0.0,
           "bead_instances": w.n_beads * T, "traffic": None, "traffic_source": None, "algorithmic_bytes_per_launch": None}
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.json.txt")) as f:
            tr = json.load(f).get(w.name)
        if tr and res["resolved"]["mode"] == tr["mode"]:
            out["traffic"] = tr["dram_bytes_per_launch"]
            out["traffic_source"] = (f"ncu dram__bytes_read.sum + dram__bytes_write.sum of one {tr['kernel']} launch = "
                                     f"{tr['langevin_steps_per_launch']} Langevin steps ({tr['profile']})")
            out["algorithmic_bytes_per_launch"] = per_bead_step * w.n_beads * T * tr["langevin_steps_per_launch"]
            out["dram_frac"] = tr["dram_bytes_per_launch"] / (tr["langevin_steps_per_launch"] * sk["us_per_langevin_step"] * 1e-6) / 1e9 / peak
            out["limited_by"] = tr.get("limited_by")
    except Exception:  # noqa: BLE001
        pass
    return out


# ---------------------------------------------------------------------------------------------- our arm
def measure(w, T, traj_offset, block, K, W, clocks_index=None, e2e=True, overrides=None):
    """Time K bench steps of `block` Langevin steps (+ one energy reduction) on the current device."""
    import torch
    import paper_1003_1148_b200 as m

    s = m.from_workload(w, n_traj=T, traj_offset=traj_offset, **(overrides or {}))
    N = w.n_beads
    cfg = s.config()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def one_step():
        s.run(block)
        return s.get_energies()

    for _ in range(W):
        one_step()
    s.sync()
    s.set_profiling(True)
    s.get_profile()
    launches0 = s.config()["launches"]
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(clocks_index) if clocks_index is not None else None
    barrier(); torch.cuda.synchronize()
    if sampler:
        sampler.__enter__()
    for a, b in ev:
        flush.fill_(1)                      # L2 flush between timed steps, outside the event pair
        a.record(); one_step(); b.record()
    torch.cuda.synchronize()
    if sampler:
        sampler.__exit__()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    barrier()
    prof = s.get_profile()
    s.set_profiling(False)
    launches = s.config()["launches"] - launches0
    ms_max = max_over_ranks(ms)
    units = sum_over_ranks(float(N) * T * block * K)
    st = list_stats(w, s)
    ab = algorithmic_bytes(st, T, cfg["compensated"], math.isinf(w.params["R_pl"]), w.params)
    res = {
        "value": units / (ms_max * 1e-3), "ms_per_step": ms_max / K, "us_per_langevin_step": ms_max * 1e3 / (K * block),
        "launches": int(launches), "resolved": {k: cfg[k] for k in ("lanes_per_bead", "block_size", "compensated", "mode", "reorder", "resident_variant")},
        "list_stats": st, "bytes": ab, "profile": prof,
    }
    # force+integrate kernel alone (its own event spans inside the library, on the same stream)
    if prof["langevin_steps"] > 0 and prof["step_ms"] > 0:
        us_fi = prof["step_ms"] * 1e3 / prof["langevin_steps"]
        n_filters_inside = prof["langevin_steps"] // w.params["nb_interval"] if cfg["mode"] in (2, 3) else 0
        bytes_per_launch_step = N * T * (ab["B_fi"] + (ab["B_filter"] / w.params["nb_interval"] if cfg["mode"] in (2, 3) else 0.0))
        res["step_kernel"] = {"us_per_langevin_step": us_fi, "achieved_gbs": bytes_per_launch_step / (us_fi * 1e-6) / 1e9,
                              "includes_l2_filter": bool(n_filters_inside), "spans": prof["step_spans"]}
    if sampler:
        res["clocks"] = sampler.summary()

    if e2e:
        # the same metric through the C ABI with HOST buffers: coordinates in, B steps, coordinates + energies out
        x_host = s.get_coords()
        for _ in range(2):
            s.set_coords(x_host); s.run(block); s.get_coords(out=x_host); s.get_energies()
        barrier(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(K):
            s.set_coords(x_host)                      # H2D of this step's input (library stages through pinned memory)
            s.run(block)
            s.get_coords(out=x_host)                  # D2H of the result
            s.get_energies()
        b.record(); torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms_e = max_over_ranks(max(a.elapsed_time(b), wall * 1e3))
        res["e2e"] = {"value": units / (ms_e * 1e-3), "unit": METRIC,
                      "h2d_bytes_per_step": int(N * T * 16), "d2h_bytes_per_step": int(N * T * 16 + T * 48)}
    s.close()
    del flush
    return res


def cpu_sample(w, T, n_steps):
    """The oracle, as it stands, on the host cores: n_steps Langevin steps + one energy evaluation."""
    from oracle import sopo
    o = sopo.from_workload(w, n_traj=T, list_builder=1 if w.n_beads > 5000 else 0)
    t0 = time.perf_counter()
    o.run(n_steps)
    o.get_energies()
    dt = time.perf_counter() - t0
    cores = sopo.num_threads()
    o.close()
    return w.n_beads * T * n_steps / dt, dt, cores


# oracle sample sizes (Langevin steps) giving roughly 10-20 s on 8 cores; multiples of pl_interval
CPU_STEPS = {0: 40000, 1: 600, 2: 1200, 3: 1200, 4: 200}
CPU_TRAJ = {1: 8}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--block", type=int, default=1000, help="Langevin steps per bench step")
    ap.add_argument("--no-sweep", action="store_true", help="skip the other four configs")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--mode", type=int, default=0)
    ap.add_argument("--lanes", type=int, default=0)
    ap.add_argument("--variant", type=int, default=0, help="mode 3 with several chunks: resident_variant (1 first design, 2 second design)")
    ap.add_argument("--sweep4", action="store_true",
                    help="config 4's sweep of the parallelisation variant (BASELINE.json configs[4]): lanes per bead x block size")
    args = ap.parse_args()
    K, W = args.steps, max(args.warmup, 0)
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from workloads import generators as gen

    if args.impl == "reference":
        if rank != 0:
            return 0
        w = gen.make_config(args.config)
        T = CPU_TRAJ.get(args.config, 1)
        n = max(100, CPU_STEPS[args.config] // 4 // 100 * 100)
        for _ in range(W):
            cpu_sample(w, T, 100)
        vals, tot = [], 0.0
        for _ in range(K):
            v, dt, cores = cpu_sample(w, T, n)
            vals.append(v); tot += dt
        value = w.n_beads * T * n * K / tot
        sample = f"{T} trajectory(ies) x {n} Langevin steps of {w.name} per bench step (incl. list rebuilds + 1 energy evaluation)"
        print(json.dumps({
            "impl": "reference", "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": args.gpus, "steps": K,
            "warmup": W, "ms_per_step": tot * 1e3 / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_beads": w.n_beads, "n_traj": T, "langevin_steps_per_step": n},
            "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}))
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    over = {}
    if args.mode:
        over["mode"] = args.mode
    if args.lanes:
        over["lanes_per_bead"] = args.lanes
    if args.variant:
        over["resident_variant"] = args.variant
    w = gen.make_config(args.config)
    T = w.n_traj
    peak, peak_src = measured_peak()
    main_res = measure(w, T, rank * T, args.block, K, W, clocks_index=local_rank if rank == 0 else None, overrides=over)

    line = {
        "metric": METRIC, "value": main_res["value"], "unit": METRIC, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": main_res["ms_per_step"], "us_per_langevin_step": main_res["us_per_langevin_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "n_beads": w.n_beads, "n_traj_per_gpu": T, "langevin_steps_per_step": args.block,
                   "per_step": "B Langevin steps incl. every list rebuild + 1 energy reduction",
                   "parallelism": f"trajectory shards x{world}, no collective",
                   "l2": "flushed between timed steps (256 MiB write outside the event pairs); state is L2-resident within a step by design",
                   **main_res["resolved"]},
        "e2e": main_res.get("e2e"), "gpu_launches": main_res["launches"], "clocks": main_res.get("clocks"),
    }
    rl = roofline_block(main_res, w, T, peak, peak_src)
    if rl:
        line["roofline"] = rl
    pr = main_res["profile"]
    line["list_kernels"] = {
        "l1_rebuild_us": pr["l1_ms"] * 1e3 / pr["l1_spans"] if pr["l1_spans"] else None, "l1_rebuilds": pr["l1_spans"],
        "standalone_filter_us": pr["filter_ms"] * 1e3 / pr["filter_spans"] if pr["filter_spans"] else None,
        "standalone_filters": pr["filter_spans"],
        "note": "CUDA-event spans inside the library: a1+a2 (+ slot localisation in mode 3) per pair-list rebuild; a3 as its own "
                "kernel (modes 2/3 filter inside the step kernel, so only the end-of-run / set_coords filters show up here)"}
    line["whole_step_gbs"] = main_res["bytes"]["B_step"] * w.n_beads * T * world / (main_res["us_per_langevin_step"] * 1e-6) / 1e9
    line["whole_step_frac"] = line["whole_step_gbs"] / world / peak

    if rank == 0 and world == 1:
        if not args.no_sweep:
            sweep = {}
            for k in range(5):
                if k == args.config:
                    continue
                wk = gen.make_config(k)
                blk = 1000 if wk.n_beads * wk.n_traj < 100000 or k == 1 else 200     # (cfg 4 launches per step: 200 suffice)
                r = measure(wk, wk.n_traj, 0, blk, 3, 3, e2e=False, overrides=over)
                sweep[wk.name] = {"value": r["value"], "us_per_langevin_step": r["us_per_langevin_step"],
                                  "step_kernel_us": r.get("step_kernel", {}).get("us_per_langevin_step"),
                                  "step_kernel_gbs": r.get("step_kernel", {}).get("achieved_gbs"),
                                  "step_kernel_frac": r.get("step_kernel", {}).get("achieved_gbs", 0.0) / peak,
                                  "whole_path_gbs": r["bytes"]["B_step"] * wk.n_beads * wk.n_traj / (r["us_per_langevin_step"] * 1e-6) / 1e9,
                                  "whole_path_frac": r["bytes"]["B_step"] * wk.n_beads * wk.n_traj / (r["us_per_langevin_step"] * 1e-6) / 1e9 / peak,
                                  "l1_rebuild_us": r["profile"]["l1_ms"] * 1e3 / r["profile"]["l1_spans"] if r["profile"]["l1_spans"] else None,
                                  "standalone_filter_us": r["profile"]["filter_ms"] * 1e3 / r["profile"]["filter_spans"] if r["profile"]["filter_spans"] else None,
                                  "roofline": roofline_block(r, wk, wk.n_traj, peak, peak_src),
                                  "B_fi": r["bytes"]["B_fi"], **r["resolved"]}
            line["workloads"] = sweep
            # variants of the path on the same inputs: the paper's pair-based scheme (mode 4, NEXT-3) on cfg 0 and cfg 3, the
            # second resident kernel (resident_variant 2) on cfg 2 and cfg 3, the paper's Hybrid Taus generator (rng 1) on cfg 3
            var = {}
            for name, k, ov in (("cfg0_mode4_pair_based", 0, {"mode": 4}), ("cfg0_mode4_pair_based_atomics", 0, {"mode": 4, "pair_atomics": 1}),
                                ("cfg3_mode4_pair_based", 3, {"mode": 4}), ("cfg3_mode1_particle_based", 3, {"mode": 1}),
                                ("cfg3_resident_variant2", 3, {"resident_variant": 2}), ("cfg2_resident_variant2", 2, {"resident_variant": 2}),
                                ("cfg3_hybrid_taus", 3, {"rng": 1})):
                wk = gen.make_config(k)
                blk = 1000 if ov.get("mode", 3) == 3 or k == 0 else 200
                r = measure(wk, wk.n_traj, 0, blk, 2, 3, e2e=False, overrides=ov)
                var[name] = {"us_per_langevin_step": r["us_per_langevin_step"], "step_kernel_us": r.get("step_kernel", {}).get("us_per_langevin_step"),
                             "value": r["value"], **r["resolved"]}
            line["variants"] = var
            # the host side of the getters at the many-runs size (256,000 bead instances): pinned staging + index permutation
            import time as _t
            import paper_1003_1148_b200 as m
            w1 = gen.make_config(1)
            s1 = m.from_workload(w1)
            x1 = s1.get_coords()
            t0 = _t.perf_counter()
            for _ in range(5):
                s1.get_coords(out=x1)
            t1 = _t.perf_counter()
            for _ in range(5):
                s1.set_coords(x1)
            s1.sync()
            t2 = _t.perf_counter()
            line["host_io_cfg1"] = {"get_coords_ms": (t1 - t0) / 5 * 1e3, "set_coords_ms_incl_list_rebuild": (t2 - t1) / 5 * 1e3,
                                    "bead_instances": w1.n_beads * w1.n_traj}
            s1.close()
        if args.sweep4:
            # thread-per-bead (1 lane) ... warp-per-bead (32 lanes) x the paper's block sizes, mode 1
            w4 = gen.make_config(4)
            rows = []
            for lanes in (1, 2, 4, 8, 32):
                for blk in (64, 128, 256):
                    r = measure(w4, w4.n_traj, 0, 200, 2, 3, e2e=False, overrides={"mode": 1, "lanes_per_bead": lanes, "block_size": blk})
                    rows.append({"lanes_per_bead": lanes, "block_size": blk, "us_per_langevin_step": r["us_per_langevin_step"],
                                 "step_kernel_us": r.get("step_kernel", {}).get("us_per_langevin_step")})
            line["cfg4_variant_sweep"] = rows
        if not args.no_cpu:
            Tc = CPU_TRAJ.get(args.config, 1)
            n = CPU_STEPS[args.config]
            v, dt, cores = cpu_sample(w, Tc, n)
            line["cpu_baseline"] = {"value": v, "unit": METRIC, "cores": cores, "kind": "oracle", "seconds": dt,
                                    "sample": f"{Tc} trajectory(ies) x {n} Langevin steps of {w.name} (incl. list rebuilds + 1 energy evaluation), fp64, OpenMP"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
