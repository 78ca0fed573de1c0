#!/usr/bin/env python
"""bench.py -- throughput of the photon-packet transport hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload torus256] [--packets P] [--clumps C]

One "step" is one pass of the whole hot path (S0-S12: tally reset, per-epoch temperature-index
update, persistent transport kernel with its S / J / E phases, range check) over one batch of `--packets`
synthetic packets of the named workload (default: BASELINE config 4, torus256, 5000 clumps, 1e8 packets).  Prints ONE JSON line (rank 0).  `value` = cell crossings per second with the inputs resident
in HBM; `e2e` = the same metric through the C ABI with HOST buffers (grid/tables host->device and
E_abs/T/SED device->host inside the timed region).

--impl reference times the CPU oracle (oracle/) as it stands on the host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, os.path.join(ROOT, "oracle")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

METRIC = "cell crossings/s (photon-packet transport, packets/s alongside)"
UNIT = "crossings/s"
ALGO_BYTES_PER_CROSSING = 5.0      # rho fp32 + species u8 read per crossing
ALGO_BYTES_PER_DUSTY = 16.0        # 8 B read + 8 B write of the int64 Lucy atomic


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="torus256")
    ap.add_argument("--packets", type=int, default=0, help="packets per step (0 = the configuration's full count)")
    ap.add_argument("--clumps", type=int, default=5000)
    ap.add_argument("--ref-packets", type=int, default=30_000_000, help="oracle sample size per step (about 15 s on 16 cores)")
    ap.add_argument("--bmax", type=int, default=0, help="experiment: epoch_Bmax override (0 = library default)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def make_workload(args):
    from paper_1203_2941_b200 import workloads as W

    kw = {}
    if args.workload in ("torus256", "torus512"):
        kw["n_clumps"] = args.clumps if args.workload == "torus256" else 20000
    w = W.make(args.workload, **kw)
    n = args.packets if args.packets > 0 else w.n_packets
    return w, n


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.f.flush()
            self.f.seek(0)
            self.rows = [r.strip().split(", ") for r in self.f.read().strip().splitlines() if r.strip()]
            self.f.close()
            os.unlink(self.f.name)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.strip().lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(w, n_sample, seed, threads):
    """Time the oracle as it stands on a bounded sample of the workload (its own epoch schedule for n_sample)."""
    import oracle as orc

    o = orc.Oracle.from_workload(w)
    t0 = time.perf_counter()
    r = o.run(n_sample, seed, n_threads=threads)
    dt = time.perf_counter() - t0
    o.close()
    return r, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as orc

    w, n_full = make_workload(args)
    threads = orc.max_threads()
    n_s = min(args.ref_packets, n_full)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(w, max(1000, n_s // 100), w.seed, threads)
    tot_c = tot_p = 0
    tot_t = 0.0
    for s in range(args.steps):
        r, dt = oracle_sample(w, n_s, w.seed + s, threads)
        tot_c += r["crossings"]; tot_p += r["packets"]; tot_t += dt
    val = tot_c / tot_t
    sample = f"{n_s} packets/step of {w.name} (full step = {n_full}), oracle B&W epochs for that N, {threads} OpenMP threads"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "packets_per_s": tot_p / tot_t,
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "n_clumps": w.meta.get("n_clumps"),
                   "n_nu": w.n_nu, "n_species": w.n_species, "packets_per_step": n_s},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def reduce_over_ranks(elapsed, counts, device, world):
    """Whole-job figures of N independent replicas: the elapsed time is the MAX over
    ranks, the unit counts are SUMMED.  Uses the default process group (NCCL on GPUs, gloo in the CPU test)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([elapsed], dtype=torch.float64, device=device)
    c = torch.tensor([float(x) for x in counts], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in c.tolist()]


def replica_seed(base_seed, rank):
    """Seed of rank's replica: same problem, disjoint Philox keys."""
    return base_seed + 1000 * rank


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1203_2941_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.load_library()

    w, n_packets = make_workload(args)
    seed = replica_seed(w.seed, rank)  # N > 1: independent replicas of the same problem

    # ------------------------------------------------------------------ resident-input arm
    ctx = B.Context(w, device=str(dev), inputs_on_device=True)
    blocks, threads, smem = ctx.launch_config()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        ctx.run(n_packets, seed, want_stats=False, epoch_Bmax=args.bmax)
    barrier()
    stats0 = None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tot = {"crossings": 0, "dusty_crossings": 0, "packets": 0, "gpu_launches": 0, "transport_ms": 0.0, "update_ms": 0.0,
           "epochs": 0}
    with ClockSampler(local) as clocks:
        barrier()
        ev0.record()
        for i in range(args.steps):
            ctx.run(n_packets, seed + i, want_stats=False, time_kernels=1, epoch_Bmax=args.bmax)
            if i < args.steps - 1:
                # counters are reset by the next run: read them (tiny D2H, inside the timed region, honest)
                st = ctx.stats()
                for k in tot:
                    tot[k] += st[k]
        ev1.record()
        barrier()
    st = ctx.stats()
    for k in tot:
        tot[k] += st[k]
    ms = ev0.elapsed_time(ev1)
    ms_all, (crossings_all, packets_all, dusty_all) = reduce_over_ranks(
        ms, [tot["crossings"], tot["packets"], tot["dusty_crossings"]], dev, world)
    value = crossings_all / (ms_all * 1e-3)

    # roofline of the dominant kernel (k_transport), this rank: algorithmic bytes / its own launch time
    algo_bytes = ALGO_BYTES_PER_CROSSING * tot["crossings"] + ALGO_BYTES_PER_DUSTY * tot["dusty_crossings"]
    n_launch = max(1, tot["epochs"])
    peak, peak_src = measured_peak()
    achieved = algo_bytes / (tot["transport_ms"] * 1e-3) / 1e9 if tot["transport_ms"] > 0 else 0.0
    roofline = {
        "bound": "hbm", "kernel": "k_transport", "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": algo_bytes / n_launch, "launches": n_launch,
        "avg_launch_ms": tot["transport_ms"] / n_launch,
        "kernel_share_of_step": tot["transport_ms"] / (ms if ms > 0 else 1.0),
        "bytes_per_crossing": algo_bytes / max(1, tot["crossings"]),
        "traffic": None,
    }
    # DRAM traffic of one k_transport launch from the committed ncu capture (profiles/traffic.csv), scaled from the
    # captured launch (2^22 packets) to this run's average launch by packets
    prof = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(prof):
        try:
            import csv
            for row in csv.DictReader(open(prof)):
                if row["workload"] == w.name:
                    per_packet = float(row["dram_bytes_per_launch"]) / float(row["launch_packets"])
                    roofline["traffic"] = per_packet * tot["packets"] / n_launch
                    roofline["traffic_source"] = "profiles/" + row["source"]
        except Exception:
            pass
    ctx.close()

    # ------------------------------------------------------------------ end-to-end arm (host buffers through the C ABI)
    e2e = None
    if not args.no_e2e:
        rho_h = torch.from_numpy(np.ascontiguousarray(w.rho)).pin_memory()
        sp_h = torch.from_numpy(np.ascontiguousarray(w.species)).pin_memory()
        nc = w.n_cells
        E_h = torch.empty(nc, dtype=torch.float64).pin_memory()
        T_h = torch.empty(nc, dtype=torch.float32).pin_memory()
        sed_h = torch.empty(w.n_dir * w.n_nu, dtype=torch.float64).pin_memory()
        nbytes = B.mcrt_workspace_bytes(w.nx, w.ny, w.nz, w.n_species, w.n_nu, len(w.T_grid), w.n_dir, 0)
        ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        stream = torch.cuda.current_stream(dev).cuda_stream

        def e2e_step(sd):
            c = B.mcrt_grid_create(w.nx, w.ny, w.nz, w.cell_size_cm, rho_h, sp_h, w.n_species, B.MCRT_HOST, ws, nbytes)
            B.mcrt_set_stream(c, stream)
            B.mcrt_dust_tables(c, w.nu_hz, w.kappa_abs, w.kappa_sca, w.g, w.T_grid)
            B.mcrt_source(c, w.L_erg_s, w.T_star_K, w.L_nu_weights, w.source_pos_cm)
            B.mcrt_escape_bins(c, w.abs_mu_edges)
            s = B.mcrt_run(c, n_packets, sd)
            B.mcrt_read(c, E_abs_lucy=E_h, T_lucy=T_h, SED=sed_h, where=B.MCRT_HOST)
            B.mcrt_destroy(c)
            return s

        e2e_step(seed)  # warm-up
        barrier()
        t0 = time.perf_counter()
        c_e2e = 0
        e2e_steps = max(1, min(args.steps, 2))
        for i in range(e2e_steps):
            c_e2e += e2e_step(seed + i)["crossings"]
        barrier()
        dt = time.perf_counter() - t0
        dt_all, (c_all,) = reduce_over_ranks(dt, [float(c_e2e)], dev, world)
        nsf = w.n_species * w.n_nu
        h2d = nc * 5 + 8 * (4 * nsf + 2 * w.n_nu + w.n_species * len(w.T_grid) + len(w.T_grid)
                            + 2 * nsf * len(w.T_grid) + w.n_dir + 1)
        d2h = nc * 12 + 8 * w.n_dir * w.n_nu
        e2e = {"value": c_all / dt_all, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": e2e_steps, "ms_per_step": 1e3 * dt_all / e2e_steps,
               "includes": "grid_create+dust_tables+source+run+read(E_lucy,T_lucy,SED)+destroy with pinned host buffers"}

    # ------------------------------------------------------------------ CPU baseline (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle as orc  # bench.py's cpu_baseline leg is allowed to execute oracle/

        nth = orc.max_threads()
        n_s = min(args.ref_packets, n_packets)
        r, dt = oracle_sample(w, n_s, w.seed, nth)
        cpu = {"value": r["crossings"] / dt, "unit": UNIT, "cores": nth, "kind": "oracle",
               "packets_per_s": r["packets"] / dt,
               "sample": f"{n_s} packets of {w.name} (oracle as is, its own epoch schedule for that N, {dt:.1f} s)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "packets_per_s": packets_all / (ms_all * 1e-3),
            "crossings_per_packet": crossings_all / max(1.0, packets_all),
            "dusty_fraction": dusty_all / max(1.0, crossings_all),
            "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "n_clumps": w.meta.get("n_clumps"),
                       "n_nu": w.n_nu, "n_species": w.n_species, "packets_per_step": n_packets,
                       "mode": "bw_epoch", "launch": {"blocks": blocks, "threads": threads, "smem": smem},
                       "l2": "inputs larger than L2: cell words + tallies %.0f MB (dusty part %.0f MB) vs 126 MB; tallies reset and "
                             "the per-epoch update streams all cells between transport launches"
                             % (w.n_cells * 32 / 1e6, float((w.rho > 0).sum()) * 32 / 1e6),
                       "epoch_Bmax": args.bmax if args.bmax else "default 2^22",
                       "parallelism": "replicas" if world > 1 else "single"},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": int(tot["gpu_launches"]),
            "clocks": clocks.summary(),
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
