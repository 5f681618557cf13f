#!/usr/bin/env python
"""Benchmark of the hot path: one step = one dgfs_collide over the whole spatial batch of config
c2 (BASELINE.json configs[2]: N=32, N_rho=32, M=12, 2 species, 4096 points) per GPU.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c2] [--nx n]

Prints ONE JSON line (rank 0).  metric = pair-evals/s = spatial points x species pairs per second,
whole job.  See DESIGN.md "Measurement" for the roofline arithmetic.
"""
import argparse
import dataclasses
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "collision evals/s (spatial pts x species pairs) at N=32"
UNIT = "pair-evals/s"
# FP64 DFMA pipe: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz.  The same
# pipe is also measured live with dgfs_measure_fp64_peak (dependency-free DFMA chains) and reported.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
PAPER_P100_PAIR_EVALS_PER_S = 1.0 / 0.01057      # Table 1 P:316 (N=32, N_rho=32, M=12), 1 x P100
# dram__bytes_read.sum + dram__bytes_write.sum of one k_xy launch over 512 points (all pairs, one radial node) at
# the c2 operating point, from the `ncu --set full` capture summarised in profiles/r01_v1_ncu.md
NCU_DRAM_BYTES_PER_POINT = {"k_xy": (2.842e9 + 0.4463e9) / 512}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--nx", type=int, default=0, help="override the batch size (debugging only; reported)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nyquist-filter", action="store_true",
                    help="time the variant operator Q(P f_p, P f_q) (dgfs_params.nyquist_filter); not the headline metric")
    return ap.parse_args()


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons = index, False, [], set()
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def oracle_sample(cfg, n_points):
    """Time the oracle, as it stands, on n_points points of the workload (all pairs), taken alternately from
    the start and from the middle of the batch (both halves of the c2 mix).  Returns (pair_evals, seconds, cores)."""
    from workloads import make_points
    from oracle.tables import precompute
    from oracle.collide import collide_pairs
    xs = [(i // 2) + (cfg.nx // 2 if i % 2 else 0) for i in range(n_points)]
    f = make_points(cfg, xs)
    tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha)   # create: untimed
    t0 = time.perf_counter()
    collide_pairs(tab, f)
    dt = time.perf_counter() - t0
    return n_points * cfg.ns * cfg.ns, dt, 1


def run_reference(args, cfg, rank):
    """--impl reference: the CPU oracle on the host cores (kind = oracle)."""
    if rank != 0:
        return
    sample_pts = 2
    times = []
    evals = 0
    for i in range(args.warmup + args.steps):
        evals, dt, cores = oracle_sample(cfg, sample_pts)
        if i >= args.warmup:
            times.append(dt)
        if sum(times) > 240:
            break
    t = sum(times) / len(times)
    val = evals / t
    sample = "%d point(s) x %d pairs of %s per step (oracle collide_pairs, numpy single thread)" % (
        sample_pts, cfg.ns * cfg.ns, cfg.name)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(times), "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_desc(cfg, cfg.nx, args.gpus),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_desc(cfg, nx, ngpus):
    return {"workload": "%s: homogeneous %d-species Ar/Kr VHS collide, N=%d, N_rho=%d, M=%d, L=%g, "
                        "nx=%d points per GPU (half near-equilibrium, half bi-Maxwellian)" % (
                            cfg.name, cfg.ns, cfg.N, cfg.N_rho, cfg.M, cfg.L, nx),
            "N": cfg.N, "N_rho": cfg.N_rho, "M": cfg.M, "ns": cfg.ns, "nx_per_gpu": nx,
            "pair_evals_per_step": nx * cfg.ns * cfg.ns * ngpus,
            "parallelism": "replicated tables, nx sharded over %d GPU(s), no collective" % ngpus,
            "l2": "inputs (%.2f GB per GPU) exceed the 126 MB L2; no flush needed" % (
                nx * cfg.ns * cfg.N ** 3 * 8 / 1e9)}


def main():
    args = parse()
    from workloads import get_config, make_points
    cfg = get_config(args.workload)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import __graft_entry__ as entry
    if local == 0:
        entry.build()
    if world > 1:
        dist.barrier()
    from paper_1903_04670_b200 import Dgfs
    from paper_1903_04670_b200.parallel import rank_seed, max_over_ranks, whole_job_rate

    nx = args.nx if args.nx > 0 else cfg.nx
    # weak scaling: every rank owns its own nx points (rank r draws them with seed + 1000 r)
    rcfg = dataclasses.replace(cfg, seed=rank_seed(cfg.seed, rank))
    if nx == cfg.nx:
        f_np = make_points(rcfg, range(nx))
    else:      # reduced batch keeps both halves of the c2 mix
        half = nx // 2
        xs = list(range(half)) + list(range(cfg.nx - (nx - half), cfg.nx))
        f_np = make_points(rcfg, xs)
    f_host = torch.from_numpy(f_np).pin_memory()
    q_host = torch.empty_like(f_host).pin_memory()
    op = Dgfs.from_config(cfg, device=local, nyquist_filter=args.nyquist_filter)
    op.reserve(nx)
    f_dev = f_host.cuda()
    q_dev = torch.empty_like(f_dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing ----------------
    for _ in range(args.warmup):
        op.collide(f_dev, q_dev)
    barrier()
    op.profile(on=True, reset=True)
    launches0 = op.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for i in range(args.steps):
        op.collide(f_dev, q_dev)
        ev[i + 1].record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = ev[0].elapsed_time(ev[-1])
    prof = op.profile(on=False)
    launches = op.launch_count() - launches0
    total_ms = max_over_ranks(total_ms)
    ms_per_step = total_ms / args.steps
    evals_per_step = nx * cfg.ns * cfg.ns * world
    value = whole_job_rate(nx * cfg.ns * cfg.ns, world, ms_per_step)

    # ---------------- end to end: pinned host -> device -> collide -> pinned host ----------------
    # dgfs_collide_host: HOST pointers in and out; the library's own streams carry the copies and the
    # kernels, and the call returns when Q is in host memory, so the region is timed on the host
    # clock between two device synchronisations (CUDA events on torch's stream would not see it).
    del f_dev, q_dev
    torch.cuda.empty_cache()

    def e2e_step():
        op.collide_host(f_host, q_host)

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3) / args.steps
    nbytes = f_host.numel() * 8

    if rank == 0:
        # ---------------- roofline of the dominant kernel class ----------------
        prof = [p for p in prof if p["launches"] > 0]
        top = max(prof, key=lambda p: p["ms"])
        ksum = sum(p["ms"] for p in prof)
        achieved = top["flops"] / (top["ms"] * 1e-3) / 1e12
        flops_step = sum(op.flops_per_pair_eval(p, q) for p in range(cfg.ns) for q in range(cfg.ns)) * nx
        from paper_1903_04670_b200 import dgfs_measure_fp64_peak
        FP64_PEAK_MEASURED_TFLOPS = dgfs_measure_fp64_peak(local, 2.0)[1]
        roofline = {
            "bound": "alu", "kernel": top["name"], "achieved": achieved, "peak": FP64_PEAK_NOMINAL_TFLOPS,
            "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_NOMINAL_TFLOPS,
            "peak_source": "FP64 DFMA pipe, 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md); "
                           "MEASURED_PEAKS.json has no fp64 entry",
            "frac_of_measured_dfma_peak": achieved / FP64_PEAK_MEASURED_TFLOPS,
            "measured_dfma_peak": FP64_PEAK_MEASURED_TFLOPS,
            "measured_dfma_peak_how": "dgfs_measure_fp64_peak: dependency-free DFMA chains, 2 s sustained, same box",
            "kernel_share_of_step": top["ms"] / ksum,
            "launch_ms": top["ms"] / top["launches"], "launches": top["launches"],
            "flops_per_launch": top["flops"] / top["launches"],
            "whole_step_tflops": flops_step / (ms_per_step * 1e-3) / 1e12 / 1.0,
            "whole_step_frac": flops_step / (ms_per_step * 1e-3) / 1e12 / FP64_PEAK_NOMINAL_TFLOPS,
            "traffic": (NCU_DRAM_BYTES_PER_POINT[top["name"]] * (nx * cfg.N_rho / top["launches"] * args.steps)
                        if top["name"] in NCU_DRAM_BYTES_PER_POINT and (cfg.N, cfg.N_rho, cfg.M) == (32, 32, 12) else None),
            "traffic_note": "DRAM bytes per launch of the dominant kernel, scaled from the ncu capture in "
                            "profiles/r01_v1_ncu.md (6.42 MB per point and radial node); algorithmic bytes per point: "
                            "4.72 MB z-shifted half planes + 0.79 MB S + 0.83 MB T for the three pairs that run",
            "kernels": [{"name": p["name"], "launches": p["launches"], "ms": round(p["ms"], 3),
                         "tflops": (p["flops"] / (p["ms"] * 1e-3) / 1e12 if p["ms"] > 0 else None)} for p in prof],
        }
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            npts = 4
            ev_n, dt, cores = oracle_sample(cfg, npts)
            cpu = {"value": ev_n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": "%d points of %s (two from each half of the batch), all %d pairs, %.1f s (oracle "
                             "collide_pairs, numpy, one thread, tables untimed)" % (npts, cfg.name, cfg.ns * cfg.ns, dt)}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": value / world / PAPER_P100_PAIR_EVALS_PER_S if cfg.name == "c2" else None,
            "vs_baseline_note": "per-GPU value / 94.6 pair-evals/s: paper Table 1 (P:316), 1 x Tesla P100, same "
                                "(N, N_rho, M) operating point, BKW workload; context, not the target",
            "dtype": "f64", "data": "synthetic",
            "config": dict(workload_desc(cfg, nx, world), **({"variant": "nyquist_filter"} if args.nyquist_filter else {})),
            "clocks": sampler.summary(),
            "e2e": {"value": evals_per_step / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                    "call": "dgfs_collide_host (C ABI, pinned host buffers in and out, host clock)"},
            "gpu_launches": launches,
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
        print(json.dumps(out))
    op.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
