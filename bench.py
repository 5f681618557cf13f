#!/usr/bin/env python
"""Benchmark of the hot path.  Default workload: config c2 of BASELINE.json (N=32, N_rho=32, M=12, 2 species, 4096
points per GPU); one step = one dgfs_collide over the whole spatial batch.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c0|c1|c2|c3|c4|couette] [--nx n]

c3 / couette: one step = one dgfs_step (SSP-RK3, three collide calls) / dgfs_step_euler step of the DG slab.
Prints ONE JSON line (rank 0).  metric = pair-evals/s = spatial points x species pairs per second, whole job.
See DESIGN.md section 8 for the roofline arithmetic.
"""
import argparse
import dataclasses
import json
import multiprocessing as mp
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "collision evals/s (spatial pts x species pairs) at N=32"
UNIT = "pair-evals/s"
# FP64 DFMA pipe: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz.  The same pipe is also
# measured live with dgfs_measure_fp64_peak (dependency-free DFMA chains) and reported beside it.
FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
PAPER_P100_PAIR_EVALS_PER_S = 1.0 / 0.01057      # Table 1 P:316 (N=32, N_rho=32, M=12), 1 x P100
HBM_FALLBACK_GBS = 6650.0                        # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c0", "c1", "c2", "c3", "c4", "couette", "c4vss", "c2half"])
    ap.add_argument("--nx", type=int, default=0, help="override the batch size (debugging only; reported)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="f32: dgfs_params.precision = 1 (SURVEY 8(f) item 1; not the headline metric)")
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


# ------------------------------------------------------------------------------ the CPU oracle, timed
_ORACLE = {}


def _oracle_eval(task):
    from oracle.collide import collide_pair
    x, p, q = task
    return float(collide_pair(_ORACLE["tab"], p, q, _ORACLE["f"][x, p], _ORACLE["f"][x, q])[0])


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def sample_state(cfg, n_points):
    """n_points spatial points of the workload for the oracle: alternately from the start and from the middle of a
    homogeneous batch (both halves of the c2 mix); the first DOF of a DG state."""
    from workloads import make_points, make_dg_state
    if cfg.kind in ("dg", "couette"):
        f = make_dg_state(cfg).reshape(-1, cfg.ns, cfg.N ** 3)
        return f[:: max(1, f.shape[0] // n_points)][:n_points].copy()
    xs = [(i // 2) + (cfg.nx // 2 if i % 2 else 0) for i in range(n_points)]
    return make_points(cfg, xs)


def oracle_sample(cfg, n_points, tab=None):
    """Time the oracle, as it stands, on n_points points of the workload, all pairs: one oracle.collide.collide_pair
    per (point, pair), spread over all host cores by a forked process pool (tables built before, untimed).
    Returns (pair_evals, seconds, workers, tables)."""
    from oracle.tables import precompute
    f = sample_state(cfg, n_points)
    if tab is None:
        vss = any(a != 1.0 for row in cfg.alpha for a in row)
        kn = {"kn": cfg.kn} if cfg.kn else {}
        tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha,
                         workers=(os.cpu_count() or 1) if vss else 1, **kn)   # create: untimed
    tasks = [(x, p, q) for x in range(f.shape[0]) for p in range(cfg.ns) for q in range(cfg.ns)]
    workers = max(1, min(os.cpu_count() or 1, len(tasks)))
    _ORACLE["tab"], _ORACLE["f"] = tab, f
    t0 = time.perf_counter()
    if workers == 1:
        for t in tasks:
            _oracle_eval(t)
    else:
        with mp.get_context("fork").Pool(workers) as pool:
            pool.map(_oracle_eval, tasks, chunksize=1)
    dt = time.perf_counter() - t0
    _ORACLE.clear()
    return len(tasks), dt, workers, tab


def oracle_points(cfg):
    """Sample size giving roughly 10-30 s of CPU work per timing at 16 cores."""
    return {"c0": 4, "c1": 32, "c2": 16, "c3": 16, "c4": 4, "couette": 16, "c4vss": 4, "c2half": 16}[cfg.name]


def workload_desc(cfg, nx, ngpus, stages):
    kinds = {"bimaxwell": "bi-Maxwellian inputs", "c2mix": "half near-equilibrium, half bi-Maxwellian",
             "dg": "1-D DG slab, %d elements of order %d, diffuse walls, one SSP-RK3 step of dgfs_step" % (cfg.ne, cfg.order),
             "couette": "Couette case C-01 (Table 2), %d elements of order %d, one Euler step of dgfs_step_euler" % (cfg.ne, cfg.order)}
    vss = sum(a != 1.0 for row in cfg.alpha for a in row)
    phys = "%d species, masses %s, %d of %d pairs VSS" % (cfg.ns, "/".join("%.4g" % m for m in cfg.mass), vss, cfg.ns ** 2)
    return {"workload": "%s: %s; N=%d, N_rho=%d, M=%d, L=%g, nx=%d spatial points per GPU (%s)" % (
                cfg.name, phys, cfg.N, cfg.N_rho, cfg.M, cfg.L, nx, kinds[cfg.kind]),
            "N": cfg.N, "N_rho": cfg.N_rho, "M": cfg.M, "ns": cfg.ns, "nx_per_gpu": nx,
            "collide_calls_per_step": stages, "pair_evals_per_step": stages * nx * cfg.ns * cfg.ns * ngpus,
            "parallelism": "replicated tables, nx sharded over %d GPU(s), no collective" % ngpus,
            "l2": ("inputs (%.2f GB per GPU) exceed the 126 MB L2; no flush needed" % (nx * cfg.ns * cfg.N ** 3 * 8 / 1e9)
                   if nx * cfg.ns * cfg.N ** 3 * 8 > 126e6 else
                   "state (%.1f MB) fits the L2; 256 MB written between timed steps to flush it" % (nx * cfg.ns * cfg.N ** 3 * 8 / 1e6))}


def stages_of(cfg):
    return 3 if cfg.kind == "dg" else 1


def run_reference(args, cfg, rank):
    """--impl reference: the CPU oracle on the host cores (kind = oracle); each step a bounded sample."""
    if rank != 0:
        return
    npts = oracle_points(cfg)
    times, evals, workers, tab = [], 0, 1, None
    for i in range(args.warmup + args.steps):
        evals, dt, workers, tab = oracle_sample(cfg, npts, tab)
        if i >= args.warmup:
            times.append(dt)
        if sum(times) > 240:
            break
    t = sum(times) / len(times)
    val = evals / t
    sample = "%d point(s) x %d pairs of %s per step (oracle.collide.collide_pair per (point, pair), %d worker processes on %s)" % (
        npts, cfg.ns * cfg.ns, cfg.name, workers, cpu_model())
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(times), "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_desc(cfg, cfg.nx, args.gpus, stages_of(cfg)),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": workers, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def measured_hbm_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json (measured copy bandwidth)"
    except Exception:
        return HBM_FALLBACK_GBS, "B200_PROFILING.md fallback"


def step_traffic(cfg, prof, steps):
    """DRAM bytes of one step from this round's ncu capture (profiles/r02_traffic.json: dram__bytes_read.sum +
    dram__bytes_write.sum per launch of each kernel class at the c2 operating point, 512-point chunk), scaled by
    the launches the live run made.  None for other operating points."""
    try:
        with open(TRAFFIC_JSON) as fh:
            tj = json.load(fh)
    except Exception:
        return None, None
    if (cfg.N, cfg.N_rho, cfg.M, cfg.ns) != tuple(tj["operating_point"]):
        return None, tj
    per = tj["dram_bytes_per_launch"]
    total = 0.0
    for p in prof:
        if p["name"] in per:
            total += per[p["name"]] * p["launches"] / steps
    return total, tj


def main():
    args = parse()
    from workloads import get_config, make_points, make_dg_state
    cfg = get_config(args.workload)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

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
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    from paper_1903_04670_b200.parallel import rank_seed, max_over_ranks, whole_job_rate

    is_dg = cfg.kind in ("dg", "couette")
    stages = stages_of(cfg)
    # weak scaling: every rank owns its own nx points (rank r draws them with seed + 1000 r)
    rcfg = dataclasses.replace(cfg, seed=rank_seed(cfg.seed, rank))
    if is_dg:
        f_np = make_dg_state(rcfg)
        nx = cfg.ne * (cfg.order + 1)
        mesh = Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T, wall_u=cfg.wall_u)
    else:
        nx = args.nx if args.nx > 0 else cfg.nx
        if nx == cfg.nx:
            f_np = make_points(rcfg, range(nx))
        else:      # reduced batch keeps both halves of the c2 mix
            half = nx // 2
            f_np = make_points(rcfg, list(range(half)) + list(range(cfg.nx - (nx - half), cfg.nx)))
    f_host = torch.from_numpy(f_np).pin_memory()
    q_host = torch.empty_like(f_host).pin_memory()
    kw = {"nyquist_filter": True} if args.nyquist_filter else {}
    if args.precision == "f32":
        kw["precision"] = 1
    op = Dgfs.from_config(cfg, device=local, **kw)
    op.reserve(nx)
    f_dev = f_host.cuda()
    q_dev = torch.empty_like(f_dev)
    stream = torch.cuda.current_stream()
    small = f_dev.numel() * 8 <= 126e6
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        if is_dg:
            (api.dgfs_step if cfg.scheme == "rk3" else api.dgfs_step_euler)(op.ctx, mesh, f_dev, cfg.dt, 1)
        else:
            op.collide(f_dev, q_dev)

    # ---------------- device-resident timing (per-launch profiling OFF: nothing but the step is in the region) ------
    for _ in range(args.warmup):
        step_device()
    barrier()
    launches0 = op.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for i in range(args.steps):
        if flush is not None:
            flush.fill_(i)                 # L2 flush between timed steps, outside the timed intervals
        ev[i][0].record(stream)
        step_device()
        ev[i][1].record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    launches = op.launch_count() - launches0
    total_ms = max_over_ranks(total_ms)
    ms_per_step = total_ms / args.steps
    evals_rank = stages * nx * cfg.ns * cfg.ns
    value = whole_job_rate(evals_rank, world, ms_per_step)
    # ---------------- the same steps once more with the library's per-launch CUDA events on (per-kernel times) -------
    op.profile(on=True, reset=True)
    for i in range(args.steps):
        if flush is not None:
            flush.fill_(i)
        step_device()
    barrier()
    prof = op.profile(on=False)

    # ---------------- end to end: pinned host -> device -> step -> pinned host ----------------
    # homogeneous workloads: dgfs_collide_host (HOST pointers in and out; the library's own streams carry the copies
    # and the kernels; returns when Q is in host memory).  DG workloads: state up, one step, state down.  Timed on the
    # host clock between two device synchronisations.
    if not is_dg:
        del f_dev, q_dev
        torch.cuda.empty_cache()

    def e2e_step():
        if is_dg:
            f_dev.copy_(f_host, non_blocking=True)
            step_device()
            q_host.copy_(f_dev, non_blocking=True)
            torch.cuda.synchronize()
        else:
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
        report(args, cfg, op, prof, nx, world, stages, ms_per_step, value, e2e_ms, nbytes, launches, sampler, local, is_dg)
    op.close()
    if world > 1:
        dist.destroy_process_group()


def report(args, cfg, op, prof, nx, world, stages, ms_per_step, value, e2e_ms, nbytes, launches, sampler, local, is_dg):
    from paper_1903_04670_b200 import dgfs_measure_fp64_peak
    prof = [p for p in prof if p["launches"] > 0]
    top = max(prof, key=lambda p: p["ms"])
    ksum = sum(p["ms"] for p in prof)
    kernel_tflops = top["flops"] / (top["ms"] * 1e-3) / 1e12
    flops_step = stages * nx * sum(op.flops_per_pair_eval(p, q) for p in range(cfg.ns) for q in range(cfg.ns))
    step_tflops = flops_step / (ms_per_step * 1e-3) / 1e12
    peak_meas = dgfs_measure_fp64_peak(local, 2.0)[1]
    hbm_gbs, hbm_src = measured_hbm_gbs()
    dram_step, tj = step_traffic(cfg, prof, args.steps)
    flops_floor_ms = flops_step / (FP64_PEAK_NOMINAL_TFLOPS * 1e12) * 1e3
    evals = stages * nx * cfg.ns * cfg.ns
    alg_bytes = 24.0 * cfg.N ** 3 * evals                     # read f_p, f_q, write Q per pair evaluation
    alg_bytes_floor_ms = alg_bytes / (hbm_gbs * 1e9) * 1e3
    dram_floor_ms = dram_step / (hbm_gbs * 1e9) * 1e3 if dram_step else None
    # north_star: the roofline is the slower of flops at the FP64 peak and (algorithmic) bytes at the HBM bandwidth.
    # At 3-4 kflop per algorithmic byte the flops floor is the roofline; the DRAM traffic this pipeline really makes
    # (its intermediates) is reported beside it with its own floor, which at c2 is of the same size as the flops floor.
    bound = "alu" if flops_floor_ms >= alg_bytes_floor_ms else "hbm"
    top_traffic = tj["dram_bytes_per_launch"].get(top["name"]) if (tj and dram_step) else None
    clk = sampler.summary()
    roofline = {
        "bound": bound,
        # the WHOLE step: executed-algorithm flops of every kernel of the call / step time / nominal FP64 peak
        "frac": step_tflops / FP64_PEAK_NOMINAL_TFLOPS,
        "achieved": step_tflops, "peak": FP64_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
        "peak_source": "FP64 DFMA pipe, 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md section 8); "
                       "MEASURED_PEAKS.json has no fp64 entry",
        "scope": "whole step (every kernel of the call), flop count of the algorithm as executed"
                 + ("; precision f32: the plane jobs run on the FP32 pipe (twice the lanes), so this fraction of the FP64 peak is "
                    "for comparison with the fp64 line only, not a roofline fraction" if args.precision == "f32" else ""),
        "flops_floor_ms": flops_floor_ms, "algorithmic_bytes_floor_ms": alg_bytes_floor_ms, "step_ms": ms_per_step,
        "step_flops": flops_step, "algorithmic_bytes": alg_bytes,
        "step_dram_bytes": dram_step, "step_dram_floor_ms": dram_floor_ms,
        "step_dram_gbs": dram_step / (ms_per_step * 1e-3) / 1e9 if dram_step else None,
        "hbm_gbs": hbm_gbs, "hbm_source": hbm_src,
        "frac_of_measured_dfma_peak": step_tflops / peak_meas,
        # the same fraction against the pipe's rate at the SM clock the timed steps actually ran at (median NVML sample;
        # under the power cap the step runs below sm_max_mhz): secondary, "frac" stays against the nominal clock
        "frac_at_sm_clock": (step_tflops / (FP64_PEAK_NOMINAL_TFLOPS * clk["sm_mhz"] / clk["sm_max_mhz"])
                             if clk.get("sm_mhz") and clk.get("sm_max_mhz") else None),
        "measured_dfma_peak": peak_meas,
        "measured_dfma_peak_how": "dgfs_measure_fp64_peak: dependency-free DFMA chains, 2 s sustained, same box",
        # the dominant kernel class, from the library's per-launch CUDA events on the launching stream
        "kernel": top["name"], "kernel_frac": kernel_tflops / FP64_PEAK_NOMINAL_TFLOPS,
        "kernel_tflops": kernel_tflops, "kernel_share_of_step": top["ms"] / ksum,
        "launch_ms": top["ms"] / top["launches"], "launches": top["launches"],
        "flops_per_launch": top["flops"] / top["launches"],
        "traffic": top_traffic,
        "traffic_note": ("dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel and per step, from "
                         "profiles/r02_traffic.json (%s)" % tj.get("source", "") if tj else
                         "no ncu capture for this operating point"),
        "kernels": [{"name": p["name"], "launches": p["launches"], "ms": round(p["ms"], 3),
                     "tflops": (p["flops"] / (p["ms"] * 1e-3) / 1e12 if p["ms"] > 0 else None)} for p in prof],
    }
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        npts = oracle_points(cfg)
        ev_n, dt, workers, _ = oracle_sample(cfg, npts)
        cpu = {"value": ev_n / dt, "unit": UNIT, "cores": workers, "kind": "oracle", "cpu": cpu_model(),
               "host_cores": os.cpu_count(),
               "sample": "%d points of %s (both halves of the batch), all %d pairs, %.1f s: oracle.collide.collide_pair per "
                         "(point, pair) in %d forked worker processes, tables untimed" % (npts, cfg.name, cfg.ns * cfg.ns, dt, workers)}
    evals_step = stages * nx * cfg.ns * cfg.ns * world
    variant = {}
    if args.nyquist_filter:
        variant["variant"] = "nyquist_filter"
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": value / world / PAPER_P100_PAIR_EVALS_PER_S if cfg.name == "c2" and args.precision == "f64" else None,
        "vs_baseline_note": "per-GPU value / 94.6 pair-evals/s: paper Table 1 (P:316), 1 x Tesla P100, same "
                            "(N, N_rho, M) operating point, BKW workload; context, not the target",
        "dtype": args.precision, "data": "synthetic",
        "config": dict(workload_desc(cfg, nx, world, stages), **variant),
        "clocks": clk,
        "e2e": {"value": evals_step / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "call": ("state host -> device, one step, device -> host (pinned buffers, host clock)" if is_dg else
                         "dgfs_collide_host (C ABI, pinned host buffers in and out, host clock)")},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))


if __name__ == "__main__":
    main()
