"""Times dgfs_collide / dgfs_step on the BASELINE.json configurations other than the headline one
(bench.py measures c2).  Device-resident inputs, CUDA events on the current stream, warm.

    python -m paper_1903_04670_b200.measure_configs [c0 c1 c3 c4] [--nx-c4 64]

Prints one JSON line per configuration: pair-evals/s and the fraction of the nominal FP64 peak by the
executed-algorithm flop count (dgfs_flops_per_pair_eval)."""
import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FP64_PEAK_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def _time(torch, fn, reps):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("configs", nargs="*", default=["c0", "c1", "c3", "c4"])
    ap.add_argument("--nx-c4", type=int, default=64, help="points of c4's 2048 to run (the full batch is 0.4 PFLOP)")
    args = ap.parse_args()
    import torch
    from workloads import get_config, make_points, make_dg_state
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api
    torch.cuda.set_device(0)
    for name in args.configs:
        cfg = get_config(name)
        with Dgfs.from_config(cfg, device=0) as op:
            flops = sum(op.flops_per_pair_eval(p, q) for p in range(cfg.ns) for q in range(cfg.ns))
            if cfg.kind == "dg":
                f = torch.from_numpy(make_dg_state(cfg)).cuda()
                mesh = Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T)
                nx = cfg.ne * (cfg.order + 1)
                ms = _time(torch, lambda: api.dgfs_step(op.ctx, mesh, f, cfg.dt, 1), 2)
                evals, what = 3 * nx * cfg.ns ** 2, "one SSP-RK3 step of dgfs_step (3 collide calls of %d DOF)" % nx
                flops_step = 3 * nx * flops
            else:
                nx = cfg.nx if name != "c4" else min(cfg.nx, args.nx_c4)
                f = torch.from_numpy(make_points(cfg, range(nx))).cuda()
                Q = torch.empty_like(f)
                ms = _time(torch, lambda: op.collide(f, Q), 3 if name != "c4" else 1)
                evals, what = nx * cfg.ns ** 2, "dgfs_collide over %d of %d points" % (nx, cfg.nx)
                flops_step = nx * flops
            print(json.dumps({"config": name, "N": cfg.N, "N_rho": cfg.N_rho, "M": cfg.M, "ns": cfg.ns,
                              "what": what, "ms": ms, "pair_evals_per_s": evals / (ms * 1e-3),
                              "tflops_executed": flops_step / (ms * 1e-3) / 1e12,
                              "frac_of_nominal_fp64": flops_step / (ms * 1e-3) / 1e12 / FP64_PEAK_NOMINAL_TFLOPS}))


if __name__ == "__main__":
    main()
