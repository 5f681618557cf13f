"""Second workload: the paper's Couette case C-01 (Table 2) run to
its steady state through `dgfs_step_euler`, on one GPU.

    python -m workloads.couette_case [--dt 1e-3] [--block 250] [--tol 2e-4] [--max-steps 40000]

It lives beside the workload definitions, not in the product package: every step of the path (wall balance,
collisions of all four VSS pairs, transport, Euler update) runs in the library's kernels through `dgfs_step_euler`;
this script only drives it, and every `--block` steps reads bulk moments of the state (plain torch reductions:
diagnostics of a workload, not part of the method or of the timed path) to decide when the flow has stopped changing.
Prints ONE JSON line: steps and device time to the steady state, time per step, the moment profiles and the
self-consistency checks the paper's text allows (the DSMC curves of its Fig. 2 are images that are not in the
container): per-species mass balance (drift = mass defect of the collision term), antisymmetry of u_y about the centre plane, velocity slip at the
walls (|u_y| below the wall speed), no flow across the gap.  Context figure: the paper's run took 138 s on one
P100; its time step and stopping rule are not printed, so the two times are not comparable step by step.
"""
import argparse
import json
import time

import numpy as np


def gll(order):
    """Gauss-Lobatto-Legendre nodes and weights on [-1, 1] (diagnostics only: integrals over x)."""
    n = order
    Pn = np.polynomial.legendre.Legendre.basis(n)
    xi = np.concatenate(([-1.0], np.sort(Pn.deriv().roots().real), [1.0]))
    w = 2.0 / (n * (n + 1) * Pn(xi) ** 2)
    return xi, w


def moments(f, N, L, mass):
    """f: torch [ne][K][ns][N^3] -> n, u[3], T as torch [ne][K][ns] (Maxwellian convention of reading M-1:
    n (m / (pi T))^{3/2} exp(-m |c - u|^2 / T), so <|c - u|^2> = 3 T / (2 m))."""
    import torch
    dc = 2.0 * L / N
    c = -L + (torch.arange(N, dtype=torch.float64, device=f.device) + 0.5) * dc
    g = f.reshape(*f.shape[:3], N, N, N)
    w = dc ** 3
    n = g.sum(dim=(3, 4, 5)) * w
    mx = (g.sum(dim=(4, 5)) * c).sum(-1) * w
    my = (g.sum(dim=(3, 5)) * c).sum(-1) * w
    mz = (g.sum(dim=(3, 4)) * c).sum(-1) * w
    c2 = ((g.sum(dim=(4, 5)) * c * c).sum(-1) + (g.sum(dim=(3, 5)) * c * c).sum(-1)
          + (g.sum(dim=(3, 4)) * c * c).sum(-1)) * w
    u = torch.stack((mx, my, mz), dim=-1) / n[..., None]
    m = torch.tensor(mass, dtype=torch.float64, device=f.device)
    T = (2.0 * m / 3.0) * (c2 / n - (u * u).sum(-1))
    return n, u, T


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--dt", type=float, default=None, help="time step (default: the config's)")
    ap.add_argument("--block", type=int, default=250, help="steps between two looks at the moments")
    ap.add_argument("--tol", type=float, default=2e-4,
                    help="steady when, over a block, max |u_y change| < tol u_w and max |T change| < tol u_w^2")
    ap.add_argument("--max-steps", type=int, default=40000)
    a = ap.parse_args()

    import torch
    from workloads import get_config, make_dg_state
    from paper_1903_04670_b200 import Dgfs, Mesh1D, api

    if not torch.cuda.is_available():
        raise SystemExit("couette: needs a CUDA device (there is no CPU path)")
    torch.cuda.set_device(0)
    cfg = get_config("couette")
    dt = cfg.dt if a.dt is None else a.dt
    mesh = Mesh1D(cfg.ne, cfg.order, wall_T=cfg.wall_T, wall_u=cfg.wall_u)
    xi, wq = gll(cfg.order)
    h = 1.0 / cfg.ne
    x = np.array([[(e + 0.5 * (1.0 + s)) * h for s in xi] for e in range(cfg.ne)])
    wx = torch.tensor(np.tile(0.5 * h * wq, (cfg.ne, 1)), device="cuda")
    uw = abs(cfg.wall_u[1][1])

    with Dgfs.from_config(cfg, device=0) as op:
        f = torch.from_numpy(make_dg_state(cfg)).cuda()
        n0, _, _ = moments(f, cfg.N, cfg.L, cfg.mass)
        mass0 = (n0 * wx[..., None]).sum(dim=(0, 1))
        api.dgfs_step_euler(op.ctx, mesh, f, dt, 2)                         # warm-up: workspace, tables in L2
        f = torch.from_numpy(make_dg_state(cfg)).cuda()
        torch.cuda.synchronize()
        launches0 = api.dgfs_launch_count(op.ctx)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        dev_ms, steps, change = 0.0, 0, float("inf")
        mass1 = mass0
        _, u_prev, T_prev = moments(f, cfg.N, cfg.L, cfg.mass)
        t_host = time.perf_counter()
        while steps < a.max_steps:
            ev[0].record()
            api.dgfs_step_euler(op.ctx, mesh, f, dt, a.block)
            ev[1].record()
            torch.cuda.synchronize()
            dev_ms += ev[0].elapsed_time(ev[1])
            steps += a.block
            n, u, T = moments(f, cfg.N, cfg.L, cfg.mass)
            if not bool(torch.isfinite(u).all()):
                raise SystemExit(f"couette: the state blew up after {steps} steps of dt = {dt}")
            # u_y in units of the wall speed, T in units of the viscous-heating scale u_w^2
            change = max(float((u[..., 1] - u_prev[..., 1]).abs().max()) / uw,
                         float((T - T_prev).abs().max()) / uw ** 2)
            u_prev, T_prev = u, T
            mass_prev, mass1 = mass1, (n * wx[..., None]).sum(dim=(0, 1))
            if change < a.tol:
                break
        host_s = time.perf_counter() - t_host
        launches = api.dgfs_launch_count(op.ctx) - launches0
        # mass defect of the collision term on the final state (the fast spectral operator conserves mass only to
        # its spectral accuracy, and the diffuse walls put a jump at c_x = 0 into f); transport and walls conserve
        # mass exactly, so this must equal the drift observed over the last block
        Q = op.collide(f.reshape(-1, cfg.ns, cfg.N ** 3)).reshape(f.shape)
        q_rate = ((Q.sum(-1) * (2.0 * cfg.L / cfg.N) ** 3) * wx[..., None]).sum(dim=(0, 1)) / mass1
        drift_rate = (mass1 - mass_prev) / (a.block * dt) / mass1
        n, u, T = n.cpu().numpy(), u.cpu().numpy(), T.cpu().numpy()
        fmin = float(f.min())

    uy = u[..., 1]
    checks = {
        "steady": bool(change < a.tol),
        "mass_drift_rel": [float(v) for v in ((mass1 - mass0) / mass0).cpu().numpy()],
        "mass_drift_rate_last_block": [float(v) for v in drift_rate.cpu().numpy()],
        "collision_mass_defect_rate_final_state": [float(v) for v in q_rate.cpu().numpy()],
        "uy_antisymmetry": float(np.abs(uy + uy[::-1, ::-1]).max() / uw),
        "n_symmetry": float(np.abs(n - n[::-1, ::-1]).max() / n.max()),
        "slip": [float(1.0 - abs(uy[0, 0, p]) / uw) for p in range(cfg.ns)],
        "uy_monotone": bool(all(np.all(np.diff(uy[:, :, p].reshape(-1)) >= -1e-3 * uw) for p in range(cfg.ns))),
        "ux_max": float(np.abs(u[..., 0]).max() / uw),
        "T_range": [float(T.min()), float(T.max())],
        "f_min_over_f_max": fmin / float(make_dg_state(cfg).max()),
    }
    print(json.dumps({
        "case": "Couette C-01 (Table 2, P:345-375), dgfs_step_euler", "N": cfg.N, "N_rho": cfg.N_rho, "M": cfg.M,
        "ne": cfg.ne, "order": cfg.order, "dt": dt, "steps": steps, "t_final": steps * dt,
        "device_s": dev_ms / 1e3, "host_s": host_s, "ms_per_step": dev_ms / steps,
        "pair_evals_per_s": steps * cfg.ne * (cfg.order + 1) * cfg.ns ** 2 / (dev_ms / 1e3),
        "gpu_launches": int(launches), "last_block_change": change,
        "paper_context": "138 s on one P100 to the steady state (P:333); time step and stopping rule not printed",
        "checks": checks,
        "profiles": {"x": x.reshape(-1).tolist(),
                     "uy_over_wall_speed": [(uy[:, :, p].reshape(-1) / uw).tolist() for p in range(cfg.ns)],
                     "T": [T[:, :, p].reshape(-1).tolist() for p in range(cfg.ns)],
                     "n": [n[:, :, p].reshape(-1).tolist() for p in range(cfg.ns)]},
    }))


if __name__ == "__main__":
    main()
