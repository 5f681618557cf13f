"""Test infrastructure: the CPU oracle over many (point, pair) evaluations in forked worker processes, a per-session
cache of its tables, and a log of the achieved GPU-vs-oracle errors.  Nothing here computes anything of the method:
every number comes out of `oracle.collide.collide_pair` / `oracle.tables.precompute` as they stand.

The workers are forked after the tables exist (copy-on-write, nothing is pickled on the way in) and only ever run
numpy; they never touch CUDA, so forking from a process that holds a CUDA context is safe.
"""
import json
import multiprocessing as mp
import os
import time

import numpy as np

_STATE = {}
_TABLES = {}


def n_workers() -> int:
    env = os.environ.get("DGFS_ORACLE_WORKERS")
    return max(1, int(env)) if env else max(1, os.cpu_count() or 1)


def tables_for(cfg, **kw):
    """oracle.tables.precompute for a workload config, computed once per test session."""
    from oracle.tables import precompute
    key = (cfg.name, cfg.N, cfg.N_rho, cfg.M, tuple(sorted(kw.items())))
    if key not in _TABLES:
        vss = any(a != 1.0 for row in cfg.alpha for a in row)
        kn = {"kn": cfg.kn} if cfg.kn else {}
        _TABLES[key] = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha,
                                  workers=(n_workers() if vss else 1), **kn, **kw)
    return _TABLES[key]


def drop_tables(cfg=None):
    for k in [k for k in _TABLES if cfg is None or k[0] == cfg.name]:
        del _TABLES[k]


def _eval(task):
    from oracle.collide import collide_pair
    x, p, q = task
    return collide_pair(_STATE["tab"], p, q, _STATE["f"][x, p], _STATE["f"][x, q])


def collide_pairs_pool(tab, f, pairs=None):
    """f[nx][ns][N^3] -> Qpq[nx][ns][ns][N^3] (NaN for pairs not asked for): oracle.collide.collide_pair per
    (point, pair), distributed over the host cores."""
    nx, ns, N3 = f.shape
    pairs = list(pairs) if pairs is not None else [(p, q) for p in range(ns) for q in range(ns)]
    tasks = [(x, p, q) for x in range(nx) for (p, q) in pairs]
    _STATE["tab"], _STATE["f"] = tab, f
    nw = min(n_workers(), len(tasks))
    try:
        if nw <= 1:
            res = [_eval(t) for t in tasks]
        else:
            with mp.get_context("fork").Pool(nw) as pool:
                res = pool.map(_eval, tasks, chunksize=1)
    finally:
        _STATE.clear()
    out = np.full((nx, ns, ns, N3), np.nan)
    for (x, p, q), r in zip(tasks, res):
        out[x, p, q] = r
    return out


def collide_pool(tab, f):
    """f[nx][ns][N^3] -> Q[nx][ns][N^3] = sum_q beta_pq Q^(pq) (Eq. 1), same pool."""
    return collide_pairs_pool(tab, f).sum(axis=2)


# ------------------------------------------------------------------------------ achieved-error log
def log_path():
    return os.environ.get("DGFS_PARITY_LOG", os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))),
                                                          "gpurun_out", "parity_log.jsonl"))


def record(config, what, err, tol, **extra):
    """Append one achieved error (GPU vs oracle) to the parity log; profiles/rNN_parity.md is written from it."""
    line = dict(config=config, what=what, err=float(err), tol=float(tol), when=time.strftime("%Y-%m-%dT%H:%M:%S"), **extra)
    print("parity %s | %s: %.3e (tolerance %.1e)" % (config, what, err, tol))
    try:
        os.makedirs(os.path.dirname(log_path()), exist_ok=True)
        with open(log_path(), "a") as fh:
            fh.write(json.dumps(line) + "\n")
    except OSError:
        pass
