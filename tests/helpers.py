"""Test-side glue: build an oracle system from a workloads.Workload (tests may import both)."""
from __future__ import annotations

import numpy as np

import oracle
from workloads import Workload


def oracle_system(w: Workload, **over) -> oracle.OracleSystem:
    kw = dict(specs=[(n, np.asarray(t, dtype=np.uint8)) for n, t in w.specs], N_ref=w.N_ref,
              n_types=w.n_types, box=w.box, grid=w.grid, chiN=w.chiN, kappaN=w.kappaN, A=w.A,
              seed=w.seed, hamiltonian=0, smc_step=w.smc_step)
    if getattr(w, "bonds", None):
        kw["bonds"] = [None if b is None else np.asarray(b, dtype=np.uint32).reshape(-1, 2) for b in w.bonds]
    kw.update(over)
    return oracle.OracleSystem(**kw)


def chain_layout(w: Workload):
    """(first_bead, N) of every chain, chain-major."""
    out, g = [], 0
    for n, t in w.specs:
        N = len(t)
        for _ in range(n):
            out.append((g, N))
            g += N
    return out
