"""Seeded synthetic workloads: the five BASELINE.json melts and a Gaussian-walk start state.

This module serves both the CPU oracle and the CUDA path with *inputs* and holds none of the
method's arithmetic: no Philox, no energies, no cell index, no field formula.  It only describes
systems (chains, types, box, grid, chiN, kappaN, A, seed) and draws chain conformations from
numpy's own generator -- the conformations a dense melt of ideal Gaussian chains has
(harmonic bonds = coarse-grained Gaussian chain; BASELINE.json configs: "Gaussian
random walks, per-axis bond std R_e/sqrt(3 (N-1)), first bead uniform in the box").

The paper's own benchmark inputs (homopolymer / diblock melts given only by n, N, sqrt(Nbar),
Delta L and the box) are not available; these melts stand in for
them with the same structure (N = 16-64, sqrt(Nbar) = 32-128, Delta L ~ b_0, 16-33 beads/cell).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import List, Sequence, Tuple

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    specs: Tuple[Tuple[int, Tuple[int, ...]], ...]   # (n_chains, per-bead types of one chain)
    N_ref: int
    n_types: int
    box: Tuple[float, float, float]
    grid: Tuple[int, int, int]
    chiN: float
    kappaN: float
    A: float
    seed: int
    move: str = "local"        # "local" | "smc"
    smc_step: float = 0.0
    note: str = ""
    bonds: Tuple = ()          # per spec: None (linear chain) or a tuple of (i, j) monomer pairs; () = all linear

    @property
    def n_beads(self) -> int:
        return sum(n * len(t) for n, t in self.specs)

    @property
    def n_chains(self) -> int:
        return sum(n for n, _ in self.specs)

    @property
    def n_cells(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]

    def scaled(self, factor: float, name: str | None = None) -> "Workload":
        """Same melt with `factor` times the chains (box and grid unchanged): for bounded samples."""
        specs = tuple((max(1, int(round(n * factor))), t) for n, t in self.specs)
        return replace(self, specs=specs, name=name or f"{self.name}x{factor:g}")


def diblock(N: int, n_A: int) -> Tuple[int, ...]:
    return tuple([0] * n_A + [1] * (N - n_A))


def homopolymer(N: int, t: int = 0) -> Tuple[int, ...]:
    return tuple([t] * N)


def c1() -> Workload:
    return Workload("C1", ((2048, diblock(32, 16)),), 32, 2, (4.0, 4.0, 4.0), (16, 16, 16),
                    20.0, 50.0, 0.1, 42, note="AB diblock melt, 65,536 beads")


def c2(kappaN: float = 0.0) -> Workload:
    return Workload(f"C2k{int(kappaN)}", ((32768, homopolymer(32)),), 32, 1, (8.0, 8.0, 8.0),
                    (32, 32, 32), 0.0, kappaN, 0.1, 42, note="ideal-chain / homogeneous melt, 1.05M beads")


def c3() -> Workload:
    return Workload("C3", ((512000, diblock(32, 16)),), 32, 2, (20.0, 20.0, 10.0), (100, 100, 50),
                    30.0, 50.0, 0.1, 7, note="symmetric AB diblock melt, 16.4M beads (headline)")


def c4() -> Workload:
    return Workload("C4", ((8388608, diblock(32, 16)),), 32, 2, (64.0, 64.0, 16.0), (320, 320, 80),
                    25.0, 50.0, 0.1, 7, note="large diblock melt, 268M beads")


def c5(smc_step: float = 0.05) -> Workload:
    # f_A = 0.3 of N = 64 is 19.2 beads: 19 A + 45 B (realised f_A = 0.2969), reading R15
    return Workload("C5", ((400000, diblock(64, 19)), (200000, homopolymer(16))), 64, 2,
                    (24.0, 24.0, 24.0), (120, 120, 120), 35.0, 50.0, 0.1, 7, move="smc",
                    smc_step=smc_step, note="diblock/homopolymer blend with Smart-MC moves, 28.8M beads")


def by_name(name: str) -> Workload:
    table = {"C1": c1, "C2": c2, "C2k0": lambda: c2(0.0), "C2k50": lambda: c2(50.0), "C3": c3,
             "C4": c4, "C5": c5}
    return table[name]()


def gaussian_walks(w: Workload, seed: int | None = None) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Chain-major SoA float32 positions: first bead uniform in the box, then a random walk with
    per-axis bond standard deviation R_e0 / sqrt(3 (N_ref - 1)); unwrapped (never folded)."""
    rng = np.random.default_rng(w.seed if seed is None else seed)
    sigma = 1.0 / np.sqrt(3.0 * (w.N_ref - 1)) if w.N_ref > 1 else 0.0
    out: List[np.ndarray] = []
    for n_chains, types in w.specs:
        N = len(types)
        steps = rng.standard_normal((n_chains, N, 3)) * sigma
        steps[:, 0, :] = rng.random((n_chains, 3)) * np.asarray(w.box, dtype=np.float64)
        out.append(np.cumsum(steps, axis=1).reshape(n_chains * N, 3))
    pos = np.concatenate(out, axis=0)
    return tuple(np.ascontiguousarray(pos[:, a], dtype=np.float32) for a in range(3))  # type: ignore


def small_cases() -> Sequence[Workload]:
    """Edge and ragged cases for parity tests: odd N, N = 1, 2, non-cubic grids, mixed specs."""
    return (
        Workload("tiny_N1", ((257, (0,)),), 1, 1, (2.0, 3.0, 1.0), (4, 6, 2), 0.0, 10.0, 0.1, 1),
        Workload("tiny_N2", ((1000, (0, 1)),), 2, 2, (2.0, 2.0, 2.0), (5, 7, 3), 8.0, 20.0, 0.3, 2),
        Workload("odd_N5", ((333, (0, 0, 1, 1, 1)),), 5, 2, (3.0, 2.0, 2.5), (9, 7, 8), 12.0, 30.0, 0.2, 3),
        Workload("ragged_N33", ((77, diblock(33, 10)),), 33, 2, (3.0, 3.0, 3.0), (12, 12, 12), 15.0, 40.0, 0.1, 4),
        Workload("even_N6", ((4099, diblock(6, 3)),), 6, 2, (5.0, 4.0, 3.0), (20, 16, 12), 10.0, 25.0, 0.1, 5),
        Workload("N100", ((321, diblock(100, 50)),), 100, 2, (6.0, 6.0, 2.0), (30, 30, 10), 17.0, 50.0, 0.05, 6),
        Workload("N256", ((130, diblock(256, 64)),), 256, 2, (8.0, 8.0, 4.0), (48, 48, 24), 28.0, 50.0, 0.03, 8),
        Workload("blend", ((999, diblock(64, 19)), (501, homopolymer(16)), (13, homopolymer(7, 1))), 64, 2,
                 (6.0, 6.0, 6.0), (30, 30, 30), 35.0, 50.0, 0.1, 7),
        Workload("three_types", ((600, (0,) * 8 + (1,) * 8 + (2,) * 16),), 32, 3, (4.0, 4.0, 4.0),
                 (16, 16, 16), 20.0, 50.0, 0.1, 9),
    )
