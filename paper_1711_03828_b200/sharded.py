"""One SCMF system spread over several GPUs, one process per GPU.

The paper's parallelisation: "molecules are distributed among the MPI ranks", every rank keeps the
whole grid, and after every MC step the densities of all ranks are summed (one all-reduce of the integer
occupation numbers); every rank then computes omega redundantly.  Here a rank is a
process with one B200, the all-reduce is ``torch.distributed.all_reduce`` (NCCL over NVLink on GPUs) run
in place on the library's exchange array -- the array this rank's move kernel counts into and the field
kernel reads the sum from (no copy, no conversion in between) -- the only exchange step of the path.
Everything else is the single-GPU library: ``soma_init_shard``, ``soma_shard_moves``,
``soma_shard_exchange``, ``soma_shard_fields`` (include/soma_b200.h).

``peers=True`` replaces the all-reduce by the library's peer mode: the ranks exchange the CUDA IPC handles of
their exchange allocations once, and from then on every rank's field kernel reads all ranks' arrays over
NVLink / NVSwitch peer memory and reduces them itself -- the exchange step and a4 in one kernel.  What is left of
the collective is a barrier (a one-element all-reduce in stream order with NCCL; a stream synchronisation and a
host barrier with any other backend).

Because the Philox counter of a bead is its index in the whole system and integer sums commute, the
trajectory does not depend on the number of ranks: positions, occupation numbers and fields equal
those of the undivided system bit for bit.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import binding as B


def shard_chains(n_chains: int, rank: int, world: int) -> Tuple[int, int]:
    """Molecules [c0, c1) of ``n_chains`` that rank ``rank`` of ``world`` owns: contiguous, sizes differ by <= 1."""
    assert 0 <= rank < world
    return (n_chains * rank) // world, (n_chains * (rank + 1)) // world


def shard_layout(specs: Sequence[Tuple], rank: int, world: int):
    """Split every architecture's molecules over the ranks.

    specs: (n_chains, types[, bonds]) per architecture, the whole system.  Returns
      local_specs      the same with this rank's molecule counts
      spec_first_bead  index in the whole system of the first bead of this rank's molecules, per architecture
      global_n_beads   beads of the whole system
      slices           per architecture, the (start, stop) range of this rank's beads in the whole system's arrays
    """
    local_specs, first, slices = [], [], []
    g = 0
    for sp in specs:
        n, N = int(sp[0]), len(sp[1])
        c0, c1 = shard_chains(n, rank, world)
        local_specs.append((c1 - c0,) + tuple(sp[1:]))
        first.append(g + c0 * N)
        slices.append((g + c0 * N, g + c1 * N))
        g += n * N
    return local_specs, first, g, slices


def local_positions(xyz_global: np.ndarray, slices: Sequence[Tuple[int, int]]) -> np.ndarray:
    """This rank's columns of the whole system's (3, n_beads) position array, architectures in order."""
    return np.ascontiguousarray(np.concatenate([xyz_global[:, a:b] for a, b in slices], axis=1))


class ShardedSoma:
    """This rank's part of a system described by a ``workloads.Workload`` (rank / world from ``dist``)."""

    def __init__(self, w, dist=None, xyz0_global: Optional[np.ndarray] = None, stream: Optional[int] = None,
                 peers: bool = False):
        import torch
        self.dist = dist
        self.rank = dist.get_rank() if dist is not None else 0
        self.world = dist.get_world_size() if dist is not None else 1
        bonds = getattr(w, "bonds", None) or [None] * len(w.specs)
        specs = [(n, t, b) for (n, t), b in zip(w.specs, bonds)]
        local_specs, first, n_global, self.slices = shard_layout(specs, self.rank, self.world)
        xyz0 = None if xyz0_global is None else local_positions(np.asarray(xyz0_global, np.float32), self.slices)
        self.sim = B.Soma(local_specs, w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, w.A, w.seed, xyz0=xyz0,
                          stream=stream, spec_first_bead=first, global_n_beads=n_global)
        if getattr(w, "move", "local") == "smc":
            self.sim.set_option(B.OPT_SMC_STEP, w.smc_step)
            self.sim.set_option(B.OPT_MOVE, B.MOVE_SMC)
        self.n_beads_global = n_global
        self.n_types = w.n_types
        # the library's exchange array as a tensor (uint32 bits in int32: sums are exact modulo 2^32)
        self.exchange = self.sim.shard_exchange_tensor()
        self.peers = bool(peers) and self.world > 1
        if self.peers:
            handles = [None] * self.world
            dist.all_gather_object(handles, self.sim.shard_peer_handle())
            self.sim.shard_set_peers(self.world, self.rank,
                                     handles=[None if r == self.rank else h for r, h in enumerate(handles)])
            self._in_stream = dist.get_backend() == "nccl"
            self._token = torch.zeros(1, dtype=torch.int32, device="cuda") if self._in_stream else None
        self._exchange(advance=False)

    def _exchange(self, advance: bool) -> None:
        if self.peers:
            # every rank's kernels have counted before any rank's field kernel reads: a barrier is all that is
            # left of the collective (in stream order with NCCL: no host synchronisation)
            if self._in_stream:
                self.dist.all_reduce(self._token)
            else:
                self.sim.sync()
                self.dist.barrier()
        elif self.dist is not None and self.world > 1:
            self.dist.all_reduce(self.exchange)                   # the only collective of the path (sum), in place
        self.sim.shard_fields(advance=advance)                    # a4 from the whole system's n_i(c)

    def step(self, n_sweeps: int = 1) -> None:
        for _ in range(int(n_sweeps)):
            self.sim.shard_moves()                                # a1, a2 | a5
            self._exchange(advance=True)

    def positions(self) -> np.ndarray:
        """This rank's molecules, (3, local beads)."""
        return self.sim.positions()

    def fields(self):
        """(omega, occupation numbers of the whole system), host arrays."""
        return self.sim.fields()

    def sync(self) -> None:
        self.sim.sync()

    def destroy(self) -> None:
        self.sim.destroy()
