"""A system spread over ranks: molecules are distributed, the grid is
replicated, the occupation numbers are summed over the ranks after every sweep.  On CPU:
  * the host logic that splits the molecules (paper_1711_03828_b200.sharded),
  * the oracle's "part of a larger system" mode against the (pinned) oracle of the undivided system,
  * the exchange protocol with two gloo ranks: each rank moves its molecules, one all-reduce of the
    integer counts, every rank computes omega -- the trajectory equals the undivided one bit for bit,
    because the Philox counter is the bead's index in the whole system and integer sums commute.
"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
sys.path.insert(0, str(ROOT / "tests"))

import oracle  # noqa: E402
import workloads  # noqa: E402
from helpers import oracle_system  # noqa: E402
from paper_1711_03828_b200.sharded import local_positions, shard_chains, shard_layout  # noqa: E402


def _blend():
    return workloads.Workload("shard_blend", ((37, workloads.diblock(32, 16)), (21, workloads.homopolymer(8, 1)),
                                              (5, workloads.homopolymer(33))), 32, 2, (4.0, 4.0, 3.0), (8, 8, 6),
                              20.0, 50.0, 0.1, 11)


def test_shard_chains_partition_every_molecule_exactly_once():
    for n in (0, 1, 5, 37, 1000, 512000):
        for world in (1, 2, 3, 8):
            parts = [shard_chains(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))       # contiguous, no gap
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1                                         # balanced


def test_shard_layout_offsets_are_the_global_bead_indices():
    w = _blend()
    specs = [(n, t) for n, t in w.specs]
    seen = np.zeros(w.n_beads, np.int32)
    for rank in range(3):
        local, first, n_global, slices = shard_layout(specs, rank, 3)
        assert n_global == w.n_beads
        for (n_loc, t), f, (a, b), (n_all, _) in zip(local, first, slices, specs):
            assert a == f and b - a == n_loc * len(t)
            seen[a:b] += 1
    assert (seen == 1).all()
    # the undivided system: one rank
    local, first, n_global, slices = shard_layout(specs, 0, 1)
    assert [l[0] for l in local] == [n for n, _ in specs] and first[0] == 0 and slices[-1][1] == w.n_beads


def _run_whole(w, xyz0, n_sweeps, move, **over):
    orc = oracle_system(w, **over)
    x, y, z = (xyz0[a].copy() for a in range(3))
    om = orc.fields(orc.histogram(x, y, z))
    for sweep in range(n_sweeps):
        orc.sweep(x, y, z, om, sweep, move)
        cnt = orc.histogram(x, y, z)
        om = orc.fields(cnt)
    return np.stack([x, y, z]), cnt, om


def _part(w, rank, world, **over):
    specs = [(n, np.asarray(t, np.uint8)) for n, t in w.specs]
    local, first, n_global, slices = shard_layout(specs, rank, world)
    return oracle_system(w, specs=[(n, t) for n, t in local], spec_first_bead=first, global_n_beads=n_global, **over), slices


def test_oracle_parts_reproduce_the_undivided_oracle():
    """Three parts moved one after the other in one process, counts added by hand; local moves in fixed
    and in random set order (the order bit is drawn for the chain's index in the whole system), Smart-MC."""
    w = _blend()
    xyz0 = np.stack(workloads.gaussian_walks(w))
    for move, over in ((oracle.MOVE_LOCAL, {}), (oracle.MOVE_LOCAL, {"set_order": 1}),
                       (oracle.MOVE_SMC, {"smc_step": 0.05 / 31})):
        want_xyz, want_cnt, want_om = _run_whole(w, xyz0, 3, move, **over)
        parts = [_part(w, r, 3, **over) for r in range(3)]
        pos = [local_positions(xyz0, sl) for _, sl in parts]
        cnt = sum(p.histogram(*q).astype(np.int64) for (p, _), q in zip(parts, pos)).astype(np.uint32)
        om = parts[0][0].fields(cnt)
        for sweep in range(3):
            for (p, _), q in zip(parts, pos):
                p.sweep(q[0], q[1], q[2], om, sweep, move)
            cnt = sum(p.histogram(*q).astype(np.int64) for (p, _), q in zip(parts, pos)).astype(np.uint32)
            om = parts[0][0].fields(cnt)
        for (p, sl), q in zip(parts, pos):
            assert np.array_equal(q, local_positions(want_xyz, sl))
        assert np.array_equal(cnt, want_cnt) and np.array_equal(om, want_om)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = _blend()
    xyz0 = np.stack(workloads.gaussian_walks(w))          # seeded: the same on every rank
    part, slices = _part(w, rank, world)
    q = local_positions(xyz0, slices)

    def exchange():
        t = torch.from_numpy(part.histogram(q[0], q[1], q[2]).view(np.int32).copy())
        dist.all_reduce(t)                                 # the only collective of the path
        cnt = t.numpy().view(np.uint32)
        return cnt, part.fields(cnt)

    cnt, om = exchange()
    for sweep in range(3):
        part.sweep(q[0], q[1], q[2], om, sweep, oracle.MOVE_LOCAL)
        cnt, om = exchange()
    out[rank] = (q.copy(), cnt.copy(), om.copy(), slices)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_with_one_all_reduce_per_sweep_equal_the_undivided_run():
    w = _blend()
    xyz0 = np.stack(workloads.gaussian_walks(w))
    want_xyz, want_cnt, want_om = _run_whole(w, xyz0, 3, oracle.MOVE_LOCAL)
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    for rank in (0, 1):
        q, cnt, om, slices = res[rank]
        assert np.array_equal(q, local_positions(want_xyz, slices))
        assert np.array_equal(cnt, want_cnt) and np.array_equal(om, want_om)      # every rank holds the whole grid
