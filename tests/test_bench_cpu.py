"""Host-side logic of bench.py for more than one rank, on CPU with the gloo backend (world size 2):
the max-over-ranks timing rule, the replica aggregation, and the reference arm under torchrun
(rank 0 alone runs and prints, the other ranks exit 0 without work)."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    slowest = bench.max_over_ranks(local_ms, dist, "cpu")
    out[rank] = (slowest, bench.aggregate_moves_per_s(1000, 4, world, slowest))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_aggregation_world_size_2():
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]
    slowest, value = res[0]
    assert slowest == 15.0                              # the slower rank's time on both ranks
    assert abs(value - 2 * 1000 * 4 / 15e-3) < 1e-6     # all replicas' moves / slowest time


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "C1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_gpus_2_without_torchrun_starts_two_ranks():
    """`python bench.py --gpus 2 ...` as the driver runs it (no torchrun, no WORLD_SIZE): bench.py starts its
    two ranks itself; the reference arm's rank 0 prints the one line, which says two ranks ran."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    cmd = [sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--config", "C1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2
    assert line["cpu_baseline"]["one_thread"]["cores"] == 1 and line["cpu_baseline"]["one_thread"]["value"] > 0


def test_rank_count_must_match_gpus():
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "C1"],
                         capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert res.returncode != 0 and "rank(s) were started" in res.stderr


def test_stale_profile_entries_are_ignored(tmp_path, monkeypatch):
    import bench
    monkeypatch.setattr(bench, "ROOT", tmp_path)
    (tmp_path / "profiles").mkdir()
    (tmp_path / "paper_1711_03828_b200" / "csrc").mkdir(parents=True)
    (tmp_path / "paper_1711_03828_b200" / "csrc" / "k.cuh").write_text("v1")
    (tmp_path / "profiles" / "traffic.json").write_text(json.dumps(
        {"C3": {"dram_bytes": 5, "inst_executed": 7, "kernel_hash": bench.kernel_source_hash()}, "C1": 12345}))
    assert bench.profile_entry("C3")["dram_bytes"] == 5 and bench.profile_entry("C1") is None
    (tmp_path / "paper_1711_03828_b200" / "csrc" / "k.cuh").write_text("v2")      # the kernels changed
    assert bench.profile_entry("C3") is None


def test_ingest_ncu_csv_sums_the_launches_of_one_sweep(tmp_path, monkeypatch):
    import bench
    monkeypatch.setattr(bench, "ROOT", tmp_path)
    (tmp_path / "profiles").mkdir()
    (tmp_path / "paper_1711_03828_b200" / "csrc").mkdir(parents=True)
    (tmp_path / "paper_1711_03828_b200" / "csrc" / "k.cuh").write_text("kernels")
    csv = tmp_path / "t.csv"
    head = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"'
    row = lambda i, m, u, v: f'"{i}","1","python","h","k","1","7","(640, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","{m}","{u}","{v}"'
    csv.write_text("==PROF== Connected\n" + head + "\n" + "\n".join([
        row(0, "dram__bytes_read.sum", "Mbyte", "200.5"), row(0, "dram__bytes_write.sum", "byte", "1,000"),
        row(0, "smsp__inst_executed.sum", "inst", "70"), row(1, "dram__bytes_read.sum", "byte", "24"),
        row(1, "dram__bytes_write.sum", "byte", "6"), row(1, "smsp__inst_executed.sum", "inst", "5")]) + "\n")
    bench.ingest_ncu_csv(str(csv), "C5")
    e = bench.profile_entry("C5")
    assert e["dram_bytes"] == 200500000 + 1000 + 30 and e["inst_executed"] == 75 and e["launches"] == 2
