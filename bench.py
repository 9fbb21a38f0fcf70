#!/usr/bin/env python
"""bench.py -- attempted bead moves/s of the full SCMF step (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

A "step" is one SCMF cycle = soma_step(1): even-set moves, odd-set moves, occupation numbers,
field update over every bead of the workload.  Default workload: C3, the
16.4 M-bead symmetric diblock melt BASELINE.json's metric is quoted on.  One JSON line on stdout.

Multi-GPU: north_star runs the path on one GPU with no sharding and no collective ("replicas
only"): --gpus N runs N independent replicas (different seeds), one process per GPU,
value = total moves of all replicas / max-over-ranks time, scaling "weak".  Started without
torchrun (no WORLD_SIZE in the environment) with N > 1, bench.py starts its N ranks itself
(python -m torch.distributed.run); the line's n_gpus is the number of ranks that ran.

Numbers of the bench line: `value` = the K timed steps (one soma_step(K) call between two CUDA
events; with the default K = 200 that is 20 ms at the burst clock), `sustained` = 5000 further
sweeps in one stretch with the clocks sampled through NVML -- the board reaches its power cap
after ~0.1 s, so `sustained` is the rate a production run sees and the one the documents lead with.

--impl reference times the CPU oracle (oracle/soma_oracle.c, as it stands) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import workloads  # noqa: E402

METRIC = "attempted bead moves/s (full SCMF step)"
UNIT = "moves/s"
MOVE_BYTES_PER_BEAD = 24.0   # fused move kernel: read 12 B + write 12 B per bead per sweep
FIELD_BYTES_PER_CELL = 16.0  # field kernel: read n_t counts + write n_t omegas (n_t = 2), DESIGN.md
SCHEDULERS_PER_SM = 4         # warp schedulers per SM, one instruction per cycle each (B300_MICROARCH.md)


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons during the timed region, sampled through NVML (nvidia-ml-py) every
    millisecond from a thread of this process; nvidia-smi (~50 ms per call) as the fallback."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int, period_s: float = 0.001):
        self.index, self.period, self.samples, self.stop, self.t = index, period_s, [], threading.Event(), None
        self.nvml, self.handle, self.max_mhz, self.source, self.t_from = None, None, None, "nvidia-smi", None
        try:
            import pynvml
            pynvml.nvmlInit()
            # NVML enumerates the physical devices, CUDA the visible ones: find this CUDA device by its UUID,
            # else by its place in a plain integer CUDA_VISIBLE_DEVICES list
            self.handle = None
            try:
                import torch
                uuid = str(torch.cuda.get_device_properties(index).uuid)
                self.handle = pynvml.nvmlDeviceGetHandleByUUID(uuid if uuid.startswith("GPU-") else "GPU-" + uuid)
            except Exception:
                self.handle = None
            if self.handle is None:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                ids = [int(v) for v in vis.split(",")] if vis and all(v.strip().isdigit() for v in vis.split(",")) else None
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(ids[index] if ids and index < len(ids) else index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml, self.source = pynvml, "nvml"
        except Exception:
            self.nvml = None

    def _once(self):
        if self.nvml is not None:
            n = self.nvml
            mhz = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
            r = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
            bits = [n.nvmlClocksEventReasonHwSlowdown, n.nvmlClocksEventReasonHwThermalSlowdown,
                    n.nvmlClocksEventReasonSwThermalSlowdown, n.nvmlClocksEventReasonSwPowerCap]
            return [mhz, self.max_mhz] + [bool(r & b) for b in bits]
        out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                              "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
        f = [v.strip() for v in out.strip().split(",")]
        return [float(f[0]), float(f[1])] + [v.lower().startswith("active") for v in f[2:6]]

    def _run(self):
        while not self.stop.is_set():
            try:
                self.samples.append(self._once() + [time.perf_counter()])
            except Exception:
                if self.nvml is not None:      # NVML failed mid-run: fall back
                    self.nvml, self.source = None, "nvidia-smi"
            self.stop.wait(self.period if self.nvml is not None else 0.1)

    def __enter__(self):
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)
        if self.t_from is not None:            # keep what was sampled while the timed region ran
            inside = [s for s in self.samples if s[-1] >= self.t_from]
            self.samples = inside or self.samples[-1:]
        if not self.samples:                   # a region shorter than one sample: take one now
            try:
                self.samples.append(self._once() + [time.perf_counter()])
            except Exception:
                pass

    def mark(self):
        """The timed region starts now: samples taken earlier (warm-up) are dropped at the end."""
        self.t_from = time.perf_counter()

    def summary(self, region=None):
        """region: (t0, t1) on the perf_counter clock -- the host's estimate of when the timed region ran on the
        device; the number of samples that fall inside it is reported beside the number the statistics are over."""
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["clock query unavailable"]}
        mhz = sorted(s[0] for s in self.samples)
        reasons = [n for i, n in enumerate(self.NAMES) if any(s[2 + i] for s in self.samples)]
        out = {"sm_mhz": mhz[len(mhz) // 2], "sm_min_mhz": mhz[0], "sm_max_mhz": self.samples[0][1],
               "reasons": reasons, "samples": len(mhz), "source": self.source}
        if region is not None:
            out["samples_in_timed_region"] = sum(1 for s in self.samples if region[0] <= s[-1] <= region[1])
            out["window"] = ("samples: from the host's mark() -- the device work queued in front of the start event (spin, "
                             "pre-roll) and the timed region; samples_in_timed_region: those within the last ms_total "
                             "before the closing synchronisation returned")
        return out


def kernel_source_hash() -> str:
    """Identifies the kernels a profile entry was measured on (profiles/traffic.json)."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted((ROOT / "paper_1711_03828_b200" / "csrc").glob("*.cu*")):
        h.update(f.read_bytes())
    return h.hexdigest()[:16]


def profile_entry(name: str):
    """dram bytes and warp instructions per launch of the move kernel from the committed ncu capture, or None
    if there is none for this config or the kernels have changed since (a stale number is worse than none)."""
    f = ROOT / "profiles" / "traffic.json"
    try:
        e = json.loads(f.read_text()).get(name)
        if isinstance(e, dict) and e.get("kernel_hash") == kernel_source_hash():
            return e
    except Exception:
        pass
    return None


def ingest_ncu_csv(csv_path: str, name: str):
    """profiles/traffic.json entry from `ncu --csv --metrics dram__bytes_read.sum,dram__bytes_write.sum,
    smsp__inst_executed.sum -k regex:fused_sweep ... python bench.py --config NAME ...` (the first launch listed)."""
    import csv
    vals = {}
    with open(csv_path) as fh:
        rows = [r for r in csv.reader(fh) if len(r) > 3]
    hdr = next(r for r in rows if "Metric Name" in r)
    i_name, i_unit, i_val, i_id = hdr.index("Metric Name"), hdr.index("Metric Unit"), hdr.index("Metric Value"), hdr.index("ID")
    ids = set()
    for r in rows[rows.index(hdr) + 1:]:               # every launch in the file: the move launches of ONE sweep
        ids.add(r[i_id])
        v = float(r[i_val].replace(",", ""))
        unit = r[i_unit].lower()
        v *= {"kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9}.get(unit, 1.0)
        vals[r[i_name]] = vals.get(r[i_name], 0.0) + v
    f = ROOT / "profiles" / "traffic.json"
    d = json.loads(f.read_text()) if f.exists() else {}
    d = {k: v for k, v in d.items() if isinstance(v, dict)}
    d[name] = {"dram_bytes": int(vals["dram__bytes_read.sum"] + vals["dram__bytes_write.sum"]),
               "inst_executed": int(vals["smsp__inst_executed.sum"]), "launches": len(ids),
               "kernel_hash": kernel_source_hash(),
               "source": f"ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum,smsp__inst_executed.sum -k regex:"
                         f"(fused_sweep|generic_move) -s <5 sweeps> -c <move launches of one sweep> python bench.py --config {name} --steps 5 --warmup 3 "
                         f"--no-cpu-baseline --aged 0; python bench.py --ingest-ncu <csv> --config {name}"}
    f.write_text(json.dumps(d, indent=1, sort_keys=True) + "\n")
    print(json.dumps(d[name]))


def oracle_rate(w, steps: int, warmup: int, budget_s: float = 20.0, one_thread_too: bool = False):
    """Time the oracle, as it stands, on the host cores: full SCMF cycles on a bounded sample."""
    sys.path.insert(0, str(ROOT / "tests"))
    import oracle
    from helpers import oracle_system
    # bounded sample: a melt with the same box/grid/density structure but fewer chains if needed
    probe = w.scaled(min(1.0, 262144 / w.n_beads), name="probe")
    s = oracle_system(probe)
    x, y, z = workloads.gaussian_walks(probe)
    c = s.histogram(x, y, z)
    om = s.fields(c)
    t = time.perf_counter()
    s.step(x, y, z, c, om, 0, 1)
    per_bead = (time.perf_counter() - t) / probe.n_beads
    n_steps = max(1, steps) + max(0, warmup)
    frac = min(1.0, budget_s / (per_bead * w.n_beads * n_steps))
    sample = w if frac >= 1.0 else w.scaled(frac, name=f"{w.name}-sample")
    s = oracle_system(sample)
    x, y, z = workloads.gaussian_walks(sample)
    c = s.histogram(x, y, z)
    om = s.fields(c)
    if warmup:
        s.step(x, y, z, c, om, 0, warmup)
    t = time.perf_counter()
    s.step(x, y, z, c, om, warmup, steps)
    dt = time.perf_counter() - t
    out = {"value": sample.n_beads * steps / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
           "sample": f"{sample.n_chains} chains ({sample.n_beads} beads, {100 * sample.n_beads / w.n_beads:.1f}% of "
                     f"{w.name}; same box, grid and chain architecture), {steps} full SCMF cycles after {warmup} "
                     f"warm-up, OpenMP over chains"}
    if one_thread_too:
        # the oracle on one thread as well, on a sample a tenth of the budget long
        n_all = oracle.num_threads()
        small = w.scaled(min(1.0, 0.1 * budget_s / (per_bead * n_all * w.n_beads)), name=f"{w.name}-1thread")
        s1 = oracle_system(small)
        x, y, z = workloads.gaussian_walks(small)
        c = s1.histogram(x, y, z)
        om = s1.fields(c)
        oracle.set_num_threads(1)
        try:
            t = time.perf_counter()
            s1.step(x, y, z, c, om, 0, 1)
            out["one_thread"] = {"value": small.n_beads / (time.perf_counter() - t), "unit": UNIT, "cores": 1,
                                 "sample": f"{small.n_chains} chains ({small.n_beads} beads), 1 full SCMF cycle"}
        finally:
            oracle.set_num_threads(n_all)
    return out, dt / steps * 1e3


def max_over_ranks(value: float, dist, device) -> float:
    """Timing rule: a multi-GPU number is the slowest rank's.  dist = torch.distributed or None."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_moves_per_s(n_beads: int, steps: int, world: int, ms_total_max: float) -> float:
    """Whole-job throughput of `world` independent replicas (replicas only): all moves of
    all ranks divided by the slowest rank's time."""
    return world * n_beads * steps / (ms_total_max * 1e-3)


def all_configs(P, torch):
    """Step time of every config (profiles/*_all_configs.txt)."""
    peak, _ = peaks()
    from dataclasses import replace
    c3 = workloads.c3()
    # the C3 melt with every chain handed in as a bond list (general-architecture kernel, one launch per
    # independent set), and a melt of the same size of 3-arm stars (31 monomers: centre + 3 arms of 10)
    c3_bonds = replace(c3, name="C3bonds", bonds=(tuple((j, j + 1) for j in range(31)),))
    star = tuple((0 if k == 0 else 1 + a * 10 + k - 1, 1 + a * 10 + k) for a in range(3) for k in range(10))
    stars = replace(c3, name="stars", specs=((528516, (0,) + (0,) * 15 + (1,) * 15),), bonds=(star,))
    n100 = replace(c3, name="N100", specs=((163840, workloads.diblock(100, 50)),), N_ref=100)
    n48 = replace(c3, name="N48", specs=((341333, workloads.diblock(48, 24)),), N_ref=48)
    cases = [("C1", workloads.c1(), {}), ("C2 kappaN=50", workloads.c2(kappaN=50.0), {}), ("C3", c3, {}),
             ("C3 random set order", c3, {"order": 1}), ("C3 molecule-parallel scheme (Code 1)", c3, {"scheme": 1}),
             ("diblock melt N = 100 (25 of 32 lanes)", n100, {}), ("diblock melt N = 48 (24 of 32 lanes)", n48, {}),
             ("C3 chains as bond lists", c3_bonds, {}), ("3-arm star melt, 16.4M beads", stars, {}),
             ("C5 a_s=0.05 (literal)", workloads.c5(), {}),
             ("C5 a_s=0.05 b0^2", workloads.c5(smc_step=0.05 / 63), {}), ("C4", workloads.c4(), {})]
    for name, w, kw in cases:
        sim = P.from_workload(w)
        if "order" in kw:
            sim.set_option(P.OPT_SET_ORDER, 1)
        if "scheme" in kw:
            sim.set_option(P.OPT_SCHEME, kw["scheme"])
        n = 200 if w.n_beads < 2e6 else (50 if w.n_beads < 1e8 else 10)
        sim.step(5)
        sim.sync()
        best = float("inf")
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sim.step(n)
            e1.record()
            sim.sync()
            best = min(best, e0.elapsed_time(e1) / n)
        att, acc, _ = sim.stats()
        print(f"{name:38s} beads {w.n_beads:>10d}  {best * 1e3:9.1f} us/step  {w.n_beads / best / 1e6:8.2f} G moves/s  "
              f"24 B/move of measured HBM peak {MOVE_BYTES_PER_BEAD * w.n_beads / (best * 1e-3) / 1e9 / peak:.3f}  "
              f"acceptance {acc / max(1, att):.3f}", flush=True)
        sim.destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", type=int, default=0)
    ap.add_argument("--density", type=int, default=0)
    ap.add_argument("--aged", type=int, default=5000,
                    help="N = 1: also time this many further sweeps in one stretch (sustained clocks under the power cap; "
                         "the melt orders on the way, SURVEY 8(d)); 0: skip")
    ap.add_argument("--all-configs", action="store_true",
                    help="instead of the bench line: step time of every BASELINE.json config (soma_step(n) between two "
                         "CUDA events), C3 also in random set order, C5 with both Smart-MC steps; one text line each")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE system of N x the config's chains in a box N x as long (same density), molecules "
                         "distributed over the ranks, one all-reduce of the occupation numbers per sweep (SURVEY 8(e)); "
                         "default: N independent replicas")
    ap.add_argument("--peers", action="store_true",
                    help="with --sharded: no all-reduce -- every rank's field kernel reduces all ranks' exchange arrays "
                         "itself over peer memory (CUDA IPC / NVLink), behind a one-element all-reduce as the barrier")
    ap.add_argument("--ingest-ncu", metavar="CSV",
                    help="no run: write the profiles/traffic.json entry of --config from an ncu --csv metrics file")
    args = ap.parse_args()
    if args.ingest_ncu:
        ingest_ncu_csv(args.ingest_ncu, workloads.by_name(args.config).name)
        return
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3   # timing rule: W >= 3
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started the plain way: one process per GPU is this program's multi-GPU form, so start the ranks
        import socket
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve())] + sys.argv[1:]
        raise SystemExit(subprocess.run(cmd).returncode)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but {world} rank(s) were started")
    w = workloads.by_name(args.config)
    config = {"workload": f"{w.name}: {w.note}", "chains": w.n_chains, "beads": w.n_beads, "grid": list(w.grid),
              "box": list(w.box), "chiN": w.chiN, "kappaN": w.kappaN, "A": w.A, "seed": w.seed, "move": w.move,
              "parallelism": "replicas only" if world > 1 else "single GPU",
              "timing": "W warm-up steps (the last five at most enqueued after the synchronisation and ~10 ms of unrelated device work, directly before the start "
                        "event), K steps in one soma_step(K) call between two CUDA events, barrier + synchronize on both sides",
              "l2_policy": (f"inputs larger than L2 (positions {12 * w.n_beads / 1e6:.0f} MB > 126 MB L2); no explicit flush"
                            if 12 * w.n_beads > 126e6 else
                            f"state fits in L2 (positions {12 * w.n_beads / 1e6:.1f} MB) and stays there from sweep to sweep, "
                            "as in a production run of this system; no flush")}

    if args.impl == "reference":
        if rank != 0:
            return
        steps = min(args.steps, 3)
        base, ms = oracle_rate(w, steps, min(args.warmup, 1), one_thread_too=True)
        line = {"impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": world,
                "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config,
                "cpu_baseline": base,
                "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import torch
    import paper_1711_03828_b200 as P
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if torch.cuda.device_count() < world:
        raise SystemExit(f"bench.py: {world} ranks but only {torch.cuda.device_count()} CUDA device(s): one process per GPU")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    from dataclasses import replace
    if args.all_configs:
        if rank == 0:
            all_configs(P, torch)
        return
    if args.sharded:
        # weak scaling of one system: world x the chains in a box world x as long along x (same density, same
        # cell size); every rank moves 1/world of the molecules and holds the whole grid
        from paper_1711_03828_b200.sharded import ShardedSoma
        w = replace(w, specs=tuple((n * world, t) for n, t in w.specs), box=(w.box[0] * world, w.box[1], w.box[2]),
                    grid=(w.grid[0] * world, w.grid[1], w.grid[2]))
        config.update({"parallelism": f"one system over {world} GPU(s): molecules distributed, " +
                                      ("exchange arrays reduced by the field kernel over peer memory" if args.peers and world > 1
                                       else "exchange array all-reduced every sweep"),
                       "chains": w.n_chains, "beads": w.n_beads, "grid": list(w.grid), "box": list(w.box)})

        class _Sharded:                       # the calls bench makes, on this rank's part of the system
            def __init__(self, sh):
                self.sh, self.sim = sh, sh.sim

            def step(self, n):
                self.sh.step(n)

            def set_positions(self, xyz):
                self.sim.set_positions(xyz)
                self.sh._exchange(advance=False)

            def __getattr__(self, name):
                return getattr(self.sim, name)

        sim = _Sharded(ShardedSoma(w, dist=dist, peers=args.peers))
    else:
        wr = w if rank == 0 else replace(w, seed=w.seed + rank)   # independent replicas
        sim = P.from_workload(wr, xyz0=None)       # Gaussian-walk start drawn on the device from the seed
    sim.set_option(P.OPT_KERNEL, args.kernel)
    sim.set_option(P.OPT_DENSITY, args.density)
    nb = sim.n_beads                           # beads this rank moves

    # ---- device-resident throughput ------------------------------------------------------------
    # W warm-up steps, K timed steps between two CUDA events, barrier + synchronize on both sides.  The last (up to
    # five) warm-up steps are enqueued after the first synchronisation, directly in front of the start event, so the
    # timed region starts with the GPU busy (measured: after an idle period the first steps run slower, ~60 us in
    # all, which a 20-step region of 2 ms would carry as +3 %); the events are in stream order, so exactly the K
    # steps lie between them.
    pre_roll = min(5, args.warmup)
    config["pre_roll"] = {"steps": pre_roll, "spin": {"buffer_bytes": 256 << 20, "passes": 120, "approx_ms": 10}}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clk:      # the sampling thread is up before the GPU is left idle for the last time
        sim.step(args.warmup - pre_roll)
        barrier()
        # ~10 ms of unrelated device work (a 256 MB buffer incremented 120 times) between the synchronisation and
        # the pre-roll: the board is back at its working clocks and power state when the pre-roll starts (measured
        # on a 20-step region: 101.9 -> 101.2 us per step); no step of the workload is added or skipped
        spin = torch.empty(64 << 20, dtype=torch.float32, device="cuda")
        for _ in range(120):
            spin.add_(1.0)
        del spin
        sim.step(pre_roll)
        l0 = sim.launch_count()
        clk.mark()
        e0.record()
        sim.step(args.steps)                   # one soma_step(K) call: K x (move launch, field launch), no Python in between
        e1.record()
        barrier()
        t_end = time.perf_counter()            # the closing synchronisation has returned: the device finished just before
    ms_total = e0.elapsed_time(e1)
    timed_region = (t_end - ms_total * 1e-3 - 2e-4, t_end)
    launches = sim.launch_count() - l0
    ms_total = max_over_ranks(ms_total, dist, "cuda")
    value = aggregate_moves_per_s(nb, args.steps, world, ms_total)
    att, acc, sweeps = sim.stats()

    # ---- roofline of the dominant kernel (move kernel), CUDA events inside the library ---------
    sim.set_option(P.OPT_TIMING, 1)
    sim.kernel_times()
    n_roof = min(args.steps, 100)
    for _ in range(n_roof):
        sim.step(1)
    kms, kn = sim.kernel_times()
    sim.set_option(P.OPT_TIMING, 0)
    peak, peak_src = peaks()
    move_ms = kms[P.K_MOVE] / max(1, n_roof)            # all move launches of one sweep
    achieved = MOVE_BYTES_PER_BEAD * nb / (move_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "fused_sweep_kernel (a1+a2+a3)", "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                "ms_per_launch": move_ms / max(1, kn[P.K_MOVE] // max(1, n_roof)),
                "algorithmic_bytes_per_launch": MOVE_BYTES_PER_BEAD * nb,
                "kernel_share_of_step": {"move": kms[P.K_MOVE] / max(1e-12, sum(kms)),
                                         "density": kms[P.K_DENSITY] / max(1e-12, sum(kms)),
                                         "field": kms[P.K_FIELD] / max(1e-12, sum(kms))},
                "full_step_frac": (MOVE_BYTES_PER_BEAD * nb + FIELD_BYTES_PER_CELL * w.n_cells) * args.steps
                                  / (ms_total * 1e-3) / 1e9 / peak}
    roofline["timing_note"] = ("ms_per_launch: CUDA events around every launch inside the library (SOMA_OPT_TIMING), which "
                               "serialises the launches -- without the programmatic-dependent-launch overlap of the timed "
                               "region, so it can exceed ms_per_step; full_step_frac is from the timed region itself")
    # dram bytes and warp instructions per launch of the move kernel from the committed ncu capture of these very
    # kernels (profiles/traffic.json; an entry measured on other kernel sources is ignored)
    prof = profile_entry(w.name)
    roofline["traffic"] = prof["dram_bytes"] if prof else None
    # second roof: warp-instruction issue, one instruction per cycle and scheduler
    clocks_now = clk.summary(timed_region)
    if clocks_now.get("sm_mhz") and prof:
        n_sm = torch.cuda.get_device_properties(local_rank).multi_processor_count
        peak_ips = n_sm * SCHEDULERS_PER_SM * clocks_now["sm_mhz"] * 1e6
        roofline["issue"] = {"bound": "alu", "achieved": prof["inst_executed"] / (move_ms * 1e-3) / 1e12,
                             "peak": peak_ips / 1e12, "unit": "T warp-instr/s",
                             "frac": prof["inst_executed"] / (move_ms * 1e-3) / peak_ips,
                             "instr_per_32_moves": prof["inst_executed"] / (nb / 32.0),
                             "note": f"issue slots of {n_sm} SMs x {SCHEDULERS_PER_SM} schedulers at the sampled SM clock; "
                                     "instructions per launch from profiles/traffic.json; DESIGN.md 6.1"}

    # ---- end to end through the C ABI with host buffers ----------------------------------------
    n_e2e = max(3, min(args.steps, 20))
    xyz_h = torch.empty((3, nb), dtype=torch.float32).pin_memory().numpy()
    om_h = torch.empty((w.n_types, w.n_cells), dtype=torch.float32).pin_memory().numpy()
    cn_h = torch.empty((w.n_types, w.n_cells), dtype=torch.int32).pin_memory().numpy().view(np.uint32)
    sim.positions(xyz_h)
    for _ in range(2):
        sim.set_positions(xyz_h); sim.step(1); sim.positions(xyz_h); sim.fields(om_h, cn_h)
    barrier()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        sim.set_positions(xyz_h)          # H2D 12 B/bead (+ stage 1 on the device)
        sim.step(1)
        sim.positions(xyz_h)              # D2H 12 B/bead
        sim.fields(om_h, cn_h)            # D2H omega + counts
    barrier()
    dt = time.perf_counter() - t0
    dt = max_over_ranks(dt, dist, "cuda")
    e2e = {"value": world * nb * n_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": 12 * nb,
           "d2h_bytes_per_step": 12 * nb + 8 * w.n_types * w.n_cells, "steps": n_e2e}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config,
            "clocks": clocks_now, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "acceptance": acc / max(1, att)}
    if world == 1 and args.aged > 0 and not args.sharded:
        # The same step over a long stretch (default 5000 sweeps, ~0.5 s): the melt orders on the way
        # (PAPER.md:497 puts domain formation at ~2500 MC steps; same access pattern, other field magnitudes),
        # and the board reaches its power cap, so the SM clock is the sustained one, not the burst clock of the
        # short timed region above (the kernel is bound by instruction issue, so its time follows the clock).
        att1, acc1, _ = sim.stats()
        barrier()
        with ClockSampler(local_rank) as clk_s:
            e0.record()
            sim.step(args.aged)
            e1.record()
            barrier()
        ms_aged = e0.elapsed_time(e1)
        att2, acc2, _ = sim.stats()
        _, cnt = sim.fields()
        cnt = cnt.astype(np.float64)
        tot = np.maximum(cnt.sum(0), 1.0)
        line["sustained"] = {"sweeps": int(args.aged), "value": nb * args.aged / (ms_aged * 1e-3), "unit": UNIT,
                             "ms_per_step": ms_aged / args.aged, "clocks": clk_s.summary(),
                             "full_step_frac": (MOVE_BYTES_PER_BEAD * nb + FIELD_BYTES_PER_CELL * w.n_cells) * args.aged
                                               / (ms_aged * 1e-3) / 1e9 / peak,
                             "acceptance": (acc2 - acc1) / max(1, att2 - att1),
                             "mean_abs_phiA_minus_phiB": float(np.mean(np.abs(cnt[0] - cnt[-1]) / tot)) if w.n_types > 1 else None}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"], _ = oracle_rate(w, 2, 1, one_thread_too=True)
    sim.destroy()
    if dist is not None:
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


if __name__ == "__main__":
    main()
