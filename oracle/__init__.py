"""ctypes front-end of the CPU oracle (``oracle/soma_oracle.c``).

TEST INFRASTRUCTURE, NOT PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  Nothing in
``paper_1711_03828_b200/`` imports it and it imports nothing from there.

The wrapper only marshals arguments; every number it returns is computed by the C file, which
follows PAPER.md (arXiv:1711.03828) Eq. 2, 4, 12, 13, 15 and Code 2 step by step.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "soma_oracle.c"
_LIB = _HERE / "libsoma_oracle.so"
MAX_TYPES = 8

# -ffp-contract=off: no implicit fused multiply-add; the fp32 roundings are the ones written out.
# -mfma only lets the explicit fmaf() calls compile to one instruction (same result as libm's).
_CFLAGS = ["-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-mfma",
           "-fopenmp", "-Wall", "-Wextra"]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.run(["gcc", *_CFLAGS, str(_SRC), "-o", str(tmp), "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _System(C.Structure):
    _fields_ = [
        ("n_specs", C.c_uint32),
        ("spec_n_chains", C.POINTER(C.c_uint64)),
        ("spec_n_beads", C.POINTER(C.c_uint32)),
        ("types", C.POINTER(C.c_uint8)),
        ("n_types", C.c_uint32),
        ("N_ref", C.c_uint32),
        ("box", C.c_float * 3),
        ("grid", C.c_int32 * 3),
        ("chiN", C.c_float * (MAX_TYPES * MAX_TYPES)),
        ("kappaN", C.c_float),
        ("A", C.c_float),
        ("seed", C.c_uint64),
        ("hamiltonian", C.c_int32),
        ("smc_step", C.c_float),
        ("set_order", C.c_int32),
        ("field_every", C.c_uint32),
        ("scheme", C.c_int32),
        ("spec_n_bonds", C.POINTER(C.c_uint32)),
        ("bonds", C.POINTER(C.c_uint32)),
        ("ext_field", C.POINTER(C.c_float)),
        ("forbidden", C.POINTER(C.c_uint8)),
        ("spec_first_bead", C.POINTER(C.c_uint64)),
        ("global_n_beads", C.c_uint64),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        P = C.POINTER
        fp, u32p, u8p = P(C.c_float), P(C.c_uint32), P(C.c_uint8)
        sysp = P(_System)
        L.soma_oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.soma_oracle_philox4x32_10.restype = None
        L.soma_oracle_u23.argtypes = [C.c_uint32]
        L.soma_oracle_u23.restype = C.c_float
        L.soma_oracle_n_beads.argtypes = [sysp]
        L.soma_oracle_n_beads.restype = C.c_uint64
        L.soma_oracle_cell_index.argtypes = [sysp, C.c_float, C.c_float, C.c_float]
        L.soma_oracle_cell_index.restype = C.c_int64
        L.soma_oracle_histogram.argtypes = [sysp, fp, fp, fp, u32p]
        L.soma_oracle_histogram.restype = None
        L.soma_oracle_fields.argtypes = [sysp, u32p, fp]
        L.soma_oracle_fields.restype = None
        L.soma_oracle_local_proposal.argtypes = [sysp, C.c_uint64, C.c_uint64, fp, fp]
        L.soma_oracle_local_proposal.restype = None
        L.soma_oracle_local_delta_e.argtypes = [sysp, fp, fp, fp, fp, C.c_uint64, C.c_int, C.c_int,
                                                C.c_uint32, fp, fp, fp, fp]
        L.soma_oracle_local_delta_e.restype = None
        L.soma_oracle_metropolis.argtypes = [C.c_float, C.c_float]
        L.soma_oracle_metropolis.restype = C.c_int
        L.soma_oracle_smc_proposal.argtypes = [sysp, C.c_uint64, C.c_uint64, fp, fp]
        L.soma_oracle_smc_proposal.restype = None
        L.soma_oracle_smc_delta.argtypes = [sysp, fp, fp, fp, fp, C.c_uint64, C.c_int, C.c_int,
                                            C.c_uint32, fp, fp, fp, fp, fp]
        L.soma_oracle_smc_delta.restype = None
        L.soma_oracle_first_set.argtypes = [sysp, C.c_uint64, C.c_uint64]
        L.soma_oracle_first_set.restype = C.c_uint32
        L.soma_oracle_sweep.argtypes = [sysp, fp, fp, fp, fp, C.c_uint64, C.c_int, u8p]
        L.soma_oracle_sweep.restype = C.c_uint64
        L.soma_oracle_sets.argtypes = [sysp, C.c_uint32, u32p]
        L.soma_oracle_sets.restype = C.c_uint32
        L.soma_oracle_pick.argtypes = [sysp, C.c_uint64, C.c_uint64, C.c_uint32]
        L.soma_oracle_pick.restype = C.c_uint32
        L.soma_oracle_sweep_molecules.argtypes = [sysp, fp, fp, fp, fp, C.c_uint64, C.c_int, u8p]
        L.soma_oracle_sweep_molecules.restype = C.c_uint64
        L.soma_oracle_step.argtypes = [sysp, fp, fp, fp, u32p, fp, C.c_uint64, C.c_uint32, C.c_int, u8p]
        L.soma_oracle_step.restype = C.c_uint64
        L.soma_oracle_init_positions.argtypes = [sysp, fp, fp, fp]
        L.soma_oracle_init_positions.restype = None
        L.soma_oracle_num_threads.argtypes = []
        L.soma_oracle_num_threads.restype = C.c_int
        L.soma_oracle_set_num_threads.argtypes = [C.c_int]
        L.soma_oracle_set_num_threads.restype = None
        _lib = L
    return _lib


def _fp(a: np.ndarray):
    assert a.dtype == np.float32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _u32p(a: np.ndarray):
    assert a.dtype == np.uint32 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


def _u8p(a: Optional[np.ndarray]):
    if a is None:
        return C.POINTER(C.c_uint8)()
    assert a.dtype == np.uint8 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_uint8))


MOVE_LOCAL = 1
MOVE_SMC = 2


def philox4x32_10(ctr: Sequence[int], key: Sequence[int]) -> tuple:
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().soma_oracle_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def u23(w: int) -> float:
    return float(lib().soma_oracle_u23(int(w) & 0xFFFFFFFF))


def metropolis(dE: float, u: float) -> bool:
    return bool(lib().soma_oracle_metropolis(C.c_float(dE), C.c_float(u)))


def set_num_threads(n: int) -> None:
    lib().soma_oracle_set_num_threads(int(n))


def num_threads() -> int:
    return int(lib().soma_oracle_num_threads())


@dataclass
class OracleSystem:
    """A melt of linear chains on a periodic collocation grid.

    ``specs`` is a list of ``(n_chains, types)``: ``types`` is the per-bead type id array of one
    chain of that architecture.  Positions are three float32 arrays (chain-major, unwrapped).
    """

    specs: Sequence[tuple]
    N_ref: int
    n_types: int
    box: Sequence[float]
    grid: Sequence[int]
    chiN: object = 0.0          # scalar (all pairs) or (n_types, n_types) array
    kappaN: float = 0.0
    A: float = 0.1
    seed: int = 0
    hamiltonian: int = 0
    smc_step: float = 0.0
    set_order: int = 0          # 0: even set then odd set; 1: random order per chain and sweep
    field_every: int = 1        # fields refreshed after every field_every-th sweep
    bonds: Optional[Sequence] = None   # per spec: None (linear chain) or an (n_bonds, 2) array of monomer pairs
    scheme: int = 0             # 0: independent sets (Code 2); 1: molecule-parallel random picks (Code 1)
    ext_field: Optional[np.ndarray] = None    # (n_types, n_cells) float32 static field added to omega
    forbidden: Optional[np.ndarray] = None    # (n_cells,) uint8, 1 = no particle may enter the cell
    spec_first_bead: Optional[Sequence[int]] = None   # this system is a part of a larger one: index in the whole system
    global_n_beads: int = 0                            # of each architecture's first bead; beads of the whole system
    _keep: list = field(default_factory=list, repr=False)

    def __post_init__(self):
        self._n_chains = np.array([int(s[0]) for s in self.specs], dtype=np.uint64)
        self._n_beads = np.array([len(s[1]) for s in self.specs], dtype=np.uint32)
        self._types = np.concatenate([np.asarray(s[1], dtype=np.uint8) for s in self.specs])
        assert int(self._types.max(initial=0)) < self.n_types <= MAX_TYPES
        self._sys = _System()
        self._refresh()

    def _refresh(self):
        s = self._sys
        s.n_specs = len(self.specs)
        s.spec_n_chains = self._n_chains.ctypes.data_as(C.POINTER(C.c_uint64))
        s.spec_n_beads = self._n_beads.ctypes.data_as(C.POINTER(C.c_uint32))
        s.types = self._types.ctypes.data_as(C.POINTER(C.c_uint8))
        s.n_types = self.n_types
        s.N_ref = self.N_ref
        for a in range(3):
            s.box[a] = float(self.box[a])
            s.grid[a] = int(self.grid[a])
        chi = np.zeros((MAX_TYPES, MAX_TYPES), dtype=np.float32)
        if np.isscalar(self.chiN):
            chi[: self.n_types, : self.n_types] = np.float32(self.chiN)
            np.fill_diagonal(chi, 0.0)
        else:
            m = np.asarray(self.chiN, dtype=np.float32)
            chi[: self.n_types, : self.n_types] = m
        for i, v in enumerate(chi.ravel()):
            s.chiN[i] = float(v)
        s.kappaN = float(self.kappaN)
        s.A = float(self.A)
        s.seed = int(self.seed)
        s.hamiltonian = int(self.hamiltonian)
        s.smc_step = float(self.smc_step)
        s.set_order = int(self.set_order)
        s.field_every = int(self.field_every)
        s.scheme = int(self.scheme)
        if self.bonds is not None:
            per = [np.zeros((0, 2), np.uint32) if b is None else np.ascontiguousarray(b, dtype=np.uint32).reshape(-1, 2)
                   for b in self.bonds]
            assert len(per) == len(self.specs)
            self._nbonds = np.array([len(b) for b in per], dtype=np.uint32)
            self._bonds = np.ascontiguousarray(np.concatenate(per).reshape(-1), dtype=np.uint32)
            if self._bonds.size == 0:
                self._bonds = np.zeros(2, np.uint32)
            s.spec_n_bonds = self._nbonds.ctypes.data_as(C.POINTER(C.c_uint32))
            s.bonds = self._bonds.ctypes.data_as(C.POINTER(C.c_uint32))
        else:
            s.spec_n_bonds = C.POINTER(C.c_uint32)()
            s.bonds = C.POINTER(C.c_uint32)()
        if self.ext_field is not None:
            self._ext = np.ascontiguousarray(self.ext_field, dtype=np.float32).reshape(self.n_types, -1)
            s.ext_field = self._ext.ctypes.data_as(C.POINTER(C.c_float))
        else:
            s.ext_field = C.POINTER(C.c_float)()
        if self.forbidden is not None:
            self._forb = np.ascontiguousarray(self.forbidden, dtype=np.uint8).reshape(-1)
            s.forbidden = self._forb.ctypes.data_as(C.POINTER(C.c_uint8))
        else:
            s.forbidden = C.POINTER(C.c_uint8)()
        if self.spec_first_bead is not None:
            self._first = np.ascontiguousarray(self.spec_first_bead, dtype=np.uint64)
            s.spec_first_bead = self._first.ctypes.data_as(C.POINTER(C.c_uint64))
        else:
            s.spec_first_bead = C.POINTER(C.c_uint64)()
        s.global_n_beads = int(self.global_n_beads)

    # -- sizes -------------------------------------------------------------------------------
    @property
    def ref(self):
        self._refresh()
        return C.byref(self._sys)

    @property
    def n_beads(self) -> int:
        return int(lib().soma_oracle_n_beads(self.ref))

    @property
    def n_cells(self) -> int:
        return int(self.grid[0]) * int(self.grid[1]) * int(self.grid[2])

    def bead_types(self) -> np.ndarray:
        """Type id of every bead, chain-major (for tests that recompute things by brute force)."""
        return np.concatenate([np.tile(np.asarray(t, dtype=np.uint8), int(n)) for n, t in self.specs])

    # -- steps of the path -------------------------------------------------------------------
    def cell_index(self, x: float, y: float, z: float) -> int:
        return int(lib().soma_oracle_cell_index(self.ref, C.c_float(x), C.c_float(y), C.c_float(z)))

    def histogram(self, x, y, z) -> np.ndarray:
        counts = np.zeros((self.n_types, self.n_cells), dtype=np.uint32)
        lib().soma_oracle_histogram(self.ref, _fp(x), _fp(y), _fp(z), _u32p(counts))
        return counts

    def fields(self, counts: np.ndarray) -> np.ndarray:
        counts = np.ascontiguousarray(counts, dtype=np.uint32)
        omega = np.zeros((self.n_types, self.n_cells), dtype=np.float32)
        lib().soma_oracle_fields(self.ref, _u32p(counts), _fp(omega))
        return omega

    def local_proposal(self, bead: int, sweep: int):
        d = np.zeros(3, dtype=np.float32)
        u = C.c_float()
        lib().soma_oracle_local_proposal(self.ref, bead, sweep, _fp(d), C.byref(u))
        return d, float(u.value)

    def local_delta_e(self, x, y, z, omega, bead: int, has_l: bool, has_r: bool, type_: int, d):
        d = np.ascontiguousarray(d, dtype=np.float32)
        eb, enb = C.c_float(), C.c_float()
        rn = np.zeros(3, dtype=np.float32)
        lib().soma_oracle_local_delta_e(self.ref, _fp(x), _fp(y), _fp(z), _fp(omega), bead,
                                        int(has_l), int(has_r), type_, _fp(d), C.byref(eb),
                                        C.byref(enb), _fp(rn))
        return float(eb.value), float(enb.value), rn

    def smc_proposal(self, bead: int, sweep: int):
        g = np.zeros(3, dtype=np.float32)
        u = C.c_float()
        lib().soma_oracle_smc_proposal(self.ref, bead, sweep, _fp(g), C.byref(u))
        return g, float(u.value)

    def smc_delta(self, x, y, z, omega, bead: int, has_l: bool, has_r: bool, type_: int, g):
        g = np.ascontiguousarray(g, dtype=np.float32)
        d = np.zeros(3, dtype=np.float32)
        rn = np.zeros(3, dtype=np.float32)
        dE, lr = C.c_float(), C.c_float()
        lib().soma_oracle_smc_delta(self.ref, _fp(x), _fp(y), _fp(z), _fp(omega), bead, int(has_l),
                                    int(has_r), type_, _fp(g), _fp(d), C.byref(dE), C.byref(lr), _fp(rn))
        return d, float(dE.value), float(lr.value), rn

    def first_set(self, first_bead: int, sweep: int) -> int:
        """Which set of the chain that starts at ``first_bead`` moves first in ``sweep`` (0 even, 1 odd)."""
        return int(lib().soma_oracle_first_set(self.ref, first_bead, sweep))

    def sweep(self, x, y, z, omega, sweep: int, move_kind: int = MOVE_LOCAL,
              decisions: Optional[np.ndarray] = None) -> int:
        """One MC sweep in place (omega frozen). Returns the number of accepted moves."""
        return int(lib().soma_oracle_sweep(self.ref, _fp(x), _fp(y), _fp(z), _fp(omega), sweep,
                                           move_kind, _u8p(decisions)))

    def sets(self, spec: int) -> np.ndarray:
        """Independent set of every monomer of architecture ``spec`` (greedy first fit, reading R25)."""
        out = np.zeros(len(self.specs[spec][1]), dtype=np.uint32)
        lib().soma_oracle_sets(self.ref, spec, _u32p(out))
        return out

    def pick(self, attempt_id: int, sweep: int, N: int) -> int:
        """Particle chosen by attempt ``attempt_id`` (= first bead + k) of a chain of N beads (Code 1)."""
        return int(lib().soma_oracle_pick(self.ref, attempt_id, sweep, N))

    def sweep_molecules(self, x, y, z, omega, sweep: int, move_kind: int = MOVE_LOCAL,
                        decisions: Optional[np.ndarray] = None) -> int:
        """One sweep of the molecule-parallel scheme (Code 1) in place. decisions: one byte per attempt."""
        return int(lib().soma_oracle_sweep_molecules(self.ref, _fp(x), _fp(y), _fp(z), _fp(omega), sweep,
                                                     move_kind, _u8p(decisions)))

    def step(self, x, y, z, counts, omega, sweep0: int, n_sweeps: int, move_kind: int = MOVE_LOCAL,
             decisions: Optional[np.ndarray] = None) -> int:
        """n_sweeps SCMF cycles in place: sweep, histogram, fields."""
        return int(lib().soma_oracle_step(self.ref, _fp(x), _fp(y), _fp(z), _u32p(counts), _fp(omega),
                                          sweep0, n_sweeps, move_kind, _u8p(decisions)))

    def init_positions(self):
        nb = self.n_beads
        x, y, z = (np.zeros(nb, dtype=np.float32) for _ in range(3))
        lib().soma_oracle_init_positions(self.ref, _fp(x), _fp(y), _fp(z))
        return x, y, z
