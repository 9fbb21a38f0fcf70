"""Thin ctypes binding of libsoma_b200.so (include/soma_b200.h) -- argument marshalling only.

Every step of the SCMF cycle runs in the CUDA kernels behind the C ABI; nothing here computes.
There is no CPU fallback: loading fails loudly if the library cannot be built or found, and
``soma_init`` fails with SOMA_ENODEVICE when no sm_100 device is present.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence, Tuple

import numpy as np

from . import _build

OK = 0
OPT_HAMILTONIAN, OPT_MOVE, OPT_SMC_STEP, OPT_RECORD_DECISIONS = 1, 2, 3, 4
OPT_KERNEL, OPT_DENSITY, OPT_TIMING, OPT_SWEEP_COUNTER = 5, 6, 7, 8
OPT_LAYOUT, OPT_SORT_INTERVAL, OPT_SET_ORDER, OPT_FIELD_INTERVAL, OPT_SCHEME, OPT_PDL = 11, 12, 13, 14, 15, 16
OPT_COUNT_BITS = 17
EOVERFLOW = -7
MOVE_LOCAL, MOVE_SMC = 1, 2
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_FUSED = 0, 1, 2
DENSITY_INCREMENTAL, DENSITY_FULL = 0, 1
K_MOVE, K_DENSITY, K_FIELD, K_LAYOUT, K_COUNT = 0, 1, 2, 3, 4

# every symbol include/soma_b200.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "soma_init", "soma_step", "soma_fields", "soma_positions", "soma_set_positions", "soma_set_chi",
    "soma_set_external", "soma_set_option", "soma_stats", "soma_decisions", "soma_kernel_times", "soma_launch_count",
    "soma_n_beads", "soma_n_cells", "soma_n_types", "soma_sync", "soma_destroy", "soma_last_error",
    "soma_version", "soma_init_shard", "soma_shard_moves", "soma_shard_fields", "soma_shard_exchange",
    "soma_shard_exchange_copy", "soma_shard_peer_handle", "soma_shard_set_peers", "soma_architecture_words",
    "soma_fields_static",
)
STATIC_MAX_WORDS, STATIC_MAX_MONOMERS = 1 << 20, 256


class SomaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"soma error {code}: {msg}")
        self.code = code


class _ChainSpec(C.Structure):
    _fields_ = [("n_chains", C.c_uint64), ("n_beads", C.c_uint32), ("types", C.POINTER(C.c_uint8)),
                ("n_bonds", C.c_uint32), ("bonds", C.POINTER(C.c_uint32))]


_lib = None


def load() -> C.CDLL:
    """Build (if stale) and load the CUDA library. Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(str(path))
    vp, i32, u64 = C.c_void_p, C.c_int, C.c_uint64
    L.soma_init.argtypes = [C.POINTER(vp), C.POINTER(_ChainSpec), i32, i32, i32, C.POINTER(C.c_float),
                            C.POINTER(C.c_int), C.c_float, C.c_float, C.c_float, u64, vp, vp]
    L.soma_init_shard.argtypes = L.soma_init.argtypes + [C.POINTER(u64), u64]
    L.soma_shard_moves.argtypes = [vp]
    L.soma_shard_fields.argtypes = [vp, i32]
    L.soma_shard_exchange.argtypes = [vp, C.POINTER(vp), C.POINTER(u64)]
    L.soma_shard_exchange_copy.argtypes = [vp, vp, i32]
    L.soma_architecture_words.argtypes = [C.POINTER(_ChainSpec), vp, u64, C.POINTER(u64), C.POINTER(C.c_uint32)]
    L.soma_shard_peer_handle.argtypes = [vp, vp]
    L.soma_shard_set_peers.argtypes = [vp, i32, i32, C.POINTER(vp), vp]
    L.soma_step.argtypes = [vp, i32]
    L.soma_fields.argtypes = [vp, vp, vp, i32]
    L.soma_positions.argtypes = [vp, vp, i32]
    L.soma_set_positions.argtypes = [vp, vp, i32]
    L.soma_set_chi.argtypes = [vp, i32, i32, C.c_float]
    L.soma_set_external.argtypes = [vp, vp, vp, i32]
    L.soma_set_option.argtypes = [vp, i32, C.c_double]
    L.soma_stats.argtypes = [vp, C.POINTER(u64), C.POINTER(u64), C.POINTER(u64)]
    L.soma_decisions.argtypes = [vp, vp, i32]
    L.soma_kernel_times.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(u64)]
    L.soma_launch_count.argtypes = [vp]
    L.soma_launch_count.restype = u64
    L.soma_n_beads.argtypes = [vp]
    L.soma_n_beads.restype = u64
    L.soma_n_cells.argtypes = [vp]
    L.soma_n_cells.restype = u64
    L.soma_n_types.argtypes = [vp]
    L.soma_sync.argtypes = [vp]
    L.soma_destroy.argtypes = [vp]
    L.soma_destroy.restype = None
    L.soma_last_error.restype = C.c_char_p
    L.soma_version.restype = C.c_char_p
    L.soma_fields_static.argtypes = [C.POINTER(_ChainSpec), i32, i32, i32, C.POINTER(C.c_float), C.POINTER(C.c_int),
                                     C.c_float, C.c_float, i32, vp, vp, vp, vp]
    _lib = L
    return L


def _check(rc: int) -> None:
    if rc != OK:
        raise SomaError(rc, load().soma_last_error().decode())


def _ptr(buf) -> Tuple[int, bool]:
    """(address, is_device) of a numpy array or a torch tensor."""
    if isinstance(buf, np.ndarray):
        assert buf.flags.c_contiguous
        return buf.ctypes.data, False
    import torch  # torch is plumbing here: device memory and streams
    assert isinstance(buf, torch.Tensor) and buf.is_contiguous()
    return buf.data_ptr(), buf.is_cuda


def architecture_words(types: Sequence[int], bonds: Sequence[Tuple[int, int]]) -> Tuple[np.ndarray, int]:
    """(the Fig. 2 architecture array of a molecule type given by its bond list, number of independent sets): host only."""
    L = load()
    t = np.ascontiguousarray(types, np.uint8)
    b = np.ascontiguousarray(bonds, np.uint32).reshape(-1, 2)
    spec = _ChainSpec(1, len(t), t.ctypes.data_as(C.POINTER(C.c_uint8)), len(b), b.ctypes.data_as(C.POINTER(C.c_uint32)))
    n, n_sets = C.c_uint64(), C.c_uint32()
    _check(L.soma_architecture_words(C.byref(spec), None, 0, C.byref(n), C.byref(n_sets)))
    out = np.empty(n.value, np.uint32)
    _check(L.soma_architecture_words(C.byref(spec), C.c_void_p(out.ctypes.data), n.value, C.byref(n), C.byref(n_sets)))
    return out, int(n_sets.value)


def fields_static(specs: Sequence[Tuple[int, Sequence[int]]], N_ref: int, n_types: int, box: Sequence[float],
                  grid: Sequence[int], chiN: float, kappaN: float, xyz, omega, counts=None, hamiltonian: int = 0,
                  stream: Optional[int] = None) -> None:
    """soma_fields_static: omega (and counts) of the positions in the CUDA tensor `xyz`, written into the CUDA
    tensors `omega` / `counts` the caller brings.  For callers that must not allocate device memory (a host
    program whose allocator owns the GPU, a tool beside simulations that fill it): nothing is allocated, the
    occupation numbers live in the library's static array (n_types * cells <= STATIC_MAX_WORDS).  Calls that
    overlap on one GPU race on that array.  Synchronises `stream`."""
    L = load()
    keep = [np.ascontiguousarray(sp[1], dtype=np.uint8) for sp in specs]
    arr = (_ChainSpec * len(specs))()
    for i, (sp, t) in enumerate(zip(specs, keep)):
        arr[i].n_chains = int(sp[0])
        arr[i].n_beads = len(t)
        arr[i].types = t.ctypes.data_as(C.POINTER(C.c_uint8))
        arr[i].n_bonds = 0
        arr[i].bonds = C.POINTER(C.c_uint32)()
    cbox = (C.c_float * 3)(*[float(v) for v in box])
    cgrid = (C.c_int * 3)(*[int(v) for v in grid])
    if stream is None:
        try:
            import torch
            stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        except Exception:
            stream = 0
    px = _ptr(xyz)[0] if xyz is not None else None
    po = _ptr(omega)[0] if omega is not None else None
    pc = _ptr(counts)[0] if counts is not None else None
    _check(L.soma_fields_static(arr, len(specs), int(N_ref), int(n_types), cbox, cgrid, C.c_float(chiN),
                                C.c_float(kappaN), int(hamiltonian), C.c_void_p(px), C.c_void_p(po), C.c_void_p(pc),
                                C.c_void_p(stream or None)))


class Soma:
    """One SCMF system on the current CUDA device. Method names mirror the C ABI."""

    def __init__(self, specs: Sequence[Tuple[int, Sequence[int]]], N_ref: int, n_types: int,
                 box: Sequence[float], grid: Sequence[int], chiN: float, kappaN: float, A: float,
                 seed: int, xyz0: Optional[np.ndarray] = None, stream: Optional[int] = None,
                 spec_first_bead: Optional[Sequence[int]] = None, global_n_beads: int = 0):
        L = load()
        self._L = L
        self._h = C.c_void_p()
        # a spec is (n_chains, types) for a linear chain or (n_chains, types, bonds) with an (n_bonds, 2) bond list
        keep = [np.ascontiguousarray(sp[1], dtype=np.uint8) for sp in specs]
        keep_b = [np.ascontiguousarray(sp[2], dtype=np.uint32).reshape(-1, 2) if len(sp) > 2 and sp[2] is not None
                  else None for sp in specs]
        arr = (_ChainSpec * len(specs))()
        for i, (sp, t, bd) in enumerate(zip(specs, keep, keep_b)):
            arr[i].n_chains = int(sp[0])
            arr[i].n_beads = len(t)
            arr[i].types = t.ctypes.data_as(C.POINTER(C.c_uint8))
            arr[i].n_bonds = 0 if bd is None else len(bd)
            arr[i].bonds = C.POINTER(C.c_uint32)() if bd is None else bd.ctypes.data_as(C.POINTER(C.c_uint32))
        cbox = (C.c_float * 3)(*[float(v) for v in box])
        cgrid = (C.c_int * 3)(*[int(v) for v in grid])
        if stream is None:
            try:
                import torch
                stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
            except Exception:
                stream = 0
        p0 = None
        if xyz0 is not None:
            xyz0 = np.ascontiguousarray(xyz0, dtype=np.float32)
            p0 = xyz0.ctypes.data
        args = (C.byref(self._h), arr, len(specs), int(N_ref), int(n_types), cbox, cgrid, C.c_float(chiN),
                C.c_float(kappaN), C.c_float(A), C.c_uint64(int(seed)), C.c_void_p(p0), C.c_void_p(stream or None))
        if spec_first_bead is None:
            _check(L.soma_init(*args))
        else:   # this rank's molecules of a system spread over several GPUs (soma_init_shard)
            first = (C.c_uint64 * len(specs))(*[int(v) for v in spec_first_bead])
            _check(L.soma_init_shard(*args, first, C.c_uint64(int(global_n_beads))))
        self.n_beads_global = int(global_n_beads) if spec_first_bead is not None else None
        self.n_beads = int(L.soma_n_beads(self._h))
        self.n_cells = int(L.soma_n_cells(self._h))
        self.n_types = int(L.soma_n_types(self._h))

    # -- the C ABI, one method per entry point -------------------------------------------------
    def step(self, n_sweeps: int = 1) -> None:
        _check(self._L.soma_step(self._h, int(n_sweeps)))

    def shard_moves(self) -> None:
        _check(self._L.soma_shard_moves(self._h))

    def shard_fields(self, advance: bool = True) -> None:
        _check(self._L.soma_shard_fields(self._h, int(bool(advance))))

    def shard_exchange(self) -> Tuple[int, int]:
        """(device address, uint32 words) of the exchange array of a shard."""
        p, n = C.c_void_p(), C.c_uint64()
        _check(self._L.soma_shard_exchange(self._h, C.byref(p), C.byref(n)))
        return int(p.value), int(n.value)

    def shard_peer_handle(self) -> bytes:
        """CUDA IPC handle (64 bytes) of this rank's exchange allocation."""
        buf = C.create_string_buffer(64)
        _check(self._L.soma_shard_peer_handle(self._h, buf))
        return buf.raw

    def shard_set_peers(self, n_ranks: int, my_rank: int, peer_addresses=None, handles=None) -> None:
        """peer_addresses: per rank a device address (same process) or None; handles: per rank 64 bytes or None."""
        addr = (C.c_void_p * n_ranks)(*[C.c_void_p(a) if a else C.c_void_p(None) for a in (peer_addresses or [None] * n_ranks)])
        blob = None
        if handles is not None:
            blob = C.create_string_buffer(b"".join(h if h is not None else bytes(64) for h in handles), 64 * n_ranks)
        _check(self._L.soma_shard_set_peers(self._h, n_ranks, my_rank, addr, blob))

    def shard_exchange_tensor(self):
        """The exchange array as a torch int32 tensor on the device (no copy): what the all-reduce runs on."""
        import torch
        addr, n = self.shard_exchange()

        class _View:                                   # the CUDA array interface is all torch needs to wrap the memory
            __cuda_array_interface__ = {"shape": (n,), "typestr": "<i4", "data": (addr, False), "version": 3, "strides": None}

        return torch.as_tensor(_View(), device="cuda")

    def shard_exchange_get(self) -> np.ndarray:
        out = np.empty(self.shard_exchange()[1], np.uint32)
        _check(self._L.soma_shard_exchange_copy(self._h, C.c_void_p(out.ctypes.data), 1))
        return out

    def shard_exchange_put(self, words: np.ndarray) -> None:
        words = np.ascontiguousarray(words, np.uint32)
        assert words.size == self.shard_exchange()[1]
        _check(self._L.soma_shard_exchange_copy(self._h, C.c_void_p(words.ctypes.data), 0))

    def fields(self, omega=None, counts=None):
        """Copy omega (and counts) out. With no arguments returns new host numpy arrays."""
        if omega is None and counts is None:
            omega = np.empty((self.n_types, self.n_cells), np.float32)
            counts = np.empty((self.n_types, self.n_cells), np.uint32)
        po, do = _ptr(omega) if omega is not None else (None, None)
        pc, dc = _ptr(counts) if counts is not None else (None, None)
        dev = do if do is not None else dc
        assert dc is None or do is None or dc == do
        _check(self._L.soma_fields(self._h, C.c_void_p(po), C.c_void_p(pc), int(bool(dev))))
        return omega, counts

    def positions(self, xyz=None):
        if xyz is None:
            xyz = np.empty((3, self.n_beads), np.float32)
        p, dev = _ptr(xyz)
        _check(self._L.soma_positions(self._h, C.c_void_p(p), int(dev)))
        return xyz

    def set_positions(self, xyz) -> None:
        p, dev = _ptr(xyz)
        _check(self._L.soma_set_positions(self._h, C.c_void_p(p), int(dev)))

    def set_chi(self, i: int, j: int, chiN: float) -> None:
        _check(self._L.soma_set_chi(self._h, i, j, C.c_float(chiN)))

    def set_external(self, ext_field=None, forbidden=None) -> None:
        """ext_field: float32 (n_types, n_cells) or None; forbidden: uint8 (n_cells,) or None."""
        pe, de = _ptr(ext_field) if ext_field is not None else (None, None)
        pf, df = _ptr(forbidden) if forbidden is not None else (None, None)
        assert de is None or df is None or de == df
        dev = de if de is not None else df
        _check(self._L.soma_set_external(self._h, C.c_void_p(pe), C.c_void_p(pf), int(bool(dev))))

    def set_option(self, key: int, value: float) -> None:
        _check(self._L.soma_set_option(self._h, int(key), C.c_double(value)))

    def stats(self) -> Tuple[int, int, int]:
        a, b, c = C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(self._L.soma_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return int(a.value), int(b.value), int(c.value)

    def decisions(self, bits=None):
        if bits is None:
            bits = np.empty(((self.n_beads_global or self.n_beads) + 31) // 32, np.uint32)
        p, dev = _ptr(bits)
        _check(self._L.soma_decisions(self._h, C.c_void_p(p), int(dev)))
        return bits

    def kernel_times(self):
        ms = (C.c_double * K_COUNT)()
        n = (C.c_uint64 * K_COUNT)()
        _check(self._L.soma_kernel_times(self._h, ms, n))
        return [float(v) for v in ms], [int(v) for v in n]

    def launch_count(self) -> int:
        return int(self._L.soma_launch_count(self._h))

    def sync(self) -> None:
        _check(self._L.soma_sync(self._h))

    def destroy(self) -> None:
        if self._h:
            self._L.soma_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def unpack_decisions(bits: np.ndarray, n_beads: int) -> np.ndarray:
    """Bitmap words -> one uint8 per bead (marshalling helper for tests)."""
    return np.unpackbits(bits.view(np.uint8), bitorder="little")[:n_beads]
