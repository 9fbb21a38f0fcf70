"""soma-b200: the SCMF Monte-Carlo step of SOMA (arXiv:1711.03828) as hand-written CUDA for sm_100a.

The product is the C-ABI library ``libsoma_b200.so`` (``include/soma_b200.h``); this package only
builds it (``_build``) and marshals arguments to it (``binding``).  No CPU fallback exists.
"""
from .binding import (DENSITY_FULL, DENSITY_INCREMENTAL, KERNEL_AUTO, KERNEL_FUSED, KERNEL_GENERIC,  # noqa: F401
                      K_COUNT, K_DENSITY, K_FIELD, K_LAYOUT, K_MOVE, OPT_LAYOUT, OPT_SORT_INTERVAL, OPT_SET_ORDER, OPT_FIELD_INTERVAL, OPT_SCHEME, OPT_PDL, MOVE_LOCAL, MOVE_SMC, OPT_DENSITY,
                      OPT_HAMILTONIAN, OPT_KERNEL, OPT_MOVE, OPT_RECORD_DECISIONS, OPT_SMC_STEP,
                      OPT_SWEEP_COUNTER, OPT_TIMING, OPT_COUNT_BITS, EOVERFLOW, SYMBOLS, Soma, SomaError, load, unpack_decisions,
                      STATIC_MAX_WORDS, STATIC_MAX_MONOMERS, fields_static)
from ._build import build  # noqa: F401


def from_workload(w, xyz0=None, stream=None) -> "Soma":
    """Create a system from a ``workloads.Workload`` description (marshalling only)."""
    bonds = getattr(w, "bonds", None) or [None] * len(w.specs)
    s = Soma([(n, t, b) for (n, t), b in zip(w.specs, bonds)], w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, w.A,
             w.seed, xyz0=xyz0, stream=stream)
    if getattr(w, "move", "local") == "smc":
        s.set_option(OPT_SMC_STEP, w.smc_step)
        s.set_option(OPT_MOVE, MOVE_SMC)
    return s
