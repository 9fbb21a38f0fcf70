"""No-GPU checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/soma_b200.h declares; argument validation works; there is no CPU fallback."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

import paper_1711_03828_b200 as P

ROOT = Path(__file__).resolve().parent.parent


def _declared_symbols():
    text = (ROOT / "include" / "soma_b200.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(soma_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = P.load()
    declared = _declared_symbols()
    assert len(declared) >= 15
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(P.SYMBOLS) == declared
    assert b"sm_100a" in lib.soma_version()


def test_kernels_are_compiled_for_sm_100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", str(P.build())], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, out


def _init(**kw):
    args = dict(specs=[(10, [0, 0, 1, 1])], N_ref=4, n_types=2, box=(2.0, 2.0, 2.0), grid=(4, 4, 4),
                chiN=10.0, kappaN=20.0, A=0.1, seed=1)
    args.update(kw)
    return P.Soma(**args)


@pytest.mark.parametrize("kw,needle", [
    (dict(n_types=0), "n_types"), (dict(n_types=9), "n_types"), (dict(N_ref=0), "N_ref"),
    (dict(box=(0.0, 1.0, 1.0)), "box"), (dict(grid=(0, 4, 4)), "grid"), (dict(A=0.0), "A"),
    (dict(A=1.5), "A"), (dict(specs=[(10, [0, 2])]), "type"), (dict(grid=(2048, 2048, 2048)), "cells"),
    (dict(specs=[(2**31, [0, 0, 0, 0])]), "2^32"),
])
def test_argument_validation(kw, needle):
    with pytest.raises(P.SomaError) as e:
        _init(**kw)
    assert e.value.code == -1 and needle in str(e.value)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(P.SomaError) as e:
        _init()
    assert e.value.code == -5 and "no CPU path" in str(e.value)


def test_product_does_not_import_the_oracle():
    for p in (ROOT / "paper_1711_03828_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h"):
            assert "oracle" not in p.read_text().replace("no CPU path", ""), p
    assert "paper_1711_03828_b200" not in (ROOT / "oracle" / "__init__.py").read_text().replace(
        "``paper_1711_03828_b200/``", "")
    assert "csrc" not in (ROOT / "oracle" / "soma_oracle.c").read_text().replace(
        "paper_1711_03828_b200/csrc/", "")
