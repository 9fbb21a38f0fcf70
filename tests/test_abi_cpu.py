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


def _decode_fig2(words):
    """Walk the architecture array as the kernels do: (types, neighbour lists, set of every monomer, number of sets)."""
    N = int(words[0])
    types, nbrs, n_bond_words = [], [], 0
    for j in range(N):
        w = int(words[1 + j])
        types.append(w & 0xFF)
        at, mine = w >> 8, []
        while at:
            b = int(words[at])
            off = (b >> 5) - (1 << 27 if b >> 31 else 0)            # signed 27 bits
            assert (b >> 1) & 0xF == 0                              # bond type: harmonic
            mine.append(j + off)
            n_bond_words += 1
            at = 0 if b & 1 else at + 1
        nbrs.append(mine)
    members = words[1 + N + n_bond_words: 1 + 2 * N + n_bond_words]
    rest = words[1 + 2 * N + n_bond_words:]
    n_sets = (len(rest) - 1) // 2
    set_off, magic = rest[:n_sets + 1], rest[n_sets + 1:]
    set_of = {}
    for c in range(n_sets):
        size = int(set_off[c + 1] - set_off[c])
        assert int(magic[c]) == ((1 << 32) // size + 1) % (1 << 32)
        for j in members[set_off[c]:set_off[c + 1]]:
            set_of[int(j)] = c
    return types, nbrs, [set_of[j] for j in range(N)], n_sets


def test_architecture_words_are_the_layout_of_fig_2_and_the_sets_of_the_oracle():
    """Host logic, no GPU: the array soma_init hands to the general-architecture kernels (Fig. 2)
    decodes to the bond list it was built from -- partners in ascending order, the last-bond bit on the last one, a
    monomer without bonds marked by offset 0 -- and its independent sets are the oracle's (greedy first fit, R25)."""
    import oracle
    star = [(0, 1 + a * 4) for a in range(3)] + [(1 + a * 4 + k, 2 + a * 4 + k) for a in range(3) for k in range(3)]
    ring5 = [(0, 1), (1, 2), (2, 3), (3, 4), (4, 0)]
    comb = [(j, j + 1) for j in range(5)] + [(1, 6), (3, 7), (4, 8), (8, 9)]
    lonely = [(0, 1), (3, 2)]                                      # monomer 4 has no bond at all
    cases = [(star, 13), (ring5, 5), (comb, 10), (lonely, 5), ([(j + 1, j) for j in range(6)][::-1], 7)]
    orc = oracle.OracleSystem(specs=[(1, np.zeros(N, np.uint8)) for _, N in cases], N_ref=8, n_types=1, box=(1.0,) * 3,
                              grid=(2, 2, 2), bonds=[np.array(b, np.uint32) for b, _ in cases])
    for spec, (bonds, N) in enumerate(cases):
        types = [(3 * j + 1) % 7 for j in range(N)]
        words, n_sets = P.binding.architecture_words(types, bonds)
        got_types, nbrs, set_of, n_sets_decoded = _decode_fig2(words)
        assert int(words[0]) == N and got_types == types and n_sets == n_sets_decoded
        want = [[] for _ in range(N)]
        for i, j in bonds:
            want[i].append(j); want[j].append(i)
        assert nbrs == [sorted(v) for v in want]
        assert set_of == [int(v) for v in orc.sets(spec)]
        assert n_sets == max(set_of) + 1
    with pytest.raises(P.SomaError):
        P.binding.architecture_words([0, 0, 0], [(0, 3)])          # bond to a monomer that is not there
    with pytest.raises(P.SomaError):
        P.binding.architecture_words([0, 0, 0], [(0, 1), (1, 0)])  # the same bond twice
