"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Every expected value here comes from a closed form, a brute-force recomputation in float64 written
from a *different* formula than the oracle uses, a published known-answer vector, or a library
routine (cuRAND's host Philox generator).  Nothing is taken from the oracle itself or from the
CUDA path.  Citations are PAPER.md line numbers (arXiv:1711.03828).
"""
from __future__ import annotations

import ctypes as C
import math
from pathlib import Path

import numpy as np
import pytest

import oracle
from oracle import MOVE_LOCAL, MOVE_SMC, OracleSystem

GOLDEN = Path(__file__).resolve().parent / "golden"


# ----------------------------------------------------------------------------------------------
# P1  Philox4x32-10
# ----------------------------------------------------------------------------------------------
def test_philox_known_answer_vectors():
    rows = [l.split() for l in (GOLDEN / "philox4x32_10_kat.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def _curand_host(seed: int, offset: int, n_words: int) -> np.ndarray:
    try:
        L = C.CDLL("libcurand.so")
    except OSError:
        try:
            L = C.CDLL("/usr/local/cuda/lib64/libcurand.so")
        except OSError:
            pytest.skip("libcurand not available")
    gen = C.c_void_p()
    if L.curandCreateGeneratorHost(C.byref(gen), 161) != 0:  # CURAND_RNG_PSEUDO_PHILOX4_32_10
        pytest.skip("cuRAND host generator unavailable")
    assert L.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    assert L.curandSetGeneratorOffset(gen, C.c_ulonglong(offset)) == 0
    out = np.zeros(n_words, dtype=np.uint32)
    assert L.curandGenerate(gen, out.ctypes.data_as(C.POINTER(C.c_uint32)), C.c_size_t(n_words)) == 0
    L.curandDestroyGenerator(gen)
    return out.reshape(-1, 4)


@pytest.mark.parametrize("seed,offset", [(0, 0), (0x0123456789ABCDEF, 0), (42, 4 * 65536 * 12345),
                                         (7, 4 * 65536 * (2**32 + 99)), (2**64 - 1, 4 * 65536 * (2**45 + 3))])
def test_philox_matches_curand_host_generator(seed, offset):
    """cuRAND's host generator emits, with the default ordering, block p (4 words) =
    Philox4x32-10(counter = (p // 65536 as 64 bit, p % 65536, 0), key = seed); offset o starts at
    block o / 4.  An independent implementation of the same generator (library routine)."""
    n_blocks = 65536 + 300   # crosses one subsequence wrap so that ctr[0] changes too
    got = _curand_host(seed, offset, 4 * n_blocks)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    rng = np.random.default_rng(1)
    for b in list(range(0, 40)) + list(rng.integers(0, n_blocks, 200)) + [65535, 65536, 65537, n_blocks - 1]:
        p = offset // 4 + int(b)
        hi, sub = divmod(p, 65536)
        ctr = [hi & 0xFFFFFFFF, (hi >> 32) & 0xFFFFFFFF, sub, 0]
        assert oracle.philox4x32_10(ctr, key) == tuple(int(v) for v in got[int(b)])


# ----------------------------------------------------------------------------------------------
# P2  bits -> trial displacement / acceptance uniform
# ----------------------------------------------------------------------------------------------
def _free_beads(n, A=0.1, seed=5, **kw):
    return OracleSystem(specs=[(n, np.zeros(1, np.uint8))], N_ref=1, n_types=1, box=(4.0, 4.0, 4.0),
                        grid=(4, 4, 4), chiN=0.0, kappaN=0.0, A=A, seed=seed, **kw)


def test_u23_is_exact_mantissa_fill():
    for w in [0, 1, 511, 512, 0x80000000, 0xFFFFFFFF, 0x12345678]:
        assert oracle.u23(w) == 1.0 + (w >> 9) * 2.0**-23


def test_local_proposal_values_and_moments():
    A = 0.1
    s = _free_beads(1, A=A)
    key = [s.seed & 0xFFFFFFFF, s.seed >> 32]
    ds, us = [], []
    for bead in range(4000):
        sweep = (bead * 7919) % 13 + (1 << 33) * (bead % 3)
        d, u = s.local_proposal(bead, sweep)
        # the counter layout (bead, sweep lo, sweep hi, kind 1 << 8 | sub 0) and the word -> number map
        w = oracle.philox4x32_10([bead, sweep & 0xFFFFFFFF, sweep >> 32, 0x100], key)
        k = [v >> 9 for v in w]
        A32 = float(np.float32(A))
        for a in range(3):
            exact = A32 * ((2 * k[a] + 1) * 2.0**-23 - 1.0)
            # one fmaf(U23, 2A, fl32(A (2^-23 - 3))): error <= half an ulp of the constant 3A
            # plus half an ulp of the result
            assert abs(float(d[a]) - exact) <= 2.0**-24 * (3 * A32) * 1.34 + 2.0**-24 * A32
            assert -A32 < float(d[a]) < A32
        assert u == k[3] * 2.0**-23 and 0.0 <= u < 1.0
        ds.append(d)
        us.append(u)
    ds = np.asarray(ds, dtype=np.float64).ravel()
    n = ds.size
    assert abs(ds.mean()) < 4 * A / math.sqrt(3 * n)                      # <d> = 0
    assert abs(ds.var() - A * A / 3) < 4 * (A * A) * math.sqrt(4 / 45 / n)  # Var d = A^2/3
    us = np.asarray(us)
    assert abs(us.mean() - 0.5) < 4 / math.sqrt(12 * us.size)


def test_free_beads_all_moves_accepted_and_diffuse():
    """N = 1 'chains', chi = kappa = 0: Delta E = 0, every move is accepted, <|dr|^2> = A^2 per sweep."""
    n, A = 20000, 0.1
    s = _free_beads(n, A=A)
    rng = np.random.default_rng(0)
    x, y, z = (rng.random(n).astype(np.float32) * 4 for _ in range(3))
    x0, y0, z0 = x.copy(), y.copy(), z.copy()
    omega = np.zeros((1, s.n_cells), np.float32)
    dec = np.zeros(n, np.uint8)
    acc = s.sweep(x, y, z, omega, 3, MOVE_LOCAL, dec)
    assert acc == n and dec.all()
    dr2 = ((x - x0).astype(np.float64) ** 2 + (y - y0).astype(np.float64) ** 2 + (z - z0).astype(np.float64) ** 2)
    # Var(|d|^2) = 3 * (A^4/5 - A^4/9) = 4 A^4 / 15
    assert abs(dr2.mean() - A * A) < 4 * math.sqrt(4 * A**4 / 15 / n)


# ----------------------------------------------------------------------------------------------
# P3  incremental Delta E vs brute-force total Hamiltonian (Eq. 1-2, Eq. 13 :194)
# ----------------------------------------------------------------------------------------------
def _cell_f64(pos, box, grid):
    """Characteristic-function cell of Eq. 4 evaluated in float64 from the wrapped coordinate."""
    idx = []
    for a in range(3):
        w = math.fmod(pos[a], box[a])
        if w < 0:
            w += box[a]
        idx.append(min(int(w / (box[a] / grid[a])), grid[a] - 1))
    return (idx[0] * grid[1] + idx[1]) * grid[2] + idx[2]


def _total_H(pos, chains, types, omega, k0, box, grid):
    """H_b + H_nb^SCMF in float64: sum over bonds k0/2 r^2 + sum over beads omega_type(cell)."""
    H = 0.0
    for first, N in chains:
        for j in range(N):
            g = first + j
            if j + 1 < N:
                b = pos[g + 1] - pos[g]
                H += 0.5 * k0 * float(b @ b)
            H += float(omega[types[g], _cell_f64(pos[g], box, grid)])
    return H


def _tiny_system(seed, specs, N_ref, box, grid, A=0.1, **kw):  # kw: set_order, bonds, ...
    s = OracleSystem(specs=specs, N_ref=N_ref, n_types=2, box=box, grid=grid, chiN=0.0, kappaN=0.0,
                     A=A, seed=seed, **kw)
    rng = np.random.default_rng(seed)
    chains, g = [], 0
    pos = []
    for n, t in specs:
        for _ in range(n):
            p = rng.random(3) * np.asarray(box) + rng.integers(-2, 3, 3) * np.asarray(box)  # unwrapped
            for j in range(len(t)):
                pos.append(p.copy())
                p = p + rng.normal(0, 1 / math.sqrt(3 * max(N_ref - 1, 1)), 3)
            chains.append((g, len(t)))
            g += len(t)
    pos = np.asarray(pos, dtype=np.float32)
    omega = rng.normal(0, 1.0, (2, s.n_cells)).astype(np.float32)
    return s, chains, pos, omega


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_incremental_delta_e_matches_brute_force(seed):
    specs = [(2, np.array([0, 0, 1, 1], np.uint8)), (1, np.array([1, 0, 1], np.uint8)), (2, np.array([0], np.uint8))]
    box, grid = (1.5, 1.0, 2.0), (3, 2, 4)
    s, chains, pos, omega = _tiny_system(seed, specs, 4, box, grid, A=0.4)
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
    checked_nb = 0
    for first, N in chains:
        for j in range(N):
            g = first + j
            for sweep in range(6):
                d, _ = s.local_proposal(g, sweep)
                eb, enb, rn = s.local_delta_e(x, y, z, omega, g, j > 0, j + 1 < N, int(types[g]), d)
                assert np.array_equal(rn, pos[g] + d)            # r' = fl32(r + d), one IEEE add
                p64 = pos.astype(np.float64)
                H0 = _total_H(p64, chains, types, omega, k0, box, grid)
                p64[g] = rn.astype(np.float64)
                H1 = _total_H(p64, chains, types, omega, k0, box, grid)
                dE = H1 - H0
                assert abs((eb + enb) - dE) <= 2e-5 * (1 + abs(dE)), (g, sweep, eb, enb, dE)
                checked_nb += enb != 0.0
    assert checked_nb > 10   # the field term was exercised


def test_sweep_is_even_then_odd_with_frozen_field():
    """Replay one oracle sweep move by move with float64 brute-force energies: same decisions, same
    positions -- pins the set order of Code 2 / Fig. 1: odd beads see the
    already-moved even beads, even beads see the old odd beads."""
    specs = [(3, np.array([0, 0, 1, 1, 1], np.uint8)), (2, np.array([0, 1] * 4, np.uint8))]
    box, grid = (2.0, 2.0, 2.0), (4, 4, 4)
    s, chains, pos, omega = _tiny_system(11, specs, 8, box, grid, A=0.3)
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    for sweep in range(5):
        x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
        dec = np.zeros(len(pos), np.uint8)
        acc = s.sweep(x, y, z, omega, sweep, MOVE_LOCAL, dec)
        ref = pos.copy()
        ref_dec = np.zeros(len(pos), np.uint8)
        fragile = False
        for parity in (0, 1):
            for first, N in chains:
                for j in range(parity, N, 2):
                    g = first + j
                    d, u = s.local_proposal(g, sweep)
                    rn = ref[g] + d
                    p64 = ref.astype(np.float64)
                    H0 = _total_H(p64, chains, types, omega, k0, box, grid)
                    p64[g] = rn
                    dE = _total_H(p64, chains, types, omega, k0, box, grid) - H0
                    thr = math.exp(-dE) if dE > 0 else 2.0
                    if abs(u - thr) < 1e-5 or abs(dE) < 1e-6:
                        fragile = True      # decision within rounding of the threshold: skip sweep
                    if dE <= 0 or u < thr:
                        ref[g] = rn
                        ref_dec[g] = 1
        if not fragile:
            assert np.array_equal(dec, ref_dec)
            assert acc == int(ref_dec.sum())
            assert np.array_equal(np.stack([x, y, z], 1), ref)
        pos = np.stack([x, y, z], 1)


# ----------------------------------------------------------------------------------------------
# P4  Metropolis rule and detailed balance of the bonded part
# ----------------------------------------------------------------------------------------------
def test_metropolis_rule_exact_ratio():
    """acc(dE)/acc(-dE) = exp(-dE): downhill always, uphill iff u < exp(-dE)."""
    for dE in [-3.0, -1e-9, 0.0]:
        for u in [0.0, 0.5, 1 - 2.0**-23]:
            assert oracle.metropolis(dE, u)
    for dE in [1e-3, 0.1, 0.7, 2.0, 9.0]:
        p = math.exp(-dE)
        k = math.floor(p * 2**23)
        # u = j 2^-23 is accepted for j < p 2^23 and rejected above (2 grid points of slack for expf)
        assert oracle.metropolis(dE, max(k - 2, 0) * 2.0**-23)
        assert not oracle.metropolis(dE, min(k + 2, 2**23 - 1) * 2.0**-23) or p > 1 - 2.0**-21
    assert not oracle.metropolis(100.0, 2.0**-23)


def test_two_bead_chains_relax_to_gaussian_bonds():
    """One bond, chi = kappa = 0: stationary bond components ~ N(0, 1/k0), from a collapsed start."""
    n, N_ref = 40000, 2                       # k0 = 3 (N_ref - 1) = 3
    s = OracleSystem(specs=[(n, np.zeros(2, np.uint8))], N_ref=N_ref, n_types=1, box=(4.0,) * 3,
                     grid=(2, 2, 2), chiN=0.0, kappaN=0.0, A=0.6, seed=17)
    x, y, z = (np.full(2 * n, 2.0, np.float32) for _ in range(3))     # all bonds of length zero
    omega = np.zeros((1, 8), np.float32)
    for sweep in range(120):
        s.sweep(x, y, z, omega, sweep)
    k0 = 3.0
    for a in (x, y, z):
        b = (a[1::2] - a[0::2]).astype(np.float64)
        assert abs(b.mean()) < 5 * math.sqrt(1 / k0 / n)
        assert abs(b.var() - 1 / k0) < 5 * (1 / k0) * math.sqrt(2 / n)
        assert abs((b**4).mean() / b.var() ** 2 - 3.0) < 5 * math.sqrt(96 / n)      # Gaussian kurtosis
    b2 = sum(((a[1::2] - a[0::2]).astype(np.float64)) ** 2 for a in (x, y, z))
    # |b| Maxwell: <b^4>/<b^2>^2 = 5/3
    assert abs((b2**2).mean() / b2.mean() ** 2 - 5 / 3) < 0.03


# ----------------------------------------------------------------------------------------------
# P5  detailed balance of the field part: Boltzmann occupation of a static two-level field
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("move,kw", [(MOVE_LOCAL, {}), (MOVE_SMC, {"smc_step": 0.01})])
def test_free_beads_in_static_field_are_boltzmann_distributed(move, kw):
    n, dw = 60000, 0.8
    s = _free_beads(n, A=0.35, seed=23, **kw)
    s.box, s.grid = (2.0, 1.0, 1.0), (2, 1, 1)
    rng = np.random.default_rng(3)
    x = (rng.random(n) * 2).astype(np.float32)
    y, z = (rng.random(n).astype(np.float32) for _ in range(2))
    omega = np.array([[0.0, dw]], np.float32)
    occ = []
    for sweep in range(260):
        s.sweep(x, y, z, omega, sweep, move)
        if sweep >= 60 and sweep % 20 == 0:
            occ.append(s.histogram(x, y, z)[0].astype(np.float64))
    occ = np.mean(occ, axis=0)
    ratio = occ[1] / occ[0]
    # ~10 decorrelated samples of 60000 beads: relative error of the ratio ~ 0.4 %
    assert abs(ratio - math.exp(-dw)) < 0.02 * math.exp(-dw), ratio


# ----------------------------------------------------------------------------------------------
# P6  ideal chains: Gaussian bond statistics, <Re^2>, <Rg^2> (chi N = kappa N = 0)
# ----------------------------------------------------------------------------------------------
def _chain_stats(x, y, z, n, N):
    P = np.stack([x, y, z], -1).astype(np.float64).reshape(n, N, 3)
    b = P[:, 1:] - P[:, :-1]
    re2 = ((P[:, -1] - P[:, 0]) ** 2).sum(-1)
    rg2 = ((P - P.mean(1, keepdims=True)) ** 2).sum(-1).mean(1)
    return b, re2, rg2


@pytest.mark.parametrize("move,kw,N,stretch", [(MOVE_LOCAL, {}, 32, 1.0), (MOVE_LOCAL, {}, 8, 1.6),
                                               (MOVE_LOCAL, {}, 8, 0.3), (MOVE_SMC, {"smc_step": 0.05 / 7}, 8, 1.6)])
def test_ideal_chain_statistics(move, kw, N, stretch):
    """k0 = 3 (N-1)/Re0^2: <b_a^2> = 1/(3(N-1)), <b^2> = 1/(N-1),
    <b^4>/<b^2>^2 = 5/3, <Re^2> = 1, <Rg^2> = (N+1)/(6N).  N = 32 starts in equilibrium, which must
    be preserved; the N = 8 runs start from bonds that are too long / too short and must *relax* to
    the closed forms (their Rouse time is short), so a wrong k0 or a dropped neighbour fails."""
    n = 3000 if N == 32 else 12000
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N, n_types=1, box=(8.0,) * 3,
                     grid=(8, 8, 8), chiN=0.0, kappaN=0.0, A=0.1 if N == 32 else 0.2, seed=99, **kw)
    rng = np.random.default_rng(5)
    steps = rng.standard_normal((n, N, 3)) * stretch / math.sqrt(3 * (N - 1))
    steps[:, 0] = rng.random((n, 3)) * 8
    P = np.cumsum(steps, 1).reshape(-1, 3)
    x, y, z = (np.ascontiguousarray(P[:, a], dtype=np.float32) for a in range(3))
    omega = np.zeros((1, s.n_cells), np.float32)
    for sweep in range(60 if stretch == 1.0 else 400):
        s.sweep(x, y, z, omega, sweep, move)
    b, re2, rg2 = _chain_stats(x, y, z, n, N)
    nb = b[..., 0].size
    var_b = 1 / (3 * (N - 1))
    for a in range(3):
        # bonds of one chain are not independent samples -> 3x the iid standard error, 5 sigma
        assert abs(b[..., a].var() - var_b) < 15 * var_b * math.sqrt(2 / nb)
    b2 = (b**2).sum(-1)
    assert abs(b2.mean() * (N - 1) - 1) < 0.012
    assert abs((b2**2).mean() / b2.mean() ** 2 - 5 / 3) < 0.02
    assert abs(re2.mean() - 1.0) < 5 * math.sqrt(2 / 3 / n)                # Var(Re^2) = 2/3 <Re^2>^2
    assert abs(rg2.mean() - (N + 1) / (6 * N)) < 0.006


# ----------------------------------------------------------------------------------------------
# P7  density histogram (Eq. 4)
# ----------------------------------------------------------------------------------------------
def test_histogram_sum_rules_and_brute_force():
    box, grid = (3.0, 2.0, 2.5), (6, 5, 4)
    specs = [(200, np.array([0, 0, 1, 1, 1], np.uint8)), (50, np.array([1, 1, 0], np.uint8))]
    s = OracleSystem(specs=specs, N_ref=5, n_types=2, box=box, grid=grid, seed=1)
    rng = np.random.default_rng(8)
    nb = s.n_beads
    pos = (rng.random((nb, 3)) * 3 - 1) * np.asarray(box) * 2          # spans several periodic images
    dl = np.asarray(box) / np.asarray(grid)
    frac = np.abs((pos / dl) - np.round(pos / dl))
    pos = pos[(frac > 1e-3).all(1)]                                    # keep clear of cell faces
    pos = np.concatenate([pos, pos])[:nb].astype(np.float32)
    x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
    counts = s.histogram(x, y, z)
    types = s.bead_types()
    assert counts.dtype == np.uint32 and counts.shape == (2, 120)
    assert counts[0].sum() == (types == 0).sum() and counts[1].sum() == (types == 1).sum()
    # brute force: O(beads * cells) test of the characteristic function Pi_c on wrapped float64 coordinates
    p64 = pos.astype(np.float64)
    wrapped = p64 - np.floor(p64 / np.asarray(box)) * np.asarray(box)
    brute = np.zeros((2, 120), np.int64)
    for ix in range(grid[0]):
        for iy in range(grid[1]):
            for iz in range(grid[2]):
                lo = np.array([ix, iy, iz]) * dl
                inside = ((wrapped >= lo) & (wrapped < lo + dl)).all(1)
                c = (ix * grid[1] + iy) * grid[2] + iz                 # z fastest
                brute[0, c] = (inside & (types == 0)).sum()
                brute[1, c] = (inside & (types == 1)).sum()
    assert np.array_equal(counts.astype(np.int64), brute)
    assert s.cell_index(float(x[0]), float(y[0]), float(z[0])) == _cell_f64(p64[0], box, grid)


def test_cell_index_is_the_exact_floor_of_the_fp32_box_coordinate():
    """Reading R7: per axis t = fl32(x * fl32(1/L)); cell = floor(t n) mod n in exact arithmetic.  Checked
    with Python rationals (no floating point after t) on random coordinates over many periodic images,
    on coordinates on and next to cell faces and box faces, on tiny negative coordinates (which belong to
    the last cell, never to a cell 'n'), and far from the origin."""
    from fractions import Fraction
    box, grid = (3.0, 2.0, 2.5), (6, 5, 7)
    s = OracleSystem(specs=[(1, np.zeros(1, np.uint8))], N_ref=1, n_types=1, box=box, grid=grid, seed=1)
    rng = np.random.default_rng(5)
    xs = [rng.uniform(-40.0, 40.0, 4000).astype(np.float32)]
    faces = np.arange(-30, 31, dtype=np.float64)[:, None] * 0.5 / np.array([1.0, 2.0, 3.0, 6.0])[None, :]
    f32 = faces.astype(np.float32).ravel()
    xs += [f32, np.nextafter(f32, np.float32(np.inf)), np.nextafter(f32, np.float32(-np.inf))]
    xs += [np.array([-1e-30, -1e-10, -2.0 ** -25, -0.0, 0.0, 1e-30, 2.0 ** -25], np.float32)]
    xs += [rng.uniform(-3.0e5, 3.0e5, 2000).astype(np.float32)]
    xs = np.concatenate(xs)

    def axis(xv, L, n):
        inv_L = np.float32(1.0 / L)
        t = Fraction(float(np.float32(xv) * inv_L))          # the fp32 product, then exact
        return math.floor(t * n) % n

    for i, xv in enumerate(xs):
        yv, zv = xs[(7 * i + 3) % len(xs)], xs[(13 * i + 5) % len(xs)]
        want = (axis(xv, box[0], grid[0]) * grid[1] + axis(yv, box[1], grid[1])) * grid[2] + axis(zv, box[2], grid[2])
        assert s.cell_index(float(xv), float(yv), float(zv)) == want, (xv, yv, zv)
    # the two statements the definition is chosen for
    assert s.cell_index(-1e-30, 0.0, 0.0) == (grid[0] - 1) * grid[1] * grid[2]      # just below 0: last cell
    assert s.cell_index(0.5, 0.0, 0.0) == 1 * grid[1] * grid[2]                      # on a face: the upper cell


def test_homogeneous_melt_mean_occupancy():
    """Mean occupancy = rho_0 DeltaL^3 = beads/cells: 16 for the C1 melt."""
    from workloads import c1, gaussian_walks
    from helpers import oracle_system
    w = c1()
    s = oracle_system(w)
    x, y, z = gaussian_walks(w)
    counts = s.histogram(x, y, z)
    assert counts.sum(axis=1).tolist() == [32768, 32768]
    assert counts.sum() / s.n_cells == 16.0
    tot = counts.sum(0).astype(np.float64)
    # ideal-gas-of-chains start: Poisson (1) plus the same-chain beads sharing a cell
    assert 1.0 < tot.var() / tot.mean() < 4.0


# ----------------------------------------------------------------------------------------------
# P8  fields (Eq. 12) -- hand values and the derivative of Eq. 5-8 in float64
# ----------------------------------------------------------------------------------------------
def _field_system(hamiltonian, chiN=20.0, kappaN=50.0, n_types=2, N_ref=32):
    # 4 cells, 64 beads -> rho_0 DeltaL^3 = 16
    types = np.array(([0, 1] * 16)[:32], np.uint8) if n_types == 2 else np.arange(32, dtype=np.uint8) % n_types
    return OracleSystem(specs=[(2, types)], N_ref=N_ref, n_types=n_types, box=(4.0, 1.0, 1.0),
                        grid=(4, 1, 1), chiN=chiN, kappaN=kappaN, hamiltonian=hamiltonian)


def test_field_hand_values():
    chi0, kappa0 = 20.0 / 32, 50.0 / 32
    counts = np.array([[8, 16, 0, 4], [8, 0, 0, 20]], np.uint32)   # phi = n/16
    w0 = _field_system(0).fields(counts)
    w1 = _field_system(1).fields(counts)
    # cell 0: phi_A = phi_B = 1/2 -> K0: 0, 0 ; K1: chi0/2 each
    assert np.allclose(w0[:, 0], [0, 0], atol=1e-6) and np.allclose(w1[:, 0], [chi0 / 2] * 2, atol=1e-6)
    # cell 1: pure A, phi_A = 1 -> K0: -chi0/2, +chi0/2 ; K1: 0, chi0
    assert np.allclose(w0[:, 1], [-chi0 / 2, chi0 / 2], atol=1e-6) and np.allclose(w1[:, 1], [0, chi0], atol=1e-6)
    # cell 2: empty -> -kappa0 for both options
    assert np.allclose(w0[:, 2], [-kappa0] * 2, atol=1e-6) and np.allclose(w1[:, 2], [-kappa0] * 2, atol=1e-6)
    # cell 3: phi = (1/4, 5/4): P = kappa0/2
    assert np.allclose(w0[:, 3], [kappa0 / 2 + chi0 / 2, kappa0 / 2 - chi0 / 2], atol=1e-6)
    assert np.allclose(w1[:, 3], [kappa0 / 2 + chi0 * 1.25, kappa0 / 2 + chi0 * 0.25], atol=1e-6)


@pytest.mark.parametrize("hamiltonian", [0, 1])
@pytest.mark.parametrize("n_types", [1, 2, 3])
def test_field_is_derivative_of_the_excess_functional(hamiltonian, n_types):
    """omega_i(c) = (1/N) dK/dphi_i(c) with K = K_fluc + K_inter typed from Eq. 6-8
    (PAPER.md:141-151), each unordered pair once; central difference in float64 (K is quadratic)."""
    N_ref = 32
    rng = np.random.default_rng(4)
    chi = rng.random((n_types, n_types)) * 30
    chi = np.triu(chi, 1) + np.triu(chi, 1).T
    s = _field_system(hamiltonian, chiN=chi, kappaN=50.0, n_types=n_types, N_ref=N_ref)
    counts = rng.integers(0, 40, (n_types, 4)).astype(np.uint32)
    omega = s.fields(counts)
    nbar = s.n_beads / s.n_cells
    kappa0N, chi0N = 50.0, chi

    def K(phi):
        k = 0.5 * kappa0N * (phi.sum() - 1.0) ** 2
        for i in range(n_types):
            for j in range(i + 1, n_types):
                if hamiltonian == 0:
                    k -= chi0N[i, j] / 4 * (phi[i] - phi[j]) ** 2 * 2 / 2
                else:
                    k += chi0N[i, j] * phi[i] * phi[j]
        return k

    for c in range(4):
        phi = counts[:, c].astype(np.float64) / nbar
        for i in range(n_types):
            e = np.zeros(n_types)
            e[i] = 1e-3
            dK = (K(phi + e) - K(phi - e)) / 2e-3
            assert abs(omega[i, c] - dK / N_ref) < 2e-5 * (1 + abs(dK / N_ref)), (i, c)


# ----------------------------------------------------------------------------------------------
# P9  kappa N restrains density fluctuations -- sanity band, not an exact value
# ----------------------------------------------------------------------------------------------
def test_kappa_suppresses_density_fluctuations():
    from workloads import Workload, gaussian_walks, homopolymer
    from helpers import oracle_system
    out = {}
    for kN in (0.0, 50.0):
        w = Workload("mini", ((2048, homopolymer(32)),), 32, 1, (4.0,) * 3, (16,) * 3, 0.0, kN, 0.1, 42)
        s = oracle_system(w)
        x, y, z = gaussian_walks(w)
        counts = s.histogram(x, y, z)
        omega = s.fields(counts)
        s.step(x, y, z, counts, omega, 0, 150)
        fl = []
        for i in range(10):
            s.step(x, y, z, counts, omega, 150 + 5 * i, 5)
            n = counts[0].astype(np.float64)
            assert n.sum() == w.n_beads
            fl.append(n.var() / n.mean())
        out[kN] = float(np.mean(fl))
    assert 1.0 < out[0.0] < 4.0      # ideal chains: Poisson + intra-chain clustering
    assert out[50.0] < 0.75 * out[0.0]


# ----------------------------------------------------------------------------------------------
# Smart-MC: proposal pieces against float64 brute force
# ----------------------------------------------------------------------------------------------
def test_smc_gaussians_are_standard_normal():
    s = _free_beads(1, smc_step=0.01)
    g = np.array([s.smc_proposal(b, 1)[0] for b in range(6000)], dtype=np.float64)
    n = g.shape[0]
    for a in range(3):
        assert abs(g[:, a].mean()) < 4 / math.sqrt(n)
        assert abs(g[:, a].var() - 1) < 4 * math.sqrt(2 / n)
        assert abs((g[:, a] ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert abs(np.corrcoef(g.T)[0, 1]) < 4 / math.sqrt(n) and abs(np.corrcoef(g.T)[0, 2]) < 4 / math.sqrt(n)
    us = np.array([s.smc_proposal(b, 1)[1] for b in range(2000)])
    assert 0 <= us.min() and us.max() < 1 and abs(us.mean() - 0.5) < 4 / math.sqrt(12 * 2000)


def test_smc_proposal_is_the_documented_map_of_the_philox_words():
    """Reading R13, value by value: the Gaussians are Box-Muller on the words of the Philox call of kind 2,
    sub 0 -- u1 = 2 - U23(w0) in (0, 1], u2 = U23(w1) - 1 -> g_x = r cos(2 pi u2), g_y = r sin(2 pi u2),
    r = sqrt(-2 ln u1); w2, w3 -> g_z (the cosine branch) -- and the acceptance number is U23(word 0 of the call
    sub 1) - 1.  Recomputed here from the (P1-pinned) Philox words with Python's float64 math; the moments test
    above cannot tell cos from sin or w0 from w2, this one can."""
    seed = 0x0123456789ABCDEF
    s = _free_beads(1, seed=seed, smc_step=0.01)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    two_pi32 = float(np.float32(6.283185307179586))
    for bead, sweep in [(0, 0), (1, 0), (0, 1), (77, 3), (123456, 2**32 + 5), (2**32 - 1, 2**40 + 9)] + \
                       [(b, 11) for b in range(200)]:
        w = oracle.philox4x32_10((bead, sweep & 0xFFFFFFFF, sweep >> 32, (2 << 8) | 0), key)
        v = oracle.philox4x32_10((bead, sweep & 0xFFFFFFFF, sweep >> 32, (2 << 8) | 1), key)
        u1a, u2a = 1.0 - (w[0] >> 9) * 2.0**-23, (w[1] >> 9) * 2.0**-23
        u1b, u2b = 1.0 - (w[2] >> 9) * 2.0**-23, (w[3] >> 9) * 2.0**-23
        ra, rb = math.sqrt(-2.0 * math.log(u1a)), math.sqrt(-2.0 * math.log(u1b))
        ta, tb = float(np.float32(two_pi32 * u2a)), float(np.float32(two_pi32 * u2b))   # the angle is an fp32 product
        want = np.array([ra * math.cos(ta), ra * math.sin(ta), rb * math.cos(tb)])
        g, u = s.smc_proposal(bead, sweep)
        # fp32 logf, sqrtf, sinf / cosf and one product: a few ulp of the radius
        tol = 6.0 * np.spacing(np.float32(max(ra, rb, 1e-3)))
        assert np.all(np.abs(g.astype(np.float64) - want) <= tol), (bead, sweep, g, want)
        assert u == (v[0] >> 9) * 2.0**-23


def test_smc_energy_and_proposal_ratio_match_brute_force():
    specs = [(2, np.array([0, 0, 1, 1], np.uint8)), (1, np.array([1], np.uint8))]
    box, grid = (1.5, 1.0, 2.0), (3, 2, 4)
    a_s = 0.004
    s, chains, pos, omega = _tiny_system(5, specs, 4, box, grid, smc_step=a_s)
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))

    def force(p64, g, first, N):
        j = g - first
        F = np.zeros(3)
        if j > 0:
            F -= k0 * (p64[g] - p64[g - 1])
        if j + 1 < N:
            F -= k0 * (p64[g] - p64[g + 1])
        return F

    for first, N in chains:
        for j in range(N):
            g = first + j
            for sweep in range(4):
                gauss, _ = s.smc_proposal(g, sweep)
                d, dE, log_ratio, rn = s.smc_delta(x, y, z, omega, g, j > 0, j + 1 < N, int(types[g]), gauss)
                p64 = pos.astype(np.float64)
                F = force(p64, g, first, N)
                d64 = a_s * F + math.sqrt(2 * a_s) * gauss.astype(np.float64)
                assert np.allclose(d, d64, rtol=2e-5, atol=2e-6)
                assert np.array_equal(rn, pos[g] + d)
                H0 = _total_H(p64, chains, types, omega, k0, box, grid)
                p64[g] = rn.astype(np.float64)
                H1 = _total_H(p64, chains, types, omega, k0, box, grid)
                assert abs(dE - (H1 - H0)) < 5e-5 * (1 + abs(H1 - H0))
                Fp = force(p64, g, first, N)                       # force at r', recomputed from scratch
                dd = d.astype(np.float64)
                log_fwd = -((dd - a_s * F) ** 2).sum() / (4 * a_s)   # ln T(r -> r')
                log_rev = -((-dd - a_s * Fp) ** 2).sum() / (4 * a_s)  # ln T(r' -> r)
                assert abs(log_ratio - (log_fwd - log_rev)) < 2e-4 * (1 + abs(log_fwd - log_rev))


def test_smc_small_step_accepts_almost_everything():
    n, N = 500, 16
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N, n_types=1, box=(4.0,) * 3, grid=(4,) * 3,
                     A=0.1, seed=3, smc_step=1e-6)
    rng = np.random.default_rng(1)
    st = rng.standard_normal((n, N, 3)) / math.sqrt(3 * (N - 1))
    st[:, 0] = rng.random((n, 3)) * 4
    P = np.cumsum(st, 1).reshape(-1, 3)
    x, y, z = (np.ascontiguousarray(P[:, a], dtype=np.float32) for a in range(3))
    acc = s.sweep(x, y, z, np.zeros((1, 64), np.float32), 0, MOVE_SMC)
    assert acc > 0.99 * n * N


# ----------------------------------------------------------------------------------------------
# initial state of soma_init(xyz0 = NULL): Gaussian walks (BASELINE.json configs)
# ----------------------------------------------------------------------------------------------
def test_init_positions_statistics():
    n, N = 6000, 32
    box = (20.0, 10.0, 5.0)
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N, n_types=1, box=box, grid=(4, 4, 4), seed=7)
    x, y, z = s.init_positions()
    b, re2, rg2 = _chain_stats(x, y, z, n, N)
    nb = b[..., 0].size
    for a, arr in enumerate((x, y, z)):
        first = arr[::N].astype(np.float64)
        assert 0 <= first.min() and first.max() < box[a]
        assert abs(first.mean() - box[a] / 2) < 4 * box[a] / math.sqrt(12 * n)
        assert abs(first.var() - box[a] ** 2 / 12) < 4 * box[a] ** 2 * math.sqrt(1 / 180 / n)
        assert abs(b[..., a].mean()) < 4 * math.sqrt(1 / 93 / nb)
        assert abs(b[..., a].var() - 1 / 93) < 4 / 93 * math.sqrt(2 / nb)
        assert abs((b[..., a] ** 4).mean() / b[..., a].var() ** 2 - 3) < 4 * math.sqrt(96 / nb)
    flat = b.reshape(-1, 3)
    cc = np.corrcoef(flat.T)
    assert abs(cc[0, 1]) < 4 / math.sqrt(nb) and abs(cc[0, 2]) < 4 / math.sqrt(nb) and abs(cc[1, 2]) < 4 / math.sqrt(nb)
    assert abs(re2.mean() - 1.0) < 4 * math.sqrt(2 / 3 / n)
    assert abs(rg2.mean() - (N + 1) / (6 * N)) < 4 * 0.0026
    # reproducible from (seed, bead index) alone
    x2, _, _ = s.init_positions()
    assert np.array_equal(x, x2)


def test_init_positions_are_the_documented_map_of_the_philox_words():
    """Reading R14, value by value: kind-0 Philox words of every bead (counter = (bead, 0, 0, 0)); first bead
    L_a w_a 2^-32; each further bead adds sigma times Box-Muller Gaussians in double -- r = sqrt(-2 ln((w + 1)
    2^-32)) of w0 / w2, angle 2 pi w 2^-32 of w1 / w3, x: r_a cos, y: r_a sin, z: r_b cos -- running sum in double,
    one rounding to fp32.  Recomputed with Python's math from the (P1-pinned) words; two architectures, so the
    bead index runs on across them."""
    seed = 987654321987
    box = (3.0, 5.0, 7.0)
    specs = [(3, np.zeros(5, np.uint8)), (2, np.zeros(9, np.uint8))]
    s = OracleSystem(specs=specs, N_ref=8, n_types=1, box=box, grid=(2, 2, 2), seed=seed)
    x, y, z = s.init_positions()
    key = (seed & 0xFFFFFFFF, seed >> 32)
    sigma = 1.0 / math.sqrt(3.0 * 7.0)
    g = 0
    for n, t in specs:
        for _ in range(n):
            p = [0.0, 0.0, 0.0]
            for j in range(len(t)):
                w = oracle.philox4x32_10((g, 0, 0, 0), key)
                if j == 0:
                    p = [box[a] * (w[a] / 2.0**32) for a in range(3)]
                else:
                    ra = math.sqrt(-2.0 * math.log((w[0] + 1.0) / 2.0**32))
                    rb = math.sqrt(-2.0 * math.log((w[2] + 1.0) / 2.0**32))
                    ta, tb = 2.0 * math.pi * (w[1] / 2.0**32), 2.0 * math.pi * (w[3] / 2.0**32)
                    p = [p[0] + sigma * (ra * math.cos(ta)), p[1] + sigma * (ra * math.sin(ta)), p[2] + sigma * (rb * math.cos(tb))]
                for got, want in zip((x[g], y[g], z[g]), p):
                    # same double-precision formula; libm and Python may differ in the last bit of log / cos
                    assert abs(float(got) - want) <= np.spacing(np.float32(abs(want))) , (g, got, want)
                g += 1
    assert g == s.n_beads


# ----------------------------------------------------------------------------------------------
# P12  random order of the independent sets (Code 2) and field interval
# ----------------------------------------------------------------------------------------------
def test_first_set_is_the_documented_philox_bit_and_fair():
    """Reading R21: bit 31 of word 0 of Philox(counter = (first bead, sweep lo, sweep hi, 3 << 8)).
    Philox itself is pinned by P1, so this pins counter layout, kind and bit; fixed order gives 0."""
    seed = 0xDEADBEEF12345678
    s = OracleSystem(specs=[(4, np.zeros(4, np.uint8))], N_ref=4, n_types=1, box=(1.0,) * 3, grid=(2, 2, 2),
                     seed=seed, set_order=1)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for bead, sweep in [(0, 0), (4, 0), (8, 7), (123456, 2**32 + 5), (2**32 - 4, 2**40 + 1)]:
        w = oracle.philox4x32_10((bead, sweep & 0xFFFFFFFF, sweep >> 32, 3 << 8), key)
        assert s.first_set(bead, sweep) == w[0] >> 31
    bits = np.array([[s.first_set(4 * c, sw) for c in range(4000)] for sw in range(4)])
    assert abs(bits.mean() - 0.5) < 4 * 0.5 / math.sqrt(bits.size)          # fair
    assert abs(np.corrcoef(bits[0], bits[1])[0, 1]) < 4 / math.sqrt(4000)      # fresh every sweep
    assert abs(np.corrcoef(bits[0][:-1], bits[0][1:])[0, 1]) < 4 / math.sqrt(4000)   # and per chain
    s.set_order = 0
    assert all(s.first_set(4 * c, 3) == 0 for c in range(50))


def test_sweep_with_random_set_order_replayed_by_brute_force():
    """Replay of a sweep with set_order = 1, chain by chain, in the order first_set() names (pinned
    above), with float64 brute-force energies: the set that goes second sees the moved beads of the
    set that went first, whichever that was."""
    specs = [(4, np.array([0, 0, 1, 1, 1], np.uint8)), (3, np.array([0, 1] * 4, np.uint8))]
    box, grid = (2.0, 2.0, 2.0), (4, 4, 4)
    s, chains, pos, omega = _tiny_system(21, specs, 8, box, grid, A=0.3, set_order=1)
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    seen = set()
    compared = 0
    for sweep in range(8):
        x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
        dec = np.zeros(len(pos), np.uint8)
        s.sweep(x, y, z, omega, sweep, MOVE_LOCAL, dec)
        ref = pos.copy()
        ref_dec = np.zeros(len(pos), np.uint8)
        fragile = False
        for first, N in chains:
            bit = s.first_set(first, sweep)
            seen.add(bit)
            for parity in (bit, 1 - bit):
                for j in range(parity, N, 2):
                    g = first + j
                    d, u = s.local_proposal(g, sweep)
                    rn = ref[g] + d
                    p64 = ref.astype(np.float64)
                    H0 = _total_H(p64, chains, types, omega, k0, box, grid)
                    p64[g] = rn
                    dE = _total_H(p64, chains, types, omega, k0, box, grid) - H0
                    thr = math.exp(-dE) if dE > 0 else 2.0
                    if abs(u - thr) < 1e-5 or abs(dE) < 1e-6:
                        fragile = True
                    if dE <= 0 or u < thr:
                        ref[g] = rn
                        ref_dec[g] = 1
        if not fragile:
            compared += 1
            assert np.array_equal(dec, ref_dec)
            assert np.array_equal(np.stack([x, y, z], 1), ref)
        pos = np.stack([x, y, z], 1)
    assert seen == {0, 1} and compared >= 3


def test_random_set_order_keeps_ideal_chains_in_equilibrium():
    """Global balance: the sequence of moves does not depend on the configuration, so
    stretched chains still relax to <b^2> = 1/(N-1), <Re^2> = 1 with a random set order."""
    n, N = 12000, 8
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N, n_types=1, box=(8.0,) * 3, grid=(8, 8, 8),
                     A=0.2, seed=77, set_order=1)
    rng = np.random.default_rng(6)
    steps = rng.standard_normal((n, N, 3)) * 1.6 / math.sqrt(3 * (N - 1))
    steps[:, 0] = rng.random((n, 3)) * 8
    P = np.cumsum(steps, 1).reshape(-1, 3)
    x, y, z = (np.ascontiguousarray(P[:, a], dtype=np.float32) for a in range(3))
    omega = np.zeros((1, s.n_cells), np.float32)
    for sweep in range(400):
        s.sweep(x, y, z, omega, sweep, MOVE_LOCAL)
    b, re2, _ = _chain_stats(x, y, z, n, N)
    b2 = (b**2).sum(-1)
    assert abs(b2.mean() * (N - 1) - 1) < 0.012
    assert abs(re2.mean() - 1.0) < 5 * math.sqrt(2 / 3 / n)


def test_field_interval_refreshes_omega_after_every_kth_sweep():
    """Reading R22: step() with field_every = 3 is sweep + histogram every sweep, fields after sweeps
    3, 6, ... only -- composed here from the separately pinned pieces."""
    kw = dict(specs=[(200, np.array([0] * 4 + [1] * 4, np.uint8))], N_ref=8, n_types=2, box=(2.0,) * 3,
              grid=(4, 4, 4), chiN=15.0, kappaN=30.0, A=0.2, seed=3)
    rng = np.random.default_rng(8)
    P = np.cumsum(rng.standard_normal((200, 8, 3)) * 0.2 + (rng.random((200, 1, 3)) * 2) * (np.arange(8)[None, :, None] == 0), 1)
    xyz = [np.ascontiguousarray(P.reshape(-1, 3)[:, a], dtype=np.float32) for a in range(3)]
    a = OracleSystem(field_every=3, **kw)
    xa = [v.copy() for v in xyz]
    ca = a.histogram(*xa)
    oa = a.fields(ca)
    a.step(*xa, ca, oa, 0, 7)
    b = OracleSystem(**kw)
    xb = [v.copy() for v in xyz]
    ob = b.fields(b.histogram(*xb))
    for sweep in range(7):
        b.sweep(*xb, ob, sweep)
        if (sweep + 1) % 3 == 0:
            ob = b.fields(b.histogram(*xb))
    assert all(np.array_equal(u, v) for u, v in zip(xa, xb))
    assert np.array_equal(oa, ob) and np.array_equal(ca, b.histogram(*xb))


# ----------------------------------------------------------------------------------------------
# P13  external fields: forbidden cells and a type-specific static field
# ----------------------------------------------------------------------------------------------
def test_external_field_hand_values():
    """omega = Eq. 12 + ext; forbidden cells are +inf for every type; phi is normalised with the
    accessible volume, so a melt that fills the allowed half of a box uniformly has omega = ext."""
    grid = (2, 2, 2)
    forb = np.array([1, 0, 1, 0, 1, 0, 1, 0], np.uint8)                    # every cell with iz = 0
    ext = np.arange(16, dtype=np.float32).reshape(2, 8) * 0.25
    s = OracleSystem(specs=[(8, np.array([0, 0, 1, 1], np.uint8))], N_ref=4, n_types=2, box=(1.0,) * 3, grid=grid,
                     chiN=12.0, kappaN=40.0, ext_field=ext, forbidden=forb)
    counts = np.zeros((2, 8), np.uint32)
    counts[:, forb == 0] = 4                                               # 32 beads over 4 allowed cells
    om = s.fields(counts)
    assert np.all(np.isposinf(om[:, forb == 1]))
    assert np.allclose(om[:, forb == 0], ext[:, forb == 0], atol=1e-6)      # phi_A = phi_B = 1/2: Eq. 12 gives 0
    s2 = OracleSystem(specs=[(8, np.array([0, 0, 1, 1], np.uint8))], N_ref=4, n_types=2, box=(1.0,) * 3, grid=grid,
                      chiN=12.0, kappaN=40.0)
    counts2 = np.full((2, 8), 2, np.uint32)
    assert np.allclose(s2.fields(counts2), 0.0, atol=1e-6)                   # same melt without walls
    s3 = OracleSystem(specs=[(8, np.array([0, 0, 1, 1], np.uint8))], N_ref=4, n_types=2, box=(1.0,) * 3, grid=grid,
                      chiN=12.0, kappaN=40.0, ext_field=ext)
    assert np.allclose(s3.fields(counts2), ext, atol=1e-6)


def test_confined_free_beads_stay_out_of_forbidden_cells_and_follow_the_external_field():
    """Free beads (N = 1, chi = kappa = 0) in a slit: walls = the two outer z layers, a two-level
    attraction inside.  Through step() (fields refreshed every sweep): no bead ever enters a wall
    cell, and the occupation ratio of the two levels is exp(-delta) (Boltzmann)."""
    n, grid, box = 20000, (4, 4, 8), (2.0, 2.0, 4.0)
    cells = 4 * 4 * 8
    iz = np.arange(cells) % 8
    forb = ((iz == 0) | (iz == 7)).astype(np.uint8)
    delta = 0.7
    ext = np.where((iz == 1) | (iz == 6), -delta, 0.0).astype(np.float32)[None, :]   # attraction next to the walls
    s = OracleSystem(specs=[(n, np.zeros(1, np.uint8))], N_ref=1, n_types=1, box=box, grid=grid, A=0.4, seed=17,
                     ext_field=ext, forbidden=forb)
    rng = np.random.default_rng(9)
    x = (rng.random(n) * 2).astype(np.float32); y = (rng.random(n) * 2).astype(np.float32)
    z = (0.5 + rng.random(n) * 3.0).astype(np.float32)                       # inside the slit
    counts = s.histogram(x, y, z)
    omega = s.fields(counts)
    occ_lo = occ_hi = 0
    for block in range(30):
        s.step(x, y, z, counts, omega, 10 * block, 10)
        assert counts[0, forb == 1].sum() == 0
        if block >= 5:
            occ_lo += int(counts[0, (iz == 1) | (iz == 6)].sum())
            occ_hi += int(counts[0, (iz >= 2) & (iz <= 5)].sum())
    # 2 attractive layers vs 4 neutral layers: ratio of per-cell occupations = exp(delta)
    ratio = (occ_lo / 2) / (occ_hi / 4)
    assert abs(ratio / math.exp(delta) - 1) < 0.03


# ----------------------------------------------------------------------------------------------
# P14  molecule-parallel scheme: N random picks per molecule and sweep (Code 1)
# ----------------------------------------------------------------------------------------------
def test_pick_is_the_documented_philox_word_and_uniform():
    """Reading R24: i = floor(w0 N / 2^32), w0 = word 0 of Philox(counter = (attempt id, sweep, kind 4));
    uniform over 0..N-1, so "on average each particle is attempted once per MC step"."""
    seed = 0x0123456789ABCDEF
    s = OracleSystem(specs=[(4, np.zeros(5, np.uint8))], N_ref=5, n_types=1, box=(1.0,) * 3, grid=(2, 2, 2), seed=seed)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for attempt, sweep, N in [(0, 0, 5), (7, 3, 32), (2**32 - 1, 2**33 + 9, 100), (12345, 1, 1)]:
        w = oracle.philox4x32_10((attempt, sweep & 0xFFFFFFFF, sweep >> 32, 4 << 8), key)
        assert s.pick(attempt, sweep, N) == (w[0] * N) >> 32 < N
    N, n = 7, 70000
    picks = np.array([s.pick(a, 5, N) for a in range(n)])
    hist = np.bincount(picks, minlength=N)
    assert hist.min() > 0 and np.all(np.abs(hist - n / N) < 4.5 * math.sqrt(n / N))
    assert abs(np.corrcoef(picks[:-1], picks[1:])[0, 1]) < 4 / math.sqrt(n)


def test_molecule_sweep_replayed_by_brute_force():
    """Replay of Code 1 attempt by attempt with float64 brute-force energies: the k-th attempt of a
    chain moves the particle pick() names with the random numbers of counter word first + k, and sees
    every earlier accepted move of its chain (also of the same particle picked twice)."""
    specs = [(4, np.array([0, 0, 1, 1, 1], np.uint8)), (3, np.array([0, 1] * 4, np.uint8))]
    box, grid = (2.0, 2.0, 2.0), (4, 4, 4)
    s, chains, pos, omega = _tiny_system(31, specs, 8, box, grid, A=0.3)
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    compared, repeats = 0, 0
    for sweep in range(8):
        x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
        dec = np.zeros(len(pos), np.uint8)
        acc = s.sweep_molecules(x, y, z, omega, sweep, MOVE_LOCAL, dec)
        ref = pos.copy()
        ref_dec = np.zeros(len(pos), np.uint8)
        fragile = False
        for first, N in chains:
            picked = [s.pick(first + k, sweep, N) for k in range(N)]
            repeats += N - len(set(picked))
            for k, i in enumerate(picked):
                g = first + i
                d, u = s.local_proposal(first + k, sweep)
                rn = ref[g] + d
                p64 = ref.astype(np.float64)
                H0 = _total_H(p64, chains, types, omega, k0, box, grid)
                p64[g] = rn
                dE = _total_H(p64, chains, types, omega, k0, box, grid) - H0
                thr = math.exp(-dE) if dE > 0 else 2.0
                if abs(u - thr) < 1e-5 or abs(dE) < 1e-6:
                    fragile = True
                if dE <= 0 or u < thr:
                    ref[g] = rn
                    ref_dec[first + k] = 1
        if not fragile:
            compared += 1
            assert np.array_equal(dec, ref_dec) and acc == int(ref_dec.sum())
            assert np.array_equal(np.stack([x, y, z], 1), ref)
        pos = np.stack([x, y, z], 1)
    assert compared >= 3 and repeats > 0


def test_molecule_scheme_relaxes_ideal_chains():
    """Each single move satisfies detailed balance and the pick does not depend on the configuration,
    so stretched ideal chains relax to <b^2> = 1/(N-1), <Re^2> = 1 under Code 1 as under Code 2."""
    n, N = 12000, 8
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N, n_types=1, box=(8.0,) * 3, grid=(8, 8, 8),
                     A=0.2, seed=78, scheme=1)
    rng = np.random.default_rng(7)
    steps = rng.standard_normal((n, N, 3)) * 1.6 / math.sqrt(3 * (N - 1))
    steps[:, 0] = rng.random((n, 3)) * 8
    P = np.cumsum(steps, 1).reshape(-1, 3)
    x, y, z = (np.ascontiguousarray(P[:, a], dtype=np.float32) for a in range(3))
    counts = s.histogram(x, y, z)
    omega = s.fields(counts)                      # chi = kappa = 0: identically zero
    s.step(x, y, z, counts, omega, 0, 600)        # step() dispatches on scheme
    b, re2, _ = _chain_stats(x, y, z, n, N)
    b2 = (b**2).sum(-1)
    assert abs(b2.mean() * (N - 1) - 1) < 0.012
    assert abs(re2.mean() - 1.0) < 5 * math.sqrt(2 / 3 / n)


# ----------------------------------------------------------------------------------------------
# P15  general molecular architectures: bond lists, independent sets
# ----------------------------------------------------------------------------------------------
def _star(arms, arm_len):
    """Bonds of a star: monomer 0 is the centre, arm a holds monomers 1 + a*arm_len ... in order."""
    bonds = []
    for a in range(arms):
        prev = 0
        for k in range(arm_len):
            j = 1 + a * arm_len + k
            bonds.append((prev, j))
            prev = j
    return np.array(bonds, np.uint32)


def test_independent_sets_are_greedy_first_fit_and_valid():
    star, ring5 = _star(3, 4), np.array([(0, 1), (1, 2), (2, 3), (3, 4), (4, 0)], np.uint32)
    lin = np.array([(j, j + 1) for j in range(6)], np.uint32)
    s = OracleSystem(specs=[(1, np.zeros(13, np.uint8)), (1, np.zeros(5, np.uint8)), (1, np.zeros(7, np.uint8)),
                            (1, np.zeros(7, np.uint8))], N_ref=8, n_types=1, box=(1.0,) * 3, grid=(2, 2, 2),
                     bonds=[star, ring5, lin, None])
    for spec, bonds, N in [(0, star, 13), (1, ring5, 5), (2, lin, 7)]:
        sets = s.sets(spec)
        nbrs = [[] for _ in range(N)]
        for i, j in bonds:
            nbrs[i].append(j); nbrs[j].append(i)
        for j in range(N):
            earlier = {int(sets[k]) for k in nbrs[j] if k < j}
            assert sets[j] == min(c for c in range(N) if c not in earlier)     # first fit in monomer order
            assert all(sets[k] != sets[j] for k in nbrs[j])                    # members are not bonded
    assert list(s.sets(1)) == [0, 1, 0, 1, 2]                                  # odd ring needs a third set
    assert list(s.sets(2)) == [0, 1, 0, 1, 0, 1, 0] == list(s.sets(3))         # linear chain: even / odd (Fig. 1)
    assert s.sets(0)[0] == 0 and set(s.sets(0)[[1, 5, 9]]) == {1}              # star: centre, then first arm beads


@pytest.mark.parametrize("move,kw", [(MOVE_LOCAL, {}), (MOVE_SMC, {"smc_step": 0.004})])
def test_linear_chain_given_as_bonds_reproduces_the_chain_code(move, kw):
    N, n = 9, 40
    types = np.array([0, 0, 0, 1, 1, 1, 1, 0, 0], np.uint8)
    lin = np.array([(j + 1, j) if j % 2 else (j, j + 1) for j in range(N - 1)][::-1], np.uint32)   # shuffled on purpose
    common = dict(specs=[(n, types)], N_ref=N, n_types=2, box=(2.0,) * 3, grid=(4, 4, 4), A=0.3, seed=5, **kw)
    a, b = OracleSystem(**common), OracleSystem(bonds=[lin], **common)
    rng = np.random.default_rng(3)
    P = np.cumsum(rng.standard_normal((n, N, 3)) * 0.2 + (rng.random((n, 1, 3)) * 2) * (np.arange(N)[None, :, None] == 0), 1)
    xa = [np.ascontiguousarray(P.reshape(-1, 3)[:, c], dtype=np.float32) for c in range(3)]
    xb = [v.copy() for v in xa]
    omega = rng.normal(0, 1, (2, 64)).astype(np.float32)
    for sweep in range(6):
        da, db = np.zeros(n * N, np.uint8), np.zeros(n * N, np.uint8)
        assert a.sweep(*xa, omega, sweep, move, da) == b.sweep(*xb, omega, sweep, move, db)
        assert np.array_equal(da, db) and all(np.array_equal(u, v) for u, v in zip(xa, xb))


def _total_H_bonds(pos, mols, bond_lists, types, omega, k0, box, grid):
    H = 0.0
    for (first, N), bonds in zip(mols, bond_lists):
        for i, j in bonds:
            b = pos[first + i] - pos[first + j]
            H += 0.5 * k0 * float(b @ b)
        for j in range(N):
            H += float(omega[types[first + j], _cell_f64(pos[first + j], box, grid)])
    return H


def test_general_architecture_sweep_replayed_by_brute_force():
    """Star and ring molecules: replay of a sweep set by set (sets from the test above), members in
    monomer order, with the total Hamiltonian (all bonds + field) recomputed in float64."""
    star, ring = _star(3, 2), np.array([(0, 1), (1, 2), (2, 3), (3, 4), (4, 0)], np.uint32)
    specs = [(3, np.array([0, 1, 1, 0, 0, 1, 1], np.uint8)), (2, np.array([0, 0, 1, 1, 1], np.uint8))]
    box, grid = (2.0, 2.0, 2.0), (4, 4, 4)
    s, mols, pos, omega = _tiny_system(41, specs, 8, box, grid, A=0.3, bonds=[star, ring])
    bond_lists = [star] * 3 + [ring] * 2
    set_lists = [s.sets(0)] * 3 + [s.sets(1)] * 2
    types = s.bead_types()
    k0 = 3.0 * (s.N_ref - 1)
    compared = 0
    for sweep in range(8):
        x, y, z = (np.ascontiguousarray(pos[:, a]) for a in range(3))
        dec = np.zeros(len(pos), np.uint8)
        s.sweep(x, y, z, omega, sweep, MOVE_LOCAL, dec)
        ref, ref_dec, fragile = pos.copy(), np.zeros(len(pos), np.uint8), False
        for (first, N), sets in zip(mols, set_lists):
            for i_set in range(int(sets.max()) + 1):
                for j in range(N):
                    if sets[j] != i_set:
                        continue
                    g = first + j
                    d, u = s.local_proposal(g, sweep)
                    rn = ref[g] + d
                    p64 = ref.astype(np.float64)
                    H0 = _total_H_bonds(p64, mols, bond_lists, types, omega, k0, box, grid)
                    p64[g] = rn
                    dE = _total_H_bonds(p64, mols, bond_lists, types, omega, k0, box, grid) - H0
                    thr = math.exp(-dE) if dE > 0 else 2.0
                    if abs(u - thr) < 1e-5 or abs(dE) < 1e-6:
                        fragile = True
                    if dE <= 0 or u < thr:
                        ref[g] = rn
                        ref_dec[g] = 1
        if not fragile:
            compared += 1
            assert np.array_equal(dec, ref_dec)
            assert np.array_equal(np.stack([x, y, z], 1), ref)
        pos = np.stack([x, y, z], 1)
    assert compared >= 3


def test_ideal_star_polymers_relax_to_gaussian_tree_statistics():
    """Every bond is the spring of Eq. 2, so in an ideal branched molecule the mean-square distance of
    two monomers p bonds apart along the tree is p / (N_ref - 1) R_e0^2."""
    arms, arm_len, n, N_ref = 3, 4, 8000, 9
    N = 1 + arms * arm_len
    s = OracleSystem(specs=[(n, np.zeros(N, np.uint8))], N_ref=N_ref, n_types=1, box=(8.0,) * 3, grid=(8, 8, 8),
                     A=0.2, seed=12, bonds=[_star(arms, arm_len)])
    rng = np.random.default_rng(2)
    P = (rng.random((n, 1, 3)) * 8 + rng.standard_normal((n, N, 3)) * 0.05)      # collapsed start: must swell
    x, y, z = (np.ascontiguousarray(P.reshape(-1, 3)[:, a], dtype=np.float32) for a in range(3))
    omega = np.zeros((1, s.n_cells), np.float32)
    for sweep in range(500):
        s.sweep(x, y, z, omega, sweep, MOVE_LOCAL)
    Q = np.stack([x, y, z], -1).astype(np.float64).reshape(n, N, 3)
    def msd(i, j):
        return ((Q[:, i] - Q[:, j]) ** 2).sum(-1).mean()
    b2 = 1.0 / (N_ref - 1)
    tip = [a * arm_len + arm_len for a in range(arms)]
    for (i, j, p) in [(0, 1, 1), (0, tip[0], arm_len), (tip[0], tip[1], 2 * arm_len), (tip[1], tip[2], 2 * arm_len),
                      (2, 3, 1), (1, 5, 2)]:
        assert abs(msd(i, j) / (p * b2) - 1) < 0.03 + 4 * math.sqrt(2 / 3 / n), (i, j, p, msd(i, j))
