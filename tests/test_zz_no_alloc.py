"""soma_fields_static: stage 1 (occupation numbers, Eq. 4, and omega, Eq. 12) for callers that must not allocate.

Some users of this library cannot call cudaMalloc where they need the fields of a configuration: a tool that runs
beside simulations which already fill the GPU, a host program whose own allocator owns the device memory (torch
here, which lends the buffers below), a loop that must not stall the streams running next to it.  For them the
library keeps the occupation numbers of this one entry point in an array that is part of its image (4 MiB per GPU,
n_types * cells <= STATIC_MAX_WORDS) and allocates nothing.  The array is shared by all calls and keeps what the
last call wrote, so the test calls twice in a row with different systems and expects both results to equal the
allocating path's (a context made by soma_init on the same positions, read with soma_fields).

This file sorts last on purpose: under `pytest -x` a failure here hides no other test.
"""
import numpy as np
import pytest

import paper_1711_03828_b200 as P
import workloads


def _by_name(name):
    return next(w for w in workloads.small_cases() if w.name == name)


def _existing_path(w, xyz):
    """omega and counts of the positions xyz from the allocating path: soma_init + soma_fields, 32-bit planes."""
    sim = P.from_workload(w, xyz0=xyz)
    sim.set_option(P.OPT_COUNT_BITS, 32)
    omega, counts = sim.fields()
    sim.destroy()
    return omega, counts


def _static_path(w, xyz, with_counts=True):
    import torch
    d_xyz = torch.from_numpy(xyz).cuda()
    # poisoned outputs: whatever is not written shows
    d_omega = torch.full((w.n_types, w.n_cells), float("nan"), dtype=torch.float32, device="cuda")
    d_counts = torch.full((w.n_types, w.n_cells), -1, dtype=torch.int32, device="cuda") if with_counts else None
    P.fields_static(w.specs, w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, d_xyz, d_omega, d_counts)
    return d_omega.cpu().numpy(), (d_counts.cpu().numpy().view(np.uint32) if with_counts else None)


def _assert_same(w, got, want):
    omega, counts = got
    omega_ref, counts_ref = want
    if counts is not None:
        assert np.array_equal(counts, counts_ref), w.name                      # integers: bit-exact
        assert int(counts.sum()) == w.n_beads
    # the fields' tolerance of the parity tests (1e-5 relative, R16); the arithmetic is the same kernel's,
    # so they are in fact expected to be identical
    scale = max(1.0, float(np.abs(omega_ref).max()))
    assert np.all(np.isfinite(omega)), w.name
    assert float(np.abs(omega - omega_ref).max()) <= 1e-5 * scale, w.name


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_allocating_path():
    # call 1: three architectures, two types, 54,000 words of the array; call 2: one architecture, three types
    # (the any-number-of-types field kernel), 12,288 words -- a smaller part of the array, still holding call 1's numbers
    first, second = _by_name("blend"), _by_name("three_types")
    xyz1 = np.stack(workloads.gaussian_walks(first))
    xyz2 = np.stack(workloads.gaussian_walks(second))
    got1 = _static_path(first, xyz1)
    got2 = _static_path(second, xyz2)
    _assert_same(first, got1, _existing_path(first, xyz1))
    _assert_same(second, got2, _existing_path(second, xyz2))
    # and the first system again, now over the second's leftovers, without the optional counts output
    got3 = _static_path(first, xyz1, with_counts=False)
    assert np.array_equal(got3[0], got1[0])


@pytest.mark.gpu
def test_a_grid_that_nearly_fills_the_array_and_the_other_hamiltonian():
    import torch
    w = workloads.c3().scaled(0.05, "C3x0.05")        # 25,600 chains on C3's grid: 1,000,000 of the 1,048,576 words
    assert 0.9 * P.STATIC_MAX_WORDS < w.n_types * w.n_cells <= P.STATIC_MAX_WORDS
    xyz = np.stack(workloads.gaussian_walks(w))
    _assert_same(w, _static_path(w, xyz), _existing_path(w, xyz))
    sim = P.from_workload(w, xyz0=xyz)
    sim.set_option(P.OPT_COUNT_BITS, 32)
    sim.set_option(P.OPT_HAMILTONIAN, 1)
    omega_ref, _ = sim.fields()
    sim.destroy()
    d_omega = torch.empty((w.n_types, w.n_cells), dtype=torch.float32, device="cuda")
    P.fields_static(w.specs, w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, torch.from_numpy(xyz).cuda(), d_omega,
                    hamiltonian=1)
    assert float(np.abs(d_omega.cpu().numpy() - omega_ref).max()) <= 1e-5 * max(1.0, float(np.abs(omega_ref).max()))


@pytest.mark.gpu
def test_host_pointers_and_bad_coordinates_are_refused():
    import torch
    w = _by_name("tiny_N2")
    xyz = np.stack(workloads.gaussian_walks(w))
    d_omega = torch.empty((w.n_types, w.n_cells), dtype=torch.float32, device="cuda")
    with pytest.raises(P.SomaError) as e:                      # a host array where device memory is expected
        P.fields_static(w.specs, w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, xyz, d_omega)
    assert e.value.code == -1 and "dev_xyz" in str(e.value)
    bad = xyz.copy()
    bad[1, 7] = np.nan
    with pytest.raises(P.SomaError) as e:
        P.fields_static(w.specs, w.N_ref, w.n_types, w.box, w.grid, w.chiN, w.kappaN, torch.from_numpy(bad).cuda(), d_omega)
    assert e.value.code == -6
    # the array is usable afterwards
    _assert_same(w, _static_path(w, xyz), _existing_path(w, xyz))


def test_sizes_beyond_the_static_array_are_refused_before_the_device_is_touched():
    """No GPU needed: the limits are checked first, and the message names them."""
    w = workloads.c3()
    with pytest.raises(P.SomaError) as e:                      # 120^3 cells x 2 types = 3,456,000 words
        P.fields_static(w.specs, w.N_ref, w.n_types, (24.0, 24.0, 24.0), (120, 120, 120), w.chiN, w.kappaN, None, None)
    assert e.value.code == -1 and str(P.STATIC_MAX_WORDS) in str(e.value) and "soma_init" in str(e.value)
    with pytest.raises(P.SomaError) as e:                      # exactly one word too many
        P.fields_static([(4, [0, 0])], 2, 1, (1.0, 1.0, 1.0), (P.STATIC_MAX_WORDS + 1, 1, 1), 0.0, 1.0, None, None)
    assert e.value.code == -1 and str(P.STATIC_MAX_WORDS) in str(e.value)
    with pytest.raises(P.SomaError) as e:                      # 257 monomers
        P.fields_static([(4, [0] * 257)], 2, 1, (1.0, 1.0, 1.0), (4, 4, 4), 0.0, 1.0, None, None)
    assert e.value.code == -1 and str(P.STATIC_MAX_MONOMERS) in str(e.value)
