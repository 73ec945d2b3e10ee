"""GPU parity with an external field h (Eq. 1): CUDA path
through the C ABI against the CPU oracle, bit for bit: tables, packed spins, temperature
permutation, energies, overlaps."""
import numpy as np
import pytest

from ea_inputs import temperature_ladder
from util_pack import words_to_spins

pytestmark = pytest.mark.gpu


def _mods():
    import __graft_entry__ as ge
    ge.build()
    import paper_1311_5582_b200 as pkg
    from oracle import Oracle
    return pkg, Oracle


def _same_state(g, o, L, R):
    st = g.get_state()
    assert (words_to_spins(st["spin_words"], L, R) == o.spins_by_slot()).all(), "spins differ"
    assert (st["temp_of_slot"] == o.perm()[0]).all(), "temperature permutation differs"
    assert (st["energy_by_slot"] == o.energy_by_slot()).all(), "energies by slot differ"
    assert (g.energy() == o.energy()).all(), "energies differ"


@pytest.mark.parametrize("L,nT,R,h,swap,asc", [
    (4, 6, 40, 1, 1, False),
    (4, 5, 33, -2, 2, False),      # even h, odd n_T, swap every 2nd sweep
    (6, 4, 70, 3, 1, True),        # ascending betas, L = 6, ragged R
    (8, 8, 64, -1, 1, False),      # a shape the resident kernel would take at h = 0
    (2, 3, 5, 7, 1, False),        # L = 2, |h| > 6: one spin state always flips
    (16, 4, 32, 2, 0, False),      # no PT
])
def test_field_trajectory_matches_oracle(L, nT, R, h, swap, asc):
    pkg, Oracle = _mods()
    betas = 1.0 / temperature_ladder(nT, 0.6, 2.5)
    if asc:
        betas = betas[::-1].copy()
    g = pkg.EA(L, nT, R, betas, 19)
    o = Oracle(L, nT, R, betas, 19)
    g.set_field(h)
    o.set_field(h)
    fast = abs(h) <= 2 and L <= 16               # |h| <= 2 on the resident kernels' lattices, else the generic path
    assert g.get_field() == h
    assert g.get_kernel() == (pkg.binding.EA_KERNEL_RESIDENT if fast else pkg.binding.EA_KERNEL_GENERIC)
    assert L < 32
    ga, gs = g.get_field_tables()
    oa, os_ = o.field_tables()
    assert (ga == oa).all() and (gs == os_).all()          # both sides hold identical tables
    _same_state(g, o, L, R)                                  # energies include the field term
    for n in (1, 4, 7):
        g.sweep(n, swap)
        o.sweep(n, swap)
        _same_state(g, o, L, R)
    pairs = [[0, 1], [R - 1, -1], [2, 2]]
    assert (g.overlap(pairs) == o.overlap(pairs)).all()
    if swap:
        assert o.counters()["swap_accepted"] > 0
    # back to zero field: the fast kernels return and the trajectories still agree
    g.set_field(0)
    o.set_field(0)
    assert g.get_field() == 0
    g.sweep(5, swap)
    o.sweep(5, swap)
    _same_state(g, o, L, R)
    g.destroy()


@pytest.mark.parametrize("L,nT,R,h,swap,ns", [
    (16, 24, 64, 1, 1, 6), (16, 24, 64, -1, 1, 6), (16, 7, 40, 2, 1, 5), (16, 12, 96, -2, 2, 7),
    (8, 16, 32, 1, 1, 12), (8, 16, 40, -2, 1, 12), (8, 5, 64, 2, 3, 9), (8, 2, 32, -1, 1, 8),
    (16, 24, 33, 1, 0, 4),
    (12, 20, 64, 1, 2, 6), (12, 7, 33, -2, 1, 5), (4, 16, 40, 2, 1, 20), (6, 5, 70, -1, 1, 9), (2, 3, 5, 1, 1, 12),
])
def test_field_on_the_resident_kernel_matches_oracle_and_the_generic_kernel(L, nT, R, h, swap, ns):
    """Field |h| <= 2 in the shared-memory-resident kernel (four threshold columns of the shifted
    class index, up/down-spin count fused into the energy pass): bit for bit against the oracle,
    across several calls, and with the kernel switched in mid-run."""
    pkg, Oracle = _mods()
    betas = 1.0 / temperature_ladder(nT, 0.7, 2.2)
    g = pkg.EA(L, nT, R, betas, 23)
    o = Oracle(L, nT, R, betas, 23)
    g.set_field(h); o.set_field(h)
    assert g.get_kernel() == pkg.binding.EA_KERNEL_RESIDENT
    for n in (1, ns, 2):
        g.sweep(n, swap); o.sweep(n, swap)
        _same_state(g, o, L, R)
    g.set_kernel(pkg.binding.EA_KERNEL_GENERIC)
    g.sweep(3, swap); o.sweep(3, swap)
    _same_state(g, o, L, R)
    g.set_kernel(pkg.binding.EA_KERNEL_RESIDENT)
    g.sweep(3, swap); o.sweep(3, swap)
    _same_state(g, o, L, R)
    g.destroy()


@pytest.mark.parametrize("L,nT,R,h,swap,ns", [
    (32, 8, 32, 1, 1, 4), (32, 5, 40, -2, 1, 3), (32, 32, 32, 2, 2, 3), (32, 6, 64, -1, 0, 3), (64, 3, 32, 1, 1, 2),
])
def test_field_on_the_streaming_kernel_matches_oracle(L, nT, R, h, swap, ns):
    """Field |h| <= 2 in the streaming kernel (L = 32, 64): the same four-column route as in the
    resident kernel, the paying spins counted from the tile's index-aligned quad."""
    pkg, Oracle = _mods()
    betas = 1.0 / temperature_ladder(nT, 0.9, 2.2)
    g = pkg.EA(L, nT, R, betas, 29)
    o = Oracle(L, nT, R, betas, 29)
    g.set_field(h); o.set_field(h)
    assert g.get_kernel() == pkg.binding.EA_KERNEL_STREAM
    for n in (1, ns):
        g.sweep(n, swap); o.sweep(n, swap)
        _same_state(g, o, L, R)
    g.set_kernel(pkg.binding.EA_KERNEL_GENERIC)
    g.sweep(2, swap); o.sweep(2, swap)
    _same_state(g, o, L, R)
    g.destroy()


def test_field_restrictions_and_errors():
    pkg, _ = _mods()
    betas = 1.0 / temperature_ladder(4, 0.8, 2.0)
    g = pkg.EA(16, 4, 32, betas, 3)
    auto = g.get_kernel()
    assert auto != pkg.binding.EA_KERNEL_GENERIC
    with pytest.raises(pkg.EAError):
        g.get_field_tables()                                 # no field set
    with pytest.raises(pkg.EAError):
        g.set_field(65)
    g.set_field(3)                                           # |h| > 2: generic kernels only
    assert g.get_kernel() == pkg.binding.EA_KERNEL_GENERIC
    with pytest.raises(pkg.EAError) as e:
        g.set_kernel(pkg.binding.EA_KERNEL_RESIDENT)
    assert e.value.code == -5
    g.set_field(2)                                           # |h| <= 2: the resident kernel runs
    assert g.get_kernel() == pkg.binding.EA_KERNEL_RESIDENT
    g.set_kernel(pkg.binding.EA_KERNEL_GENERIC)
    assert g.get_kernel() == pkg.binding.EA_KERNEL_GENERIC
    g.set_kernel(pkg.binding.EA_KERNEL_AUTO)
    with pytest.raises(pkg.EAError) as e:
        g.set_kernel(pkg.binding.EA_KERNEL_TILED)
    assert e.value.code == -5
    acc, swp = g.get_tables()                                # still the zero-field tables
    with pytest.raises(pkg.EAError) as e:
        g.set_tables(acc, swp)
    assert e.value.code == -5
    g.set_field(0)
    assert g.get_kernel() == auto
    g.set_tables(acc, swp)
    g.destroy()


def test_measurement_series_with_field():
    pkg, Oracle = _mods()
    from oracle import binder_ratio
    L, nT, R, h = 4, 4, 64, 1
    betas = 1.0 / temperature_ladder(nT, 0.8, 2.0)
    g = pkg.EA(L, nT, R, betas, 5)
    o = Oracle(L, nT, R, betas, 5)
    for x in (g, o):
        x.pair_couplings()
        x.set_field(h)
    wp = [[0, 1], [0, -1]]
    g.measure_begin(wp)
    g.measure(4, 2, 1)
    acc = o.measure(4, 2, 1, wp)
    m = g.get_moments()
    assert (m["q1"].astype(object) == acc["q1"]).all() and (m["q2"].astype(object) == acc["q2"]).all()
    assert (m["e1"].astype(object) == acc["e1"]).all() and (m["e2"].astype(object) == acc["e2"]).all()
    gb, ob = g.get_binder(), binder_ratio(acc)
    assert (np.abs(gb - ob) <= 1e-12 * np.abs(ob)).all()
    g.destroy()
