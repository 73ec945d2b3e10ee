"""Second workload (R24): the paper's own multispin coding, bits of a word =
temperature replicas of one realization, one random number per replica (ea_set_layout), against
the oracle's per-replica draw mode.  Integer work: bit for bit."""
import numpy as np
import pytest

from ea_inputs import random_couplings, random_spins, temperature_ladder
from oracle import Oracle
from util_pack import words_to_spins

pytestmark = pytest.mark.gpu


def _pair(L, nT, R, seed, Tlo=0.6, Thi=2.0, r0=0):
    from paper_1311_5582_b200 import EA, EA_LAYOUT_REPLICA_BITS
    betas = 1.0 / temperature_ladder(nT, Tlo, Thi)
    g = EA(L, nT, R, betas, seed, first_realization=r0)
    g.set_layout(EA_LAYOUT_REPLICA_BITS)
    o = Oracle(L, nT, R, betas, seed, r0=r0)
    o.set_draw_mode(1)
    return g, o


def _same(g, o, L, R):
    st = g.get_state()
    assert (words_to_spins(st["spin_words"], L, R) == o.spins_by_slot()).all(), "spins differ"
    assert (st["temp_of_slot"] == o.perm()[0]).all(), "temperature permutation differs"
    assert (st["energy_by_slot"] == o.energy_by_slot()).all(), "energies by slot differ"
    assert (g.energy() == o.energy()).all(), "energies differ"


@pytest.mark.parametrize("L,nT,R,ns,swap", [(4, 6, 5, 30, 1), (2, 3, 33, 20, 1), (6, 5, 7, 12, 2), (8, 16, 40, 10, 1),
                                           (12, 20, 4, 6, 2), (16, 24, 3, 5, 1), (4, 40, 3, 15, 1), (4, 1, 3, 5, 1),
                                           (8, 7, 4, 9, 0), (32, 4, 2, 2, 1)])
def test_replica_layout_matches_oracle(L, nT, R, ns, swap):
    from paper_1311_5582_b200 import EA_KERNEL_REPLICA
    g, o = _pair(L, nT, R, 17 + L)
    assert g.get_kernel() == EA_KERNEL_REPLICA
    _same(g, o, L, R)
    g.sweep(ns, swap); o.sweep(ns, swap)
    _same(g, o, L, R)
    g.sweep(3, swap); o.sweep(3, swap)         # continuation of a call sequence
    _same(g, o, L, R)
    pairs = [[0, min(1, R - 1)], [R - 1, -1]]
    assert (g.overlap(pairs) == o.overlap(pairs)).all()
    g.destroy()


def test_inputs_sharding_and_switching_layouts():
    from paper_1311_5582_b200 import EA_LAYOUT_REALIZATION_BITS, EA_LAYOUT_REPLICA_BITS
    L, nT, R = 4, 6, 40
    g, o = _pair(L, nT, R, 5, r0=64)
    J, s = random_couplings(R, L ** 3, 1), random_spins(R, nT, L ** 3, 2)
    g.set_couplings(J); o.set_couplings(J)
    g.set_spins(s); o.set_spins(s)
    g.sweep(8, 1); o.sweep(8, 1)
    _same(g, o, L, R)
    # back to the first coding in mid-run, and again to the second: the state carries over
    g.set_layout(EA_LAYOUT_REALIZATION_BITS); o.set_draw_mode(0)
    g.sweep(5, 1); o.sweep(5, 1)
    _same(g, o, L, R)
    g.set_layout(EA_LAYOUT_REPLICA_BITS); o.set_draw_mode(1)
    g.sweep(5, 1); o.sweep(5, 1)
    _same(g, o, L, R)
    # checkpoint / resume in the second coding
    st = g.get_state()
    g.sweep(4, 1)
    end = g.get_state()
    g.set_state(st)
    g.sweep(4, 1)
    again = g.get_state()
    assert (words_to_spins(end["spin_words"], L, R) == words_to_spins(again["spin_words"], L, R)).all()   # padding bits aside
    assert (end["temp_of_slot"] == again["temp_of_slot"]).all()
    o.sweep(4, 1)
    _same(g, o, L, R)
    g.destroy()


def test_unsupported_combinations_are_refused():
    from paper_1311_5582_b200 import EA, EAError, EA_LAYOUT_REPLICA_BITS
    g = EA(4, 4, 3, 1.0 / temperature_ladder(4, 0.6, 2.0), 1)
    g.set_field(1)
    with pytest.raises(EAError):
        g.set_layout(EA_LAYOUT_REPLICA_BITS)
    g.set_field(0)
    g.set_layout(EA_LAYOUT_REPLICA_BITS)
    with pytest.raises(EAError):
        g.set_field(1)
    with pytest.raises(EAError):
        g.set_kernel(1)
    g.destroy()


@pytest.mark.parametrize("L,nT,R,p,layout", [(4, 6, 40, 0.3, 0), (8, 8, 33, 0.9, 0), (16, 5, 64, 0.5, 0), (32, 3, 32, 0.75, 0),
                                             (12, 4, 7, 1.0, 0), (6, 6, 5, 0.2, 1)])
def test_seeded_bond_concentration_matches_oracle(L, nT, R, p, layout):
    """+-J couplings with bond concentration p (ea_seed_couplings, R25) are the
    oracle's bit for bit, on a sharded handle too, and the trajectories that follow agree."""
    from paper_1311_5582_b200 import EA
    betas = 1.0 / temperature_ladder(nT, 0.7, 2.2)
    g = EA(L, nT, R, betas, 41, first_realization=64)
    o = Oracle(L, nT, R, betas, 41, r0=64)
    g.set_layout(layout); o.set_draw_mode(layout)
    g.seed_couplings(p); o.seed_couplings(p)
    assert (g.get_couplings() == o.couplings()).all()
    _same(g, o, L, R)
    g.sweep(6, 1); o.sweep(6, 1)
    _same(g, o, L, R)
    g.destroy()
