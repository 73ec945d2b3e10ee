"""Data-moving swap (SURVEY 8(f3) second half, R26, ea_set_swap_mode): an accepted swap
exchanges the two lattices bit by bit under the word's acceptance mask, temperatures stay with the
slots.  Against the oracle's swap mode 1, on every sweep kernel.  Integer work: bit for bit."""
import numpy as np
import pytest

from ea_inputs import temperature_ladder
from oracle import Oracle
from util_pack import words_to_spins

pytestmark = pytest.mark.gpu


def _pair(L, nT, R, seed, field=0, kernel=None, r0=0):
    from paper_1311_5582_b200 import EA, EA_SWAP_MOVE
    betas = 1.0 / temperature_ladder(nT, 0.6, 2.0)
    g = EA(L, nT, R, betas, seed, first_realization=r0)
    o = Oracle(L, nT, R, betas, seed, r0=r0)
    if field:
        g.set_field(field); o.set_field(field)
    if kernel is not None:
        g.set_kernel(kernel)
    g.set_swap_mode(EA_SWAP_MOVE)
    o.set_swap_mode(1)
    return g, o


def _same(g, o, L, R, nT):
    st = g.get_state()
    assert (words_to_spins(st["spin_words"], L, R) == o.spins_by_slot()).all(), "spins differ"
    assert (st["temp_of_slot"] == np.arange(nT)).all(), "temperatures must stay with the slots"
    assert (st["energy_by_slot"] == o.energy_by_slot()).all(), "energies by slot differ"
    assert (g.energy() == o.energy()).all(), "energies differ"


# kernel ids: 0 auto, 1 generic (persistent), 2 resident, 3 tiled, 4 stream, 6 generic stepwise
@pytest.mark.parametrize("L,nT,R,ns,swap,kernel,field", [
    (4, 6, 5, 30, 1, 0, 0), (2, 3, 33, 20, 1, 0, 0), (6, 5, 40, 12, 2, 0, 0), (8, 16, 40, 10, 1, 2, 0),
    (16, 24, 33, 6, 1, 2, 0), (16, 7, 3, 7, 3, 3, 0), (32, 4, 34, 3, 1, 4, 0), (8, 9, 4, 9, 1, 1, 0),
    (8, 9, 4, 9, 2, 6, 0), (14, 3, 2, 4, 1, 0, 0), (8, 6, 35, 8, 1, 0, 1), (16, 5, 3, 5, 1, 0, -2),
    (4, 5, 3, 6, 1, 0, 3), (4, 1, 3, 5, 1, 0, 0), (8, 7, 4, 9, 0, 0, 0)])
def test_moving_swaps_match_oracle(L, nT, R, ns, swap, kernel, field):
    if nT < 2:
        from paper_1311_5582_b200 import EA, EA_SWAP_MOVE, EAError
        g = EA(L, nT, R, np.array([1.0]), 3)
        with pytest.raises(EAError):
            g.set_swap_mode(EA_SWAP_MOVE)
        g.destroy()
        return
    g, o = _pair(L, nT, R, 23 + L, field=field, kernel=kernel or None)
    _same(g, o, L, R, nT)
    g.sweep(ns, swap); o.sweep(ns, swap)
    _same(g, o, L, R, nT)
    g.sweep(3, swap); o.sweep(3, swap)           # continuation: the swap cadence follows the global sweep index
    _same(g, o, L, R, nT)
    pairs = [[0, min(1, R - 1)], [R - 1, -1]]
    assert (g.overlap(pairs) == o.overlap(pairs)).all()
    if swap and L <= 8:                          # small lattices: some exchange has really happened
        assert 0 < o.counters()["swap_accepted"]
    g.destroy()


def test_mode_rules_and_word_independence():
    from paper_1311_5582_b200 import EA, EA_LAYOUT_REPLICA_BITS, EA_SWAP_MOVE, EA_SWAP_PERMUTE, EAError
    L, nT, R = 4, 6, 40
    g, o = _pair(L, nT, R, 5, r0=64)
    assert g.get_swap_mode() == EA_SWAP_MOVE
    with pytest.raises(EAError):
        g.set_layout(EA_LAYOUT_REPLICA_BITS)            # no moving swaps in the paper's coding
    g.sweep(9, 1); o.sweep(9, 1)
    _same(g, o, L, R, nT)
    # the second word of a 40-realization problem is the first word of the problem that starts at r0 + 32
    g2, o2 = _pair(L, nT, 8, 5, r0=96)
    g2.sweep(9, 1)
    a = words_to_spins(g.get_state()["spin_words"], L, R)[32:]
    b = words_to_spins(g2.get_state()["spin_words"], L, 8)
    assert (a == b).all()
    # back to index-permuting swaps at any time (the permutation is the identity); the other way only then
    g.set_swap_mode(EA_SWAP_PERMUTE); o.set_swap_mode(0)
    g.sweep(4, 1); o.sweep(4, 1)
    st = g.get_state()
    assert (words_to_spins(st["spin_words"], L, R) == o.spins_by_slot()).all()
    assert (st["temp_of_slot"] == o.perm()[0]).all()
    with pytest.raises(EAError):
        g.set_swap_mode(EA_SWAP_MOVE)                   # permutation no longer the identity
    # checkpoint / resume in moving mode
    st = g2.get_state()
    g3, _ = _pair(L, nT, 8, 5, r0=96)
    g3.set_state(st)
    g2.sweep(5, 2); g3.sweep(5, 2)
    assert (g2.get_state()["spin_words"] == g3.get_state()["spin_words"]).all()
    for x in (g, g2, g3):
        x.destroy()
