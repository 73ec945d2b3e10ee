"""Pins for the oracle's +-J couplings with bond concentration p (R25;
PAPER.md:341 "other distributions of the couplings").  Expected values: closed forms of iid bonds
and an independent Python Philox, never oracle code."""
import numpy as np
import pytest

from oracle import Oracle, philox4x32_10


def _mk(L=4, nT=3, R=6, seed=0xABCDEF0123, r0=0):
    return Oracle(L, nT, R, np.linspace(1.2, 0.4, nT), seed, r0=r0)


def test_closed_forms_p_one_and_zero():
    o = _mk()
    s = o.spins_by_slot().copy()
    o.seed_couplings(1.0)
    assert (o.couplings() == 1).all()                      # ferromagnet
    assert (o.spins_by_slot() == s).all()                  # spins are kept
    L, N = 4, 64
    s3 = s.reshape(6, 3, L, L, L).astype(np.int64)
    E = -sum((s3 * np.roll(s3, -1, axis=ax)).sum(axis=(2, 3, 4)) for ax in (4, 3, 2))
    assert (o.energy_by_slot() == E).all()                 # energies recomputed: -sum s s
    o.seed_couplings(0.0)
    assert (o.couplings() == -1).all() and (o.energy_by_slot() == -E).all()
    with pytest.raises(ValueError):
        o.seed_couplings(1.5)


def test_counter_convention_against_an_independent_philox():
    seed, r0, L, R = 0x1122334455667788, 32, 4, 3
    o = _mk(L=L, R=R, seed=seed, r0=r0)
    p = 0.3
    o.seed_couplings(p)
    J = o.couplings()
    thr = int(np.floor(p * 2.0 ** 32))
    k0, k1 = seed & 0xFFFFFFFF, seed >> 32
    for r in range(R):
        for d in range(3):
            for i in range(0, L ** 3, 7):
                u = philox4x32_10(0, i, r0 + r, (5 << 16) | d, k0, k1)[0]
                assert J[r, d, i] == (1 if u < thr else -1)


@pytest.mark.parametrize("p", [0.3, 0.5, 0.9])
def test_bond_and_frustration_fractions(p):
    """iid bonds: fraction of +1 = p, and a plaquette (product of its four bonds = -1) is
    frustrated with probability (1 - (2p - 1)^4) / 2."""
    L, R = 8, 32
    o = Oracle(L, 2, R, np.array([1.0, 0.5]), 7)
    o.seed_couplings(p)
    J = o.couplings().astype(np.int64).reshape(R, 3, L, L, L)       # [r][d][z][y][x], d = x, y, z
    n = J.size
    assert abs((J == 1).mean() - p) < 4 * np.sqrt(p * (1 - p) / n)
    Jx, Jy = J[:, 0], J[:, 1]
    plaq = Jx * np.roll(Jy, -1, axis=3) * np.roll(Jx, -1, axis=2) * Jy      # xy plaquettes
    f = (plaq == -1).mean()
    expect = (1 - (2 * p - 1) ** 4) / 2
    assert abs(f - expect) < 4 * np.sqrt(0.25 / plaq.size) + 1e-3
    # realizations are independent of each other and of r0 (word independence)
    part = Oracle(L, 2, 8, np.array([1.0, 0.5]), 7, r0=0)
    part.seed_couplings(p)
    assert (part.couplings() == o.couplings()[:8]).all()


def test_trajectory_with_seeded_couplings_keeps_energy_bookkeeping():
    o = Oracle(4, 6, 5, np.linspace(1.5, 0.5, 6), 3, check=True)
    o.seed_couplings(0.8)
    o.sweep(40, 1)
    assert o.check_failures() == 0
