"""Pins for the oracle's second draw convention (R24): the paper's own
multispin coding puts the temperature replicas of ONE realization into a word and gives every
replica its own random number (PAPER.md:87, :91 Figure 3, :186, :281).  In the oracle that is
`set_draw_mode(1)`: one Philox draw per (site, realization, slot) instead of one per
(site, word, slot).  Expected values come from brute force / closed forms written in the tests
(the exact 256-state sweep matrix and its helpers live in test_oracle_chain.py), never from the
oracle.
"""
import numpy as np

from ea_inputs import CONFIGS, betas_for, random_pm1
from oracle import Oracle, philox4x32_10
from test_oracle_chain import H_numpy, L2_TS, _cesaro, _sweep_matrix, _time_average


def _mk(L, nT, R, betas, seed, r0=0, **kw):
    o = Oracle(L, nT, R, betas, seed, r0=r0, **kw)
    o.set_draw_mode(1)
    return o


def test_mode_switch_and_default():
    o = Oracle(4, 2, 3, np.array([1.0, 0.5]), 3)
    assert o.draw_mode() == 0
    o.set_draw_mode(1)
    assert o.draw_mode() == 1
    try:
        o.set_draw_mode(2)
        assert False
    except ValueError:
        pass


def test_first_flip_decisions_follow_the_counter_convention():
    """One half-sweep by hand: parity-0 sites of every (r, k) flip iff
    PX(0, q, r0 + r, (6<<16)|k)[l] < acc[tau][n_sat], with n_sat from a numpy Hamiltonian."""
    L, nT, R, seed, r0 = 4, 3, 5, 0x1234567890ABCDEF, 64
    betas = np.array([1.2, 0.8, 0.3])
    o = _mk(L, nT, R, betas, seed, r0=r0)
    J, s0 = o.couplings(), o.spins_by_slot().copy()
    acc, _ = o.tables()
    k0, k1 = seed & 0xFFFFFFFF, seed >> 32
    expect = s0.copy()
    for r in range(R):
        for k in range(nT):
            H0 = H_numpy(s0[r, k], J[r], L)
            for i in range(L ** 3):
                x, y, z = i % L, (i // L) % L, i // (L * L)
                if (x + y + z) & 1:
                    continue
                f = s0[r, k].copy(); f[i] = -f[i]
                c = (H_numpy(f, J[r], L) - H0 + 12) // 4          # dE = 4 n_sat - 12
                j = (x >> 1) + (L // 2) * (y + L * z)
                u = philox4x32_10(0, j >> 2, r0 + r, (6 << 16) | k, k0, k1)[j & 3]
                if u < int(acc[k, c]):                           # identity permutation at the start
                    expect[r, k, i] = -s0[r, k, i]
    # parity-0 sites do not interact, so their decisions all refer to the start state, and the
    # parity-1 half of the sweep leaves them alone: compare the even sites after one full sweep
    o.sweep(1, 0)
    got = o.spins_by_slot()
    even = np.array([((i % L) + (i // L) % L + i // (L * L)) % 2 == 0 for i in range(L ** 3)])
    assert (got[:, :, even] == expect[:, :, even]).all()


def test_realizations_are_independent_of_their_neighbours_in_a_word():
    # with per-realization draws ANY subset of realizations reproduces itself (r0 multiple of 32
    # is an API rule, so shift by 32), and two realizations of one word no longer share draws
    b = betas_for(CONFIGS[1])
    full = _mk(4, 16, 40, b, 3)
    full.sweep(9, 1)
    part = _mk(4, 16, 8, b, 3, r0=32)
    part.sweep(9, 1)
    assert (part.spins_by_slot() == full.spins_by_slot()[32:]).all()
    assert (part.energy() == full.energy()[32:]).all()
    shared = Oracle(4, 16, 40, b, 3)
    shared.sweep(9, 1)
    assert (shared.spins_by_slot() != full.spins_by_slot()).any()


def test_incremental_energy_composition_and_beta_zero():
    cfg = CONFIGS[1]
    o = _mk(cfg.L, cfg.n_temps, 6, betas_for(cfg), cfg.seed, check=True)
    o.sweep(150, 1)
    assert o.check_failures() == 0
    s, J, E = o.spins_by_slot(), o.couplings(), o.energy_by_slot()
    for r in range(o.R):
        for k in range(0, o.nT, 5):
            assert E[r, k] == H_numpy(s[r, k], J[r], cfg.L)
    a = _mk(4, 5, 7, np.linspace(1.5, 0.4, 5), 8); a.sweep(7, 2); a.sweep(6, 2)
    c = _mk(4, 5, 7, np.linspace(1.5, 0.4, 5), 8); c.sweep(13, 2)
    assert (a.spins_by_slot() == c.spins_by_slot()).all() and (a.perm()[0] == c.perm()[0]).all()
    z = _mk(4, 3, 33, np.zeros(3), 9)
    s0 = z.spins_by_slot()
    z.sweep(1, 1)
    cn = z.counters()
    assert cn["accepted"] == cn["attempts"] == 64 * 3 * 33 and cn["swap_accepted"] == cn["swap_attempts"]
    assert (z.spins_by_slot() == -s0).all()


def test_gauge_covariance_bit_exact():
    L, nT, R, N = 4, 6, 3, 64
    b = betas_for(CONFIGS[1])[:nT]
    a, g = _mk(L, nT, R, b, 21), _mk(L, nT, R, b, 21)
    eps = random_pm1((R, N), 99)
    J = a.couplings()
    Jg = J.copy()
    e3 = eps.reshape(R, L, L, L)
    for d, ax in ((0, 3), (1, 2), (2, 1)):
        Jg[:, d] = (J[:, d].reshape(R, L, L, L) * e3 * np.roll(e3, -1, axis=ax)).reshape(R, N)
    g.set_couplings(Jg)
    g.set_spins(a.spins_by_slot() * eps[:, None, :])
    a.sweep(40, 1); g.sweep(40, 1)
    assert (a.spins_by_slot() * eps[:, None, :] == g.spins_by_slot()).all()
    assert (a.energy() == g.energy()).all() and (a.perm()[0] == g.perm()[0]).all()


def test_L2_chain_vs_exact_enumeration_with_and_without_pt():
    """Same Markov kernel as the first convention (the sweep matrix does not know where the
    uniform numbers come from): time averages of E against the exact 256-state Cesaro limit
    without PT, and against the canonical average with PT on the ergodic instances."""
    R = 6
    betas = 1.0 / L2_TS
    o = _mk(2, len(betas), R, betas, 78)
    J, s0 = o.couplings(), o.spins_by_slot()
    mean, err = _time_average(o, 16000, 40, 0)
    z = np.zeros((R, len(betas)))
    for r in range(R):
        for t, b in enumerate(betas):
            P, E, idx = _sweep_matrix(J[r], b)
            mu = _cesaro(P, idx[tuple(s0[r, t])])
            z[r, t] = (mean[r, t] - mu @ E) / max(err[r, t], 1e-3)
    assert (np.abs(z) < 4.0).all() and np.sqrt((z ** 2).mean()) < 1.5, z
    o = _mk(2, len(betas), R, betas, 79)
    J = o.couplings()
    o.sweep(500, 1)
    mean, err = _time_average(o, 16000, 40, 1)
    zs = []
    for r in range(R):
        ok, exact = True, []
        for b in betas:
            P, E, idx = _sweep_matrix(J[r], b)
            pi = np.exp(-b * (E - E.min())); pi /= pi.sum()
            A = np.stack([_cesaro(P, n, 10) for n in (0, 85, 170, 255)])
            ok &= np.abs(A @ E - pi @ E).max() < 2e-2
            exact.append(pi @ E)
        if ok:
            zs.append((mean[r] - np.array(exact)) / np.maximum(err[r], 1e-3))
    zs = np.array(zs)
    assert len(zs) >= 3 and (np.abs(zs) < 4.0).all() and np.sqrt((zs ** 2).mean()) < 1.5, zs
