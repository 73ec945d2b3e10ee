"""Pins for the oracle's external field h (Eq. 1; the 14-column table "7 local
energies x 2 spins"; R21).

H = -sum J s s + h sum s with integer h.  Expected values come from numpy Hamiltonians written
here, from exact enumeration of the 2^3 lattice, from closed forms, or from an exact symmetry.
"""
import itertools
import math

import numpy as np

from oracle import Oracle
from test_oracle_chain import H_numpy, _cesaro, _time_average


def H_field(s, J, L, h):
    return H_numpy(s, J, L) + h * int(s.astype(np.int64).sum())


def test_energy_and_delta_E_with_field_by_flip_and_recompute():
    for L, h in ((4, 1), (4, -3), (2, 2), (6, 7)):
        R, nT = 2, 2
        o = Oracle(L, nT, R, np.array([1.0, 0.5]), 5)
        o.set_field(h)
        assert o.field() == h
        J, s = o.couplings(), o.spins_by_slot()
        E = o.energy_by_slot()
        for r in range(R):
            for k in range(nT):
                H0 = H_field(s[r, k], J[r], L, h)
                assert E[r, k] == H0 == o.energy_from_scratch(r, k)
                for i in range(0, L ** 3, 3):
                    f = s[r, k].copy()
                    f[i] = -f[i]
                    c = o.n_sat(k, r, i)
                    assert H_field(f, J[r], L, h) - H0 == 4 * c - 12 - 2 * h * int(s[r, k, i])


def test_incremental_energy_equals_recomputed_with_field_and_pt():
    L, nT, R = 4, 6, 40
    betas = 1.0 / np.geomspace(0.6, 3.0, nT)
    for h in (1, -2, 5):
        o = Oracle(L, nT, R, betas, 21, check=True)
        o.set_field(h)
        o.sweep(30, 1)
        assert o.check_failures() == 0
        c = o.counters()
        assert 0 < c["accepted"] < c["attempts"] and 0 < c["swap_accepted"] < c["swap_attempts"]
        tau, sigma = o.perm()
        assert (np.take_along_axis(tau, sigma, axis=1) == np.arange(nT)).all()
        N = L ** 3
        assert ((o.energy() - (3 * N + h * N)) % 2 == 0).all()      # parity of H is fixed


def test_field_tables_closed_forms():
    L, nT, h = 2, 5, 3
    betas = 1.0 / np.array([0.5, 0.8, 1.3, 2.0, 3.5])
    o = Oracle(L, nT, 1, betas, 1)
    o.set_field(h)
    accf, swpf = o.field_tables()
    N, Mf = L ** 3, (3 + abs(h)) * L ** 3
    assert accf.shape == (nT, 7, 2) and swpf.shape == (nT - 1, 2 * Mf + 1)
    for t in range(nT):
        for c in range(7):
            for sp in (0, 1):
                dE = 4 * c - 12 - 2 * h * (2 * sp - 1)
                v = int(accf[t, c, sp])
                if dE <= 0:
                    assert v == 1 << 32
                else:
                    assert abs(v - math.floor(math.ldexp(math.exp(-betas[t] * dE), 32))) <= 1
    # monotone: hotter accepts more; more satisfied bonds accept less
    assert (np.diff(accf.astype(np.int64), axis=0) >= 0).all()
    assert (np.diff(accf.astype(np.int64), axis=1) <= 0).all()
    for t in range(nT - 1):
        db = betas[t] - betas[t + 1]
        for d2 in (-Mf, -17, -1, 0, 1, 9, Mf):
            v = int(swpf[t, d2 + Mf])
            x = db * (2 * d2)
            assert v == (1 << 32) if x >= 0 else abs(v - math.floor(math.ldexp(math.exp(x), 32))) <= 1
    # h = 0 restores the zero-field behaviour exactly
    a = Oracle(4, 3, 33, np.array([1.2, 0.9, 0.4]), 8)
    b = Oracle(4, 3, 33, np.array([1.2, 0.9, 0.4]), 8)
    a.set_field(4)
    a.set_field(0)
    a.sweep(12, 1)
    b.sweep(12, 1)
    assert (a.spins_by_slot() == b.spins_by_slot()).all() and (a.energy() == b.energy()).all()


def test_global_flip_symmetry_is_bit_exact():
    """(s, h) -> (-s, -h) leaves every dE unchanged and the draws depend on position only, so the
    two trajectories are complements of each other forever, with equal energies and swaps."""
    L, nT, R = 4, 5, 37
    betas = 1.0 / np.geomspace(0.7, 2.5, nT)
    a = Oracle(L, nT, R, betas, 13)
    b = Oracle(L, nT, R, betas, 13)
    b.set_spins(-a.spins_by_slot())
    a.set_field(2)
    b.set_field(-2)
    for _ in range(4):
        a.sweep(5, 1)
        b.sweep(5, 1)
        assert (a.spins_by_slot() == -b.spins_by_slot()).all()
        assert (a.energy_by_slot() == b.energy_by_slot()).all()
        assert (a.perm()[0] == b.perm()[0]).all()
    assert a.counters()["swap_accepted"] > 0


def test_strong_field_saturates_in_one_sweep():
    """h = -8 (H = ... + h sum s favours s = +1): a down spin always gains energy by flipping
    (dE = 4c - 28 < 0), an up spin loses at least 4; at T = 0.1 the threshold of dE >= 4 is
    floor(2^32 e^-40) = 0.  After one sweep every spin is up and stays up: m = N, exactly."""
    L, nT, R = 4, 2, 20
    o = Oracle(L, nT, R, np.array([10.0, 10.0]), 3)
    o.set_field(-8)
    o.sweep(1, 0)
    assert (o.spins_by_slot() == 1).all()
    o.sweep(3, 1)
    assert (o.spins_by_slot() == 1).all()
    J = o.couplings()
    assert o.energy()[0, 0] == -int(J[0].astype(np.int64).sum()) - 8 * L ** 3


def _sweep_matrix_field(J, beta, h, L=2):
    """Exact one-sweep transition matrix on the 2^3 lattice from the definition (stage A then
    stage B; P = min(1, exp(-beta dE))) with H = -sum J s s + h sum s."""
    N = L ** 3
    states = [np.array(c, dtype=np.int8) for c in itertools.product((-1, 1), repeat=N)]
    idx = {tuple(s): n for n, s in enumerate(states)}
    E = np.array([H_field(s, J, L, h) for s in states], dtype=np.float64)

    def stage(p):
        P = np.zeros((len(states),) * 2)
        sites = [i for i in range(N) if ((i & 1) + ((i >> 1) & 1) + ((i >> 2) & 1)) % 2 == p]
        for n, s in enumerate(states):
            q = []
            for i in sites:
                f = s.copy(); f[i] = -f[i]
                q.append(min(1.0, np.exp(-beta * (E[idx[tuple(f)]] - E[n]))))
            for mask in itertools.product((0, 1), repeat=len(sites)):
                f = s.copy(); pr = 1.0
                for m, i, qi in zip(mask, sites, q):
                    if m:
                        f[i] = -f[i]; pr *= qi
                    else:
                        pr *= 1.0 - qi
                if pr > 0.0:
                    P[n, idx[tuple(f)]] += pr
        return P

    return stage(0) @ stage(1), E, idx


def test_L2_chain_with_field_vs_exact_enumeration():
    """Odd h: dE = 4c - 12 -+ 2h is never 0, every flip probability is strictly inside (0, 1) or
    1 with a reverse < 1, the chain is ergodic, and the Monte Carlo <E>(T) must equal the
    canonical average over the 256 states (north_star's enumeration pin, now with a field);
    with and without parallel tempering."""
    R, h = 5, 1
    Ts = np.array([1.0, 1.6, 2.5, 4.0])
    betas = 1.0 / Ts
    exact = np.zeros((R, len(Ts)))
    o = Oracle(2, len(betas), R, betas, 41)
    o.set_field(h)
    J, s0 = o.couplings(), o.spins_by_slot()
    for r in range(R):
        for t, b in enumerate(betas):
            P, E, idx = _sweep_matrix_field(J[r], b, h)
            pi = np.exp(-b * (E - E.min())); pi /= pi.sum()
            assert np.abs(pi @ P - pi).max() < 1e-14              # Boltzmann is stationary
            mu = _cesaro(P, idx[tuple(s0[r, t])], doublings=17)
            assert abs(mu @ E - pi @ E) < 5e-3                      # and it is the long-run law
            exact[r, t] = pi @ E
    for swap_interval in (0, 1):
        o = Oracle(2, len(betas), R, betas, 41)
        o.set_field(h)
        o.sweep(200, swap_interval)
        mean, err = _time_average(o, 24000, 40, swap_interval)
        z = (mean - exact) / np.maximum(err, 1e-3)
        assert (np.abs(z) < 4.0).all() and np.sqrt((z ** 2).mean()) < 1.7, z
