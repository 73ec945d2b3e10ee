"""Pins for the oracle's Markov chain: local field, energy bookkeeping, Metropolis,
parallel tempering (readings R1-R6, R11).

All "expected" values come from brute force written here in plain Python/numpy over
+-1 arrays (never from oracle code), from closed forms, or from tests/golden/*.txt.
"""
import itertools
import os

import numpy as np
import pytest

from ea_inputs import CONFIGS, betas_for, random_couplings, random_pm1
from oracle import Oracle


def H_numpy(s, J, L):
    """-sum J s s over the 3 forward bonds of every site; s[N], J[3][N], site = x + L(y + L z)."""
    s3 = s.reshape(L, L, L).astype(np.int64)          # [z][y][x]
    J3 = J.reshape(3, L, L, L).astype(np.int64)
    H = 0
    for d, ax in ((0, 2), (1, 1), (2, 0)):
        H -= int((J3[d] * s3 * np.roll(s3, -1, axis=ax)).sum())
    return H


def test_energy_from_scratch_matches_numpy_roll():
    for L, R, nT in ((2, 3, 2), (4, 5, 3), (6, 2, 2)):
        o = Oracle(L, nT, R, np.linspace(1.0, 0.5, nT), 11)
        J = o.couplings()
        s = o.spins_by_slot()
        for r in range(R):
            for k in range(nT):
                assert o.energy_from_scratch(r, k) == H_numpy(s[r, k], J[r], L)
        E = o.energy()   # identity permutation at start
        assert E[0, 0] == H_numpy(s[0, 0], J[0], L)
        N = L ** 3
        assert ((E - 3 * N) % 2 == 0).all() and (np.abs(E) <= 3 * N).all()


def test_delta_E_is_4nsat_minus_12_by_flip_and_recompute():
    L, R, nT = 4, 2, 2
    o = Oracle(L, nT, R, np.array([1.0, 0.5]), 5)
    J = o.couplings()
    s = o.spins_by_slot()
    for r in range(R):
        for k in range(nT):
            H0 = H_numpy(s[r, k], J[r], L)
            for i in range(L ** 3):
                f = s[r, k].copy()
                f[i] = -f[i]
                c = o.n_sat(k, r, i)
                assert 0 <= c <= 6
                assert H_numpy(f, J[r], L) - H0 == 4 * c - 12
    # L = 2: the two neighbours along an axis coincide; both bond slots count
    o = Oracle(2, 1, 1, np.array([1.0]), 5)
    J, s = o.couplings()[0], o.spins_by_slot()[0, 0]
    H0 = H_numpy(s, J, 2)
    for i in range(8):
        f = s.copy(); f[i] = -f[i]
        assert H_numpy(f, J, 2) - H0 == 4 * o.n_sat(0, 0, i) - 12


def test_incremental_energy_equals_recomputed_every_sweep():
    for cid, ns in ((1, 200), (2, 3)):
        cfg = CONFIGS[cid]
        o = Oracle(cfg.L, cfg.n_temps, min(cfg.R, 8), betas_for(cfg), cfg.seed, check=True)
        o.sweep(ns, cfg.swap_interval)
        assert o.check_failures() == 0
        s, J, E = o.spins_by_slot(), o.couplings(), o.energy_by_slot()
        for r in range(o.R):
            for k in range(0, o.nT, 5):
                assert E[r, k] == H_numpy(s[r, k], J[r], cfg.L)


def test_beta_zero_accepts_everything():
    L, nT, R = 4, 3, 33
    o = Oracle(L, nT, R, np.zeros(nT), 9)
    s0 = o.spins_by_slot()
    o.sweep(1, 1)
    c = o.counters()
    assert c["accepted"] == c["attempts"] == L ** 3 * nT * R
    assert c["swap_accepted"] == c["swap_attempts"] == R * (nT // 2)
    assert (o.spins_by_slot() == -s0).all()          # every spin flipped exactly once
    o.sweep(1, 0)
    assert (o.spins_by_slot() == s0).all()


def test_gauge_covariance_bit_exact():
    # s_i -> eps_i s_i, J_ij -> eps_i J_ij eps_j leaves every n_sat, hence every decision,
    # unchanged: draws depend on position only.
    cfg = CONFIGS[1]
    L, nT, R, N = 4, 6, 3, 64
    b = betas_for(cfg)[:nT]
    a = Oracle(L, nT, R, b, 21)
    g = Oracle(L, nT, R, b, 21)
    eps = random_pm1((R, N), 99)
    J = a.couplings()
    Jg = J.copy()
    e3 = eps.reshape(R, L, L, L)
    for d, ax in ((0, 3), (1, 2), (2, 1)):
        Jg[:, d] = (J[:, d].reshape(R, L, L, L) * e3 * np.roll(e3, -1, axis=ax)).reshape(R, N)
    g.set_couplings(Jg)
    g.set_spins(a.spins_by_slot() * eps[:, None, :])
    assert (a.energy() == g.energy()).all()
    a.sweep(50, 1)
    g.sweep(50, 1)
    assert (a.spins_by_slot() * eps[:, None, :] == g.spins_by_slot()).all()
    assert (a.energy() == g.energy()).all()
    assert (a.perm()[0] == g.perm()[0]).all()


def test_sweep_composition_and_word_independence():
    cfg = CONFIGS[1]
    b = betas_for(cfg)
    a = Oracle(4, cfg.n_temps, 40, b, 3)
    a.sweep(7, 2); a.sweep(6, 2)
    c = Oracle(4, cfg.n_temps, 40, b, 3)
    c.sweep(13, 2)
    assert (a.spins_by_slot() == c.spins_by_slot()).all() and (a.perm()[0] == c.perm()[0]).all()
    # realizations 32..39 simulated alone (r0 = 32) reproduce word 1 of the big run
    d = Oracle(4, cfg.n_temps, 8, b, 3, r0=32)
    d.sweep(13, 2)
    assert (d.spins_by_slot() == c.spins_by_slot()[32:]).all()
    assert (d.energy() == c.energy()[32:]).all()


def _exact_mean_E(J, L, betas):
    N = L ** 3
    Es = np.array([H_numpy(np.array(cfgn, dtype=np.int8), J, L)
                   for cfgn in itertools.product((-1, 1), repeat=N)], dtype=np.float64)
    out = []
    for b in betas:
        w = np.exp(-b * (Es - Es.min()))
        out.append(float((w * Es).sum() / w.sum()))
    return np.array(out), Es


def test_L2_ferromagnet_density_of_states_golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "ferro_L2_dos.txt")
    dos, means = {}, {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        if f[0] == "T":
            means[float(f[1])] = float(f[2])
        else:
            dos[int(f[0])] = int(f[1])
    J = np.ones((3, 8), dtype=np.int8)
    Ts = sorted(means)
    exact, Es = _exact_mean_E(J, 2, [1.0 / T for T in Ts])
    vals, counts = np.unique(Es.astype(int), return_counts=True)
    assert dict(zip(vals.tolist(), counts.tolist())) == dos
    for T, e in zip(Ts, exact):
        assert abs(e - means[T]) < 1e-9
    # the oracle's Hamiltonian on the same instance
    o = Oracle(2, 1, 1, np.array([1.0]), 1)
    o.set_couplings(J[None])
    for trial in range(20):
        s = random_pm1((1, 1, 8), trial)
        o.set_spins(s)
        assert o.energy()[0, 0] == H_numpy(s[0, 0], J, 2)


def _sweep_matrix(J, beta, L=2):
    """Exact one-sweep transition matrix of the paper's chain on the 2^3 lattice, from its
    definition: stage A then stage B, each site of the stage flips
    independently with P = min(1, exp(-beta dE))."""
    N = L ** 3
    states = [np.array(c, dtype=np.int8) for c in itertools.product((-1, 1), repeat=N)]
    idx = {tuple(s): n for n, s in enumerate(states)}
    E = np.array([H_numpy(s, J, L) for s in states], dtype=np.float64)

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


def _cesaro(P, start, doublings=13):
    """(1/n) sum_{k<n} delta_start P^k, n = 2^doublings: the long-run occupation of the
    (possibly reducible / periodic) chain started at `start`."""
    A = np.eye(P.shape[0]); Pn = P.copy()
    for _ in range(doublings):
        A = 0.5 * (A + Pn @ A)
        Pn = Pn @ Pn
    return A[start]


def _time_average(o, n_meas, nbin, swap_interval):
    series = np.zeros((n_meas, o.R, o.nT))
    for it in range(n_meas):
        o.sweep(1, swap_interval)
        series[it] = o.energy()
    bins = series.reshape(nbin, n_meas // nbin, o.R, o.nT).mean(axis=1)
    return bins.mean(axis=0), bins.std(axis=0, ddof=1) / np.sqrt(nbin)


L2_TS = np.array([1.0, 1.5, 2.5, 4.0])


def test_L2_chain_vs_exact_256_state_enumeration():
    """north_star: exact enumeration of the 2^3 lattice agrees with Monte Carlo <E>(T).
    Checkerboard Metropolis with P(dE = 0) = 1 is stationary for the Boltzmann weight but
    not always irreducible on 8 sites (free spins flip deterministically), so the sharp
    prediction is the Cesaro limit of the exact 256x256 sweep matrix from the oracle's own
    start state; where that limit equals the canonical average (most instances) the test
    is literally MC-vs-enumeration."""
    R = 6
    betas = 1.0 / L2_TS
    o = Oracle(2, len(betas), R, betas, 77)
    J, s0 = o.couplings(), o.spins_by_slot()
    mean, err = _time_average(o, 24000, 40, 0)
    n_canonical = 0
    z = np.zeros((R, len(betas)))
    for r in range(R):
        for t, b in enumerate(betas):
            P, E, idx = _sweep_matrix(J[r], b)
            pi = np.exp(-b * (E - E.min())); pi /= pi.sum()
            assert np.abs(pi @ P - pi).max() < 1e-14          # detailed balance holds
            mu = _cesaro(P, idx[tuple(s0[r, t])])
            z[r, t] = (mean[r, t] - mu @ E) / max(err[r, t], 1e-3)
            n_canonical += abs(mu @ E - pi @ E) < 5e-3      # Cesaro mean converges like 1/n
    assert (np.abs(z) < 4.0).all(), z      # fixed seed: deterministic; a 400k-sweep run gives rms 0.9
    assert np.sqrt((z ** 2).mean()) < 1.7, z   # realizations of a word share draws: z correlated
    assert n_canonical >= 16                                   # of 24 (instance, T) cases


def test_L2_with_pt_matches_canonical_average():
    # with vs without parallel tempering must agree on <E>(T)
    R = 6
    betas = 1.0 / L2_TS
    o = Oracle(2, len(betas), R, betas, 77)
    J = o.couplings()
    o.sweep(500, 1)
    mean, err = _time_average(o, 24000, 40, 1)
    c = o.counters()
    assert 0 < c["swap_accepted"] < c["swap_attempts"]
    zs = []
    for r in range(R):
        ok = True
        exact = []
        for b in betas:
            P, E, idx = _sweep_matrix(J[r], b)
            pi = np.exp(-b * (E - E.min())); pi /= pi.sum()
            # instance usable if every start state has the canonical long-run energy
            A = np.stack([_cesaro(P, n, 10) for n in (0, 85, 170, 255)])
            ok &= np.abs(A @ E - pi @ E).max() < 2e-2
            exact.append(pi @ E)
        if ok:
            zs.append((mean[r] - np.array(exact)) / np.maximum(err[r], 1e-3))
    assert len(zs) >= 3
    zs = np.array(zs)
    assert (np.abs(zs) < 4.0).all() and np.sqrt((zs ** 2).mean()) < 1.7, zs


def test_pt_bookkeeping():
    cfg = CONFIGS[1]
    o = Oracle(cfg.L, cfg.n_temps, 5, betas_for(cfg), cfg.seed)
    for it in range(40):
        o.sweep(1, 0)
        Eslot_before = o.energy_by_slot().copy()
        s_before = o.spins_by_slot().copy()
        # a sweep with swap_interval=1 = sweep + swap; isolate the swap by comparing slots
        o.sweep(1, 1)
        tau, sigma = o.perm()
        for r in range(o.R):
            assert sorted(tau[r]) == list(range(o.nT))
            assert (tau[r][sigma[r]] == np.arange(o.nT)).all()     # inverse permutations
        assert (o.energy() == np.take_along_axis(o.energy_by_slot(), sigma, axis=1)).all()
    assert o.counters()["swap_rounds"] == 40
    # alternating even/odd pairs: after one round from identity only pairs (0,1),(2,3).. move
    o = Oracle(cfg.L, cfg.n_temps, 5, np.zeros(cfg.n_temps), cfg.seed)
    o.sweep(1, 1)
    tau, _ = o.perm()
    assert (tau[0] == np.arange(cfg.n_temps) ^ 1).all()
    o.sweep(1, 1)   # round 1: pairs (1,2),(3,4),...
    _, sigma = o.perm()
    exp = np.arange(cfg.n_temps) ^ 1
    for t in range(1, cfg.n_temps - 1, 2):
        exp[t], exp[t + 1] = exp[t + 1], exp[t]
    assert (sigma[0] == exp).all()


def test_overlap_identities():
    cfg = CONFIGS[1]
    o = Oracle(4, cfg.n_temps, 4, betas_for(cfg), 8)
    o.sweep(30, 1)
    N = 64
    Q = o.overlap([[0, 0], [0, 1], [1, 0], [2, -1]])
    assert (Q[0] == N).all() and (Q[1] == Q[2]).all() and ((Q - N) % 2 == 0).all()
    s = o.spins()   # by temperature index
    assert (Q[1] == (s[0].astype(int) * s[1]).sum(axis=1)).all()
    assert (Q[3] == s[2].astype(int).sum(axis=1)).all()


def test_ferromagnet_binder_crossing_near_4p51():
    # all J = +1: 3D Ising; Binder cumulants of L = 4 and L = 8 cross near T_c = 4.5115
    # (the paper prints 1/T = 0.2217).  One sample per word (R = 1): copies
    # with identical J in one word share draws and coalesce (R11).
    Ts = np.array([4.0, 4.25, 4.5, 4.75, 5.0])
    U = {}
    for L, nsw in ((4, 60000), (8, 16000)):
        o = Oracle(L, len(Ts), 1, 1.0 / Ts, 4242 + L)
        o.set_couplings(np.ones((1, 3, L ** 3), dtype=np.int8))
        o.sweep(1000, 0)
        m2 = np.zeros(len(Ts)); m4 = np.zeros(len(Ts))
        chunk = 4
        for it in range(nsw // chunk):
            o.sweep(chunk, 0)
            m = o.overlap([[0, -1]])[0] / float(L ** 3)
            m2 += m ** 2; m4 += m ** 4
        n = nsw // chunk
        U[L] = 1.0 - (m4 / n) / (3.0 * (m2 / n) ** 2)
    d = U[8] - U[4]
    assert d[0] > 0.01 and d[-1] < -0.01, (U, d)        # ordered side / disordered side
    i = int(np.nonzero(d > 0)[0].max())
    Tx = Ts[i] + (Ts[i + 1] - Ts[i]) * d[i] / (d[i] - d[i + 1])
    assert 4.25 <= Tx <= 4.8, (Tx, U)


def test_checkpoint_resume_continues_the_same_trajectory():
    """A run interrupted at sweep a and resumed from (spins by slot, tau, counters) in a fresh
    object equals the uninterrupted run: the state is exactly that tuple."""
    L, nT, R = 4, 5, 37
    betas = 1.0 / np.geomspace(0.7, 2.5, nT)
    a = Oracle(L, nT, R, betas, 15)
    a.sweep(7, 2)                                 # ends between two swap rounds (round parity matters)
    c = a.counters()
    b = Oracle(L, nT, R, betas, 99)               # another seed: nothing may leak from create
    b.set_couplings(a.couplings())
    with pytest.raises(ValueError):
        bad = a.perm()[0].copy(); bad[3, 0] = bad[3, 1]
        b.set_state(a.spins_by_slot(), bad, c["sweeps"], c["swap_rounds"])
    # the draws are keyed by the seed: resume needs the same seed
    b = Oracle(L, nT, R, betas, 15)
    b.set_couplings(a.couplings())
    b.set_state(a.spins_by_slot(), a.perm()[0], c["sweeps"], c["swap_rounds"])
    assert (b.energy() == a.energy()).all() and (b.perm()[1] == a.perm()[1]).all()
    a.sweep(9, 2); b.sweep(9, 2)
    assert (a.spins_by_slot() == b.spins_by_slot()).all()
    assert (a.perm()[0] == b.perm()[0]).all() and (a.energy() == b.energy()).all()
    ref = Oracle(L, nT, R, betas, 15)
    ref.sweep(16, 2)
    assert (ref.spins_by_slot() == b.spins_by_slot()).all() and (ref.perm()[0] == b.perm()[0]).all()
    assert b.counters()["sweeps"] == 16 and b.counters()["swap_rounds"] == 8
