"""Pins for the oracle's measurement layer (Fig. 20):
two-copy coupling set-up, exact integer moments of the overlap and of the energy, Binder ratio.

Expected values come from numpy over exported +-1 arrays (never from the oracle's own
overlap / energy routines), from closed forms, or from exact enumeration.
"""
from fractions import Fraction

import numpy as np

from ea_inputs import random_pm1
from oracle import Oracle, binder_ratio
from test_oracle_chain import H_numpy


def _q_numpy(s, ra, rb):
    """overlap by temperature index from s[r][t][site] (+-1): plain dot products."""
    a = s[ra].astype(np.int64)
    b = s[rb].astype(np.int64) if rb >= 0 else np.ones_like(a)
    return (a * b).sum(axis=1)


def test_pair_couplings_copies_first_half_and_recomputes_energies():
    L, nT, R = 4, 3, 64
    o = Oracle(L, nT, R, np.array([1.2, 0.9, 0.5]), 17)
    J0 = o.couplings()
    assert (J0[:32] != J0[32:]).any()
    assert o.pair_couplings() == 0
    J = o.couplings()
    assert (J[:32] == J0[:32]).all() and (J[32:] == J0[:32]).all()
    s = o.spins_by_slot()
    assert (s[:32] != s[32:]).any()          # the copies start from different spins
    E = o.energy_by_slot()
    for r in (0, 31, 32, 63):
        for k in range(nT):
            assert E[r, k] == H_numpy(s[r, k], J[r], L)


def test_moments_equal_numpy_recomputation_from_exported_spins():
    L, nT, R = 4, 4, 70                      # ragged: word 2 holds 6 realizations
    betas = 1.0 / np.array([0.8, 1.1, 1.5, 2.0])
    o = Oracle(L, nT, R, betas, 23)
    wp = [[0, 1], [1, 2], [2, -1], [0, 0]]
    rp = o.realization_pairs(wp)
    assert rp[1][5] == (37, 69) and rp[1][6] is None and rp[2][5] == (69, -1) and rp[2][6] is None
    acc = None
    exp = {k: np.zeros((len(wp), 32, nT), dtype=object) + 0 for k in ("q1", "q2", "q4")}
    e1 = np.zeros((R, nT), dtype=object) + 0
    e2 = np.zeros((R, nT), dtype=object) + 0
    n_meas = 6
    for m in range(n_meas):
        acc = o.measure(1, 3, 2, wp, acc)
        s = o.spins()                        # [r][t][site] by temperature index
        J = o.couplings()
        for p, row in enumerate(rp):
            for b, pr in enumerate(row):
                if pr is None:
                    continue
                q = _q_numpy(s, *pr)
                for t in range(nT):
                    v = int(q[t])
                    exp["q1"][p, b, t] += v
                    exp["q2"][p, b, t] += v ** 2
                    exp["q4"][p, b, t] += v ** 4
        for r in range(0, R, 7):
            for t in range(nT):
                e = H_numpy(s[r, t], J[r], L)
                e1[r, t] += e
                e2[r, t] += e * e
    assert acc["n"] == n_meas and o.counters()["sweeps"] == 3 * n_meas
    for k in ("q1", "q2", "q4"):
        assert (acc[k] == exp[k]).all(), k
    rows = np.arange(0, R, 7)
    assert (acc["e1"][rows] == e1[rows]).all() and (acc["e2"][rows] == e2[rows]).all()
    assert (acc["q1"][3, :, :] == n_meas * L ** 3).all()          # a realization with itself: q = N
    assert (acc["q1"][1, 6:, :] == 0).all() and not acc["valid"][1, 6:].any()
    # measure(2, ...) then measure(4, ...) == six single measurements (continuation)
    o2 = Oracle(L, nT, R, betas, 23)
    a2 = o2.measure(4, 3, 2, wp, o2.measure(2, 3, 2, wp))
    for k in ("q1", "q2", "q4", "e1", "e2"):
        assert (a2[k] == acc[k]).all(), k


def test_beta_zero_overlap_is_constant():
    """beta = 0: every sweep complements every configuration, so q(a, b) never changes and
    the magnetization alternates in sign: sum q^k = n q0^k, sum m = 0 for even n."""
    L, nT, R = 4, 2, 64
    o = Oracle(L, nT, R, np.zeros(nT), 5)
    s0 = o.spins()
    acc = o.measure(4, 1, 0, [[0, 1], [1, -1]])
    for b in (0, 13, 31):
        q0 = _q_numpy(s0, b, 32 + b)
        m0 = _q_numpy(s0, 32 + b, -1)
        for t in range(nT):
            assert acc["q1"][0, b, t] == 4 * int(q0[t])
            assert acc["q2"][0, b, t] == 4 * int(q0[t]) ** 2
            assert acc["q4"][0, b, t] == 4 * int(q0[t]) ** 4
            assert acc["q1"][1, b, t] == 0
            assert acc["q2"][1, b, t] == 4 * int(m0[t]) ** 2


def test_binder_of_all_256_states_of_the_2cube_is_one_over_N():
    """Exact enumeration: the 256 configurations of the 2^3 lattice against the all-up
    reference have the binomial moments [q^2] = N, [q^4] = 3N^2 - 2N, so g = 1/N = 0.125."""
    L, R = 2, 256
    o = Oracle(L, 1, R, np.array([1.0]), 3)
    s = np.array([[[1 if (r >> i) & 1 else -1 for i in range(8)]] for r in range(R)], dtype=np.int8)
    assert o.set_spins(s) == 0
    acc = o.measure(1, 0, 0, [[w, -1] for w in range(8)])
    assert acc["valid"].all() and acc["n"] == 1
    assert sum(int(v) for v in acc["q2"].ravel()) == 256 * 8
    assert sum(int(v) for v in acc["q4"].ravel()) == 256 * (3 * 64 - 16)
    assert sum(int(v) for v in acc["q1"].ravel()) == 0
    g = binder_ratio(acc)
    assert g.shape == (1,) and g[0] == 0.125


def test_binder_formula_on_synthetic_sums():
    rng = np.random.default_rng(0)
    P, nT, n = 3, 4, 50
    q = rng.integers(-64, 65, size=(n, P, 32, nT))
    valid = np.ones((P, 32), dtype=bool)
    valid[2, 20:] = False
    acc = {"n": n, "valid": valid,
           "q2": (q.astype(object) ** 2).sum(axis=0), "q4": (q.astype(object) ** 4).sum(axis=0)}
    g = binder_ratio(acc)
    qf = q.astype(np.float64)
    for t in range(nT):
        m2 = (qf[:, valid, t] ** 2).mean(axis=0).mean()
        m4 = (qf[:, valid, t] ** 4).mean(axis=0).mean()
        assert abs(g[t] - 0.5 * (3.0 - m4 / m2 ** 2)) < 1e-12
    # frozen copies: q = +-N every time -> g = 1 exactly; q = 0 -> undefined (NaN)
    one = {"n": 7, "valid": np.ones((1, 32), dtype=bool),
           "q2": np.full((1, 32, 2), 7 * 64 ** 2, dtype=object), "q4": np.full((1, 32, 2), 7 * 64 ** 4, dtype=object)}
    assert (binder_ratio(one) == 1.0).all()
    one["q2"][:, :, 1] = 0
    one["q4"][:, :, 1] = 0
    g = binder_ratio(one)
    assert g[0] == 1.0 and np.isnan(g[1])
    # a two-valued distribution, by hand: q in {1, 3} equally often: <q^2> = 5, <q^4> = 41
    two = {"n": 2, "valid": np.ones((1, 1), dtype=bool),
           "q2": np.array([[[10]]], dtype=object), "q4": np.array([[[82]]], dtype=object)}
    assert binder_ratio(two)[0] == float((3 - Fraction(41, 25)) / 2)


def test_round_trip_update_by_hand():
    """One replica (slot 0 of realization 0) walking 0 1 2 1 0 1 2 2 1 0 over three temperature
    indices completes two round trips; the other slots are parked in the middle."""
    from oracle import round_trip_update
    walk = [0, 1, 2, 1, 0, 1, 2, 2, 1, 0]
    label = np.zeros((1, 3), dtype=np.int8)
    trips = np.zeros(1, dtype=np.int64)
    seen = []
    for t in walk:
        round_trip_update(label, trips, np.array([[t, 1, 1]]))
        seen.append(int(trips[0]))
    assert seen == [0, 0, 0, 0, 1, 1, 1, 1, 1, 2]
    assert label[0, 1] == 0 and label[0, 2] == 0             # never touched an end
    # starting at the far end counts as well; starting at index 0 needs a visit to the far end first
    label[:] = 0; trips[:] = 0
    for t in (2, 1, 0, 0, 1, 2, 0):
        round_trip_update(label, trips, np.array([[t, 1, 1]]))
    assert trips[0] == 2


def test_round_trips_of_the_odd_even_transposition_network():
    """Equal betas: every swap is accepted (threshold 2^32), so parallel tempering is the
    odd-even transposition network: every replica moves one index per round and turns at the
    ends.  An independent simulation of that network gives the expected round-trip counts."""
    L, nT, R, rounds = 2, 6, 3, 61
    o = Oracle(L, nT, R, np.full(nT, 0.7), 9)
    acc = o.measure(rounds, 1, 1, [])
    assert o.counters()["swap_accepted"] == o.counters()["swap_attempts"] > 0
    pos = list(range(nT))                                    # pos[k] = temperature index of slot k
    label, trips = [0] * nT, 0
    for n in range(rounds):
        at = {t: k for k, t in enumerate(pos)}
        for t in range(n & 1, nT - 1, 2):                    # round n pairs (t, t+1), t = n & 1, ...
            a, b = at[t], at[t + 1]
            pos[a], pos[b] = t + 1, t
        for k in range(nT):
            if pos[k] == 0:
                trips += label[k] == 2
                label[k] = 1
            elif pos[k] == nT - 1:
                label[k] = 2
    assert trips > 0 and (acc["trips"] == trips).all()
    # without parallel tempering nobody moves
    o = Oracle(L, nT, R, 1.0 / np.linspace(0.5, 2.0, nT), 9)
    assert (o.measure(20, 1, 0, [])["trips"] == 0).all()


def test_plane_correlation_against_fourier_transform_and_closed_forms():
    """C(d) must reproduce |q~(k)|^2 summed over the three axes for every k = 2 pi m / L (a direct
    complex Fourier sum over sites, written here), sum to 3 q^2, and equal the closed forms of a
    uniform and of a striped configuration."""
    from oracle import plane_correlation
    rng = np.random.default_rng(4)
    for L in (2, 4, 6):
        N = L ** 3
        q = (2 * rng.integers(0, 2, N) - 1).astype(np.int64)
        C = plane_correlation(q, L)
        assert C.sum() == 3 * int(q.sum()) ** 2
        i = np.arange(N)
        coords = (i % L, (i // L) % L, i // (L * L))
        for m in range(L):
            k = 2 * np.pi * m / L
            direct = sum(abs((q * np.exp(1j * k * c)).sum()) ** 2 for c in coords)
            from_C = sum(np.cos(k * d) * C[d] for d in range(L))
            assert abs(direct - from_C) < 1e-6 * max(1.0, direct)
    L = 4
    N = L ** 3
    assert (plane_correlation(np.ones(N, dtype=np.int64), L) == 3 * L * L ** 4).all()
    x = np.arange(N) % L
    stripes = np.where(x < L // 2, 1, -1)                   # +1 for x < L/2: only the x planes are non-zero
    want = [L ** 4 * (L - 4 * min(d, L - d)) for d in range(L)]
    assert plane_correlation(stripes, L).tolist() == want


def test_measure_accumulates_plane_correlations_and_xi_formula():
    from oracle import correlation_length, plane_correlation
    L, nT, R = 4, 3, 64
    o = Oracle(L, nT, R, 1.0 / np.array([1.0, 2.0, 4.0]), 6)
    wp = [[0, 1], [1, -1]]
    acc = None
    exp = np.zeros((2, 32, nT, L), dtype=object) + 0
    for _ in range(3):
        acc = o.measure(1, 2, 1, wp, acc)
        s = o.spins().astype(np.int64)
        for b in (0, 7, 31):
            for t in range(nT):
                exp[0, b, t] += plane_correlation(s[b, t] * s[32 + b, t], L)
                exp[1, b, t] += plane_correlation(s[32 + b, t], L)
    for b in (0, 7, 31):
        assert (acc["corr"][:, b] == exp[:, b]).all()
    assert (acc["corr"].sum(axis=3) == 3 * acc["q2"]).all()              # sum_d C(d) = 3 q^2
    # xi from synthetic sums: C(d) = A + B cos(2 pi d / L) gives chi(0) = L A, chi(k_min) = L B / 2
    L2, A, B = 8, 1000, 600
    C = np.array([round(A + B * np.cos(2 * np.pi * d / L2)) for d in range(L2)], dtype=object)
    syn = {"n": 1, "valid": np.ones((1, 1), dtype=bool), "corr": C.reshape(1, 1, 1, L2)}
    chi0 = float(sum(C))
    chik = sum(np.cos(2 * np.pi * d / L2) * float(C[d]) for d in range(L2))
    want = np.sqrt(chi0 / chik - 1.0) / (2 * np.sin(np.pi / L2))
    assert abs(correlation_length(syn, L2)[0] - want) < 1e-12 * want
    assert abs(want - np.sqrt(L2 * A / (L2 * B / 2) - 1) / (2 * np.sin(np.pi / L2))) < 0.02 * want
    # a uniform overlap has no weight at k_min: xi undefined (NaN)
    uni = {"n": 1, "valid": np.ones((1, 1), dtype=bool), "corr": np.full((1, 1, 1, L2), 5, dtype=object)}
    assert np.isnan(correlation_length(uni, L2)[0])
