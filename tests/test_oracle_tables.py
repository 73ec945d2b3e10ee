"""Pins for the oracle's threshold tables (R5, R7-R9).

- exact value: floor(2^32 e^x) evaluated with 60-digit mpmath arithmetic (an independent
  exp); the double-precision oracle may differ by one unit only where 2^32 e^x lies within
  double rounding error of an integer, so mismatches must be <= 1 in size and very rare;
- closed forms: beta = 0 -> 2^32 everywhere; n_sat <= 3 -> 2^32; monotone in T and n_sat;
  swap table 2^32 for m >= 0 (colder replica has the higher energy) when betas descend;
  symmetry acc[t][c] depends on beta*dE only;
- worked values of SURVEY.md section 8(c) (tests/golden/acc_thresholds_worked.txt).
"""
import os

import mpmath
import numpy as np

from ea_inputs import CONFIGS, betas_for
from oracle import Oracle

TWO32 = 1 << 32


def exact_threshold(x_mpf):
    if x_mpf >= 0:
        return TWO32
    return int(mpmath.floor(mpmath.ldexp(mpmath.exp(x_mpf), 32)))


def test_acc_table_exact_vs_mpmath():
    mpmath.mp.dps = 60
    worst = 0
    nbad = 0
    ntot = 0
    for cid in (1, 3, 4, 5):
        cfg = CONFIGS[cid]
        b = betas_for(cfg)
        o = Oracle(2, cfg.n_temps, 1, b, 1)
        acc, _ = o.tables()
        for t in range(cfg.n_temps):
            for c in range(7):
                x = -(mpmath.mpf(float(b[t])) * (4 * c - 12))
                e = exact_threshold(x)
                d = abs(int(acc[t, c]) - e)
                worst = max(worst, d)
                nbad += d != 0
                ntot += 1
    assert worst <= 1 and nbad <= max(1, ntot // 200), (worst, nbad, ntot)


def test_swap_table_exact_vs_mpmath_and_structure():
    mpmath.mp.dps = 60
    cfg = CONFIGS[1]
    b = betas_for(cfg)
    o = Oracle(cfg.L, cfg.n_temps, 1, b, 1)
    _, swp = o.tables()
    M = 3 * cfg.N // 2
    assert swp.shape == (cfg.n_temps - 1, 2 * M + 1)
    nbad = 0
    for t in range(cfg.n_temps - 1):
        db = mpmath.mpf(float(b[t] - b[t + 1]))  # the double difference is part of the definition
        for m in range(-M, M + 1, 1):
            e = exact_threshold(db * (4 * m))
            d = abs(int(swp[t, m + M]) - e)
            assert d <= 1
            nbad += d != 0
        # betas descend (index 0 coldest): E_a >= E_b always swaps
        assert (swp[t, M:] == TWO32).all()
        assert (np.diff(swp[t].astype(np.int64)) >= 0).all()
    assert nbad <= 3


def test_closed_forms():
    o = Oracle(2, 4, 1, np.zeros(4), 7)
    acc, swp = o.tables()
    assert (acc == TWO32).all() and (swp == TWO32).all()      # beta = 0: accept everything
    b = betas_for(CONFIGS[4])
    o = Oracle(2, len(b), 1, b, 7)
    acc, _ = o.tables()
    assert (acc[:, :4] == TWO32).all()                        # dE <= 0
    assert (acc[:, 4:] < TWO32).all()
    a = acc.astype(np.int64)
    assert (np.diff(a[:, 3:], axis=1) <= 0).all()             # harder flips less likely
    assert (np.diff(a, axis=0) >= 0).all()                    # hotter accepts more
    # depends on beta*dE only: beta, dE=8  ==  2*beta, dE=4
    o2 = Oracle(2, 2, 1, np.array([0.3, 0.6]), 7)
    acc2, _ = o2.tables()
    assert acc2[0, 5] == acc2[1, 4]


def test_worked_values():
    path = os.path.join(os.path.dirname(__file__), "golden", "acc_thresholds_worked.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    Ts = np.array([float(r[0]) for r in rows])
    o = Oracle(2, len(Ts), 1, 1.0 / Ts, 7)
    acc, _ = o.tables()
    for t, r in enumerate(rows):
        got = [int(acc[t, c]) for c in (0, 3, 4, 5, 6)]
        assert got == [int(v) for v in r[1:]], (r[0], got)
