#!/usr/bin/env python
"""Convergence of the Binder ratio with and without parallel tempering (the experiment of the
paper's Fig. 21: 8^3 sites, 1/T = 2.0), through the library's measurement series.

Two copies of every disorder realization (ea_pair_couplings), overlap moments accumulated on the
device (ea_measure) in time windows [2^k, 2^(k+1)) sweeps; g = (3 - [<q^4>]/[<q^2>]^2)/2 at the
coldest temperature, averaged over the realization pairs.  With PT the windows settle on one
value; without PT the cold replicas are frozen and g drifts for orders of magnitude longer.

  python -m paper_1311_5582_b200.examples.binder_convergence [--L 8] [--pairs 1024] [--max-log2 20]
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))


def ladder(n_temps, t_min, t_max):
    k = np.arange(n_temps, dtype=np.float64)
    T = t_min * (t_max / t_min) ** (k / max(n_temps - 1, 1))
    T[0], T[-1] = t_min, (t_max if n_temps > 1 else t_min)
    return T


def run(L=8, pairs=1024, n_temps=16, t_min=0.5, t_max=2.0, max_log2=16, min_log2=6, seed=21,
        measure_every=8, swap_interval=1):
    """Returns (windows, g) with g[w][t] = Binder ratio by temperature index in window w."""
    from paper_1311_5582_b200 import EA
    R = 2 * pairs
    assert R % 64 == 0
    sim = EA(L, n_temps, R, 1.0 / ladder(n_temps, t_min, t_max), seed)
    sim.pair_couplings()
    W = sim.W
    word_pairs = [[w, w + W // 2] for w in range(W // 2)]
    sim.sweep(1 << min_log2, swap_interval)
    windows, out = [], []
    for k in range(min_log2, max_log2):
        n = 1 << k                                   # sweeps in the window [2^k, 2^(k+1))
        every = min(measure_every, n)
        sim.measure_begin(word_pairs)
        sim.measure(n // every, every, swap_interval)
        out.append(sim.get_binder())
        windows.append((n, 2 * n))
    sim.destroy()
    return windows, np.array(out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, default=8)
    ap.add_argument("--pairs", type=int, default=1024)
    ap.add_argument("--n-temps", type=int, default=16)
    ap.add_argument("--max-log2", type=int, default=20)
    a = ap.parse_args()
    res = {}
    for name, swap in (("with PT", 1), ("without PT", 0)):
        res[name] = run(L=a.L, pairs=a.pairs, n_temps=a.n_temps, max_log2=a.max_log2, swap_interval=swap)
    T = ladder(a.n_temps, 0.5, 2.0)
    print(f"# Binder ratio g at T = {T[0]:.3f} (1/T = {1 / T[0]:.2f}), L = {a.L}, {a.pairs} realization pairs")
    print("# window (sweeps)        with PT   without PT")
    for (w, g1), (_, g0) in zip(zip(*res["with PT"]), zip(*res["without PT"])):
        print(f"[{w[0]:8d}, {w[1]:8d})   {g1[0]:8.4f}   {g0[0]:8.4f}")
    print("# g by temperature in the last window, with PT:")
    print("# T: " + " ".join(f"{t:.3f}" for t in T))
    print("# g: " + " ".join(f"{g:.3f}" for g in res["with PT"][1][-1]))


if __name__ == "__main__":
    main()
