#!/usr/bin/env python
"""Write tests/golden/digests_cfg<N>_w<word>.json: sha256 digests of the CPU ORACLE's state
(packed spin words, temperature permutation, integer energies) at sweep checkpoints of
BASELINE.json's configs.  Calls only oracle/ (plus numpy layout helpers); never the CUDA path.

  python tests/golden/make_golden.py <config 1..5> <word> <max_sweeps>

Realization words are independent, so a word simulated alone
with r0 = 32*word reproduces that word of the full run; the GPU test runs the whole config
and compares the same words.
"""
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import numpy as np  # noqa: E402

from ea_inputs import CONFIGS, betas_for  # noqa: E402
from oracle import Oracle  # noqa: E402
from util_pack import spins_to_words, word_digest  # noqa: E402

CHECKPOINTS = [1, 10, 100, 1000, 2000, 10_000, 100_000]


def main():
    cid, word, max_sweeps = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3])
    cfg = CONFIGS[cid]
    R = min(32, cfg.R - 32 * word)
    o = Oracle(cfg.L, cfg.n_temps, R, betas_for(cfg), cfg.seed, r0=32 * word)
    out = {"config": cid, "name": cfg.name, "word": word, "realizations_in_word": R,
           "swap_interval": cfg.swap_interval, "seed": cfg.seed, "checkpoints": {}}
    path = os.path.join(HERE, f"digests_cfg{cid}_w{word}.json")
    done = 0
    t0 = time.time()
    for cp in [c for c in CHECKPOINTS if c <= min(max_sweeps, cfg.sweeps)]:
        o.sweep(cp - done, cfg.swap_interval)
        done = cp
        words = spins_to_words(o.spins_by_slot(), cfg.L)[:, 0]
        tau, _ = o.perm()
        taup = np.zeros((32, cfg.n_temps), dtype=np.uint8); taup[:R] = tau
        Ep = np.zeros((32, cfg.n_temps), dtype=np.int32); Ep[:R] = o.energy_by_slot()
        out["checkpoints"][str(cp)] = {"digest": word_digest(words, taup[:R], Ep[:R]),
                                        "E_sum": int(o.energy().astype(np.int64).sum())}
        out["oracle_seconds"] = round(time.time() - t0, 1)
        with open(path + ".tmp", "w") as f:
            json.dump(out, f, indent=1)
        os.replace(path + ".tmp", path)
        print(cid, word, cp, out["checkpoints"][str(cp)], flush=True)


if __name__ == "__main__":
    main()
