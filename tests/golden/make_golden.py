#!/usr/bin/env python
"""Write tests/golden/digests_cfg<N>_w<word>.json: sha256 digests of the CPU ORACLE's state
(packed spin words, temperature permutation, integer energies) at sweep checkpoints of
BASELINE.json's configs.  Calls only oracle/ (plus numpy layout helpers); never the CUDA path.

  python tests/golden/make_golden.py <config 1..5> <word> <max_sweeps> [state_dir]

With a state_dir the oracle's state (spins by slot as packed bits, temperature permutation,
counters) is saved there at every checkpoint and a later call resumes from it through eao_set_state
(whose interrupted-run == uninterrupted-run property tests/test_oracle_chain.py pins), so a
100000-sweep word (about 1.7 h of one core) survives an interruption.

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

CHECKPOINTS = [1, 10, 100, 200, 500, 1000, 2000, 5000] + list(range(10_000, 100_001, 10_000))


def main():
    cid, word, max_sweeps = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3])
    cfg = CONFIGS[cid]
    R = min(32, cfg.R - 32 * word)
    o = Oracle(cfg.L, cfg.n_temps, R, betas_for(cfg), cfg.seed, r0=32 * word)
    out = {"config": cid, "name": cfg.name, "word": word, "realizations_in_word": R,
           "swap_interval": cfg.swap_interval, "seed": cfg.seed, "checkpoints": {}}
    path = os.path.join(HERE, f"digests_cfg{cid}_w{word}.json")
    state_dir = sys.argv[4] if len(sys.argv) > 4 else None
    state_path = os.path.join(state_dir, f"state_cfg{cid}_w{word}.npz") if state_dir else None
    done = 0
    spent = 0.0
    if os.path.exists(path):                       # keep what an earlier call already wrote
        with open(path) as f:
            old = json.load(f)
        out["checkpoints"] = old["checkpoints"]
        spent = old.get("oracle_seconds", 0.0)
    if state_path and os.path.exists(state_path):
        st = np.load(state_path)
        bits = np.unpackbits(st["spin_bits"])[: R * cfg.n_temps * cfg.N].reshape(R, cfg.n_temps, cfg.N)
        o.set_state((2 * bits.astype(np.int8) - 1), st["tau"], int(st["sweeps"]), int(st["swap_rounds"]))
        done = int(st["sweeps"])
        print("resumed at sweep", done, flush=True)
    t0 = time.time() - (spent if done else 0.0)
    for cp in [c for c in CHECKPOINTS if done < c <= min(max_sweeps, cfg.sweeps)]:
        o.sweep(cp - done, cfg.swap_interval)
        done = cp
        if state_path:
            os.makedirs(state_dir, exist_ok=True)
            c = o.counters()
            np.savez(state_path + ".tmp.npz", spin_bits=np.packbits(o.spins_by_slot() > 0), tau=o.perm()[0],
                     sweeps=c["sweeps"], swap_rounds=c["swap_rounds"])
            os.replace(state_path + ".tmp.npz", state_path)
        words = spins_to_words(o.spins_by_slot(), cfg.L)[:, 0]
        tau, _ = o.perm()
        taup = np.zeros((32, cfg.n_temps), dtype=np.uint8); taup[:R] = tau
        Ep = np.zeros((32, cfg.n_temps), dtype=np.int32); Ep[:R] = o.energy_by_slot()
        new = {"digest": word_digest(words, taup[:R], Ep[:R]), "E_sum": int(o.energy().astype(np.int64).sum())}
        assert out["checkpoints"].get(str(cp), new) == new, f"checkpoint {cp}: recomputed digest differs from the stored one"
        out["checkpoints"][str(cp)] = new
        out["oracle_seconds"] = round(time.time() - t0, 1)
        with open(path + ".tmp", "w") as f:
            json.dump(out, f, indent=1)
        os.replace(path + ".tmp", path)
        print(cid, word, cp, out["checkpoints"][str(cp)], flush=True)


if __name__ == "__main__":
    main()
