"""Full-size parity: BASELINE.json's configs run at their full shape and length on the GPU (the
launch configuration bench.py times: AUTO kernel, all realizations) and compared with digests
the CPU oracle wrote ahead of time (tests/golden/make_golden.py, oracle only) for selected
realization words at sweep checkpoints 1, 10, 100, ... .  A digest covers the word's packed
spins, temperature permutation and integer energies, so equality is bit-exactness.
Which words / how many sweeps were affordable for the oracle is recorded in each JSON file.
"""
import glob
import json
import os

import numpy as np
import pytest

from ea_inputs import CONFIGS, betas_for
from util_pack import word_digest

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _files(cid):
    return sorted(glob.glob(os.path.join(GOLD, f"digests_cfg{cid}_w*.json")))


@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_full_config_matches_oracle_digests(cid):
    files = _files(cid)
    if not files:
        pytest.skip(f"no oracle digests for config {cid}")
    gold = [json.load(open(f)) for f in files]
    cps = sorted({int(c) for g in gold for c in g["checkpoints"]})
    cfg = CONFIGS[cid]
    from paper_1311_5582_b200 import EA
    sim = EA(cfg.L, cfg.n_temps, cfg.R, betas_for(cfg), cfg.seed)
    done, compared = 0, 0
    for cp in cps:
        sim.sweep(cp - done, cfg.swap_interval)
        done = cp
        st = sim.get_state()
        for g in gold:
            if str(cp) not in g["checkpoints"]:
                continue
            w, Rw = g["word"], g["realizations_in_word"]
            mask = np.uint32((1 << Rw) - 1)       # padding bits of a ragged word are not observable
            d = word_digest(st["spin_words"][:, w] & mask, st["temp_of_slot"][32 * w:32 * w + Rw],
                            st["energy_by_slot"][32 * w:32 * w + Rw])
            assert d == g["checkpoints"][str(cp)]["digest"], (cid, w, cp)
            E = sim.energy()[32 * w:32 * w + Rw]
            assert int(E.astype(np.int64).sum()) == g["checkpoints"][str(cp)]["E_sum"]
            compared += 1
    assert compared > 0
    sim.destroy()
