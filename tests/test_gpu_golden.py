"""Full-size parity: BASELINE.json's configs run at their full shape on the GPU (the launch
configuration bench.py times: AUTO kernel, all realizations) up to the last checkpoint the CPU
oracle has stored, and compared with the digests it wrote ahead of time
(tests/golden/make_golden.py, oracle only) for selected realization words at the checkpoints 1, 10,
100, 200, 500, 1000, 2000, 5000, 10^4, 2 10^4, ..., 10^5.  A digest covers the word's packed spins,
temperature permutation and integer energies, so equality is bit-exactness.  Coverage (recorded in
each JSON file, stated in DESIGN.md section 7): configs 1-3 every word to the config's full length;
config 4 words 0, 5, 20, 31, 40 and 63 to the full 10^5 sweeps; config 5 words 0,
3, 6 and 7 to the full 10^4 sweeps.  test_full_length_is_covered fails if a config's
longest stored checkpoint is shorter than the config."""
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


@pytest.mark.parametrize("cid", [1, 2, 3, 4, 5])
def test_full_length_is_covered(cid):
    gold = [json.load(open(f)) for f in _files(cid)]
    assert gold and max(int(c) for g in gold for c in g["checkpoints"]) == CONFIGS[cid].sweeps
