"""Full-size parity of the section 8(f) extensions: config 4's full shape (2048 realizations x 24
temperatures, L = 16) in the launch configuration `bench.py --measure-every` / `--field` times,
checked on sampled realization words.  Words never interact,
so the oracle simulates just the sampled words (r0 = 32 w) and must reproduce them bit for bit."""
import numpy as np
import pytest

from ea_inputs import CONFIGS, betas_for
from util_pack import words_to_spins

pytestmark = pytest.mark.gpu


def _mods():
    import __graft_entry__ as ge
    ge.build()
    import paper_1311_5582_b200 as pkg
    from oracle import Oracle
    return pkg, Oracle


def _word_spins(st, w, L):
    return words_to_spins(st["spin_words"][:, w:w + 1], L, 32)      # [32][k][site]


def test_cfg4_two_copy_measurement_series_on_sampled_word_pairs():
    pkg, Oracle = _mods()
    cfg = CONFIGS[4]
    betas = betas_for(cfg)
    n_meas, between = 3, 4
    half = cfg.W // 2
    g = pkg.EA(cfg.L, cfg.n_temps, cfg.R, betas, cfg.seed)
    g.pair_couplings()
    wp = [[w, w + half] for w in range(half)]
    g.measure_begin(wp)
    g.measure(n_meas, between, cfg.swap_interval)
    m = g.get_moments()
    corr = g.get_correlation()
    from oracle import plane_correlation
    st = g.get_state()
    for w in (0, 13, 31):
        a = Oracle(cfg.L, cfg.n_temps, 32, betas, cfg.seed, r0=32 * w)
        b = Oracle(cfg.L, cfg.n_temps, 32, betas, cfg.seed, r0=32 * (w + half))
        b.set_couplings(a.couplings())                        # the second copy shares the disorder
        q1 = np.zeros((32, cfg.n_temps), dtype=np.int64)
        q2 = np.zeros_like(q1)
        q4 = np.zeros((32, cfg.n_temps), dtype=object) + 0
        e1 = np.zeros((64, cfg.n_temps), dtype=np.int64)
        e2 = np.zeros_like(e1)
        cd = np.zeros((32, cfg.n_temps, cfg.L), dtype=np.int64)
        for _ in range(n_meas):
            a.sweep(between, cfg.swap_interval)
            b.sweep(between, cfg.swap_interval)
            q = (a.spins().astype(np.int64) * b.spins().astype(np.int64)).sum(axis=2)   # [32][t]
            q1 += q; q2 += q * q; q4 += q.astype(object) ** 4
            sa, sb = a.spins().astype(np.int64), b.spins().astype(np.int64)
            for bit in (0, 17, 31):
                for t in (0, 11, cfg.n_temps - 1):
                    cd[bit, t] += plane_correlation(sa[bit, t] * sb[bit, t], cfg.L)
            E = np.concatenate([a.energy(), b.energy()]).astype(np.int64)
            e1 += E; e2 += E * E
        assert (m["q1"][w] == q1).all() and (m["q2"][w].astype(np.int64) == q2).all()
        assert (m["q4"][w][..., 0].astype(object) + m["q4"][w][..., 1].astype(object) * (1 << 64) == q4).all()
        for bit in (0, 17, 31):
            for t in (0, 11, cfg.n_temps - 1):
                assert (corr[w, bit, t] == cd[bit, t]).all()
        rows = np.r_[32 * w:32 * w + 32, 32 * (w + half):32 * (w + half) + 32]
        assert (m["e1"][rows] == e1).all() and (m["e2"][rows].astype(np.int64) == e2).all()
        assert (_word_spins(st, w, cfg.L) == a.spins_by_slot()).all()
        assert (_word_spins(st, w + half, cfg.L) == b.spins_by_slot()).all()
        assert (st["temp_of_slot"][32 * w:32 * w + 32] == a.perm()[0]).all()
    assert m["n"] == n_meas
    gb = g.get_binder()
    assert np.isfinite(gb).all() and (gb > -0.5).all() and (gb <= 1.0).all()
    g.destroy()


def test_cfg4_with_field_on_sampled_words():
    pkg, Oracle = _mods()
    cfg = CONFIGS[4]
    betas = betas_for(cfg)
    h, sweeps = 1, 6
    g = pkg.EA(cfg.L, cfg.n_temps, cfg.R, betas, cfg.seed)
    g.set_field(h)
    g.sweep(sweeps, cfg.swap_interval)
    st = g.get_state()
    E = g.energy()
    for w in (0, 40, 63):
        o = Oracle(cfg.L, cfg.n_temps, 32, betas, cfg.seed, r0=32 * w)
        o.set_field(h)
        o.sweep(sweeps, cfg.swap_interval)
        assert (_word_spins(st, w, cfg.L) == o.spins_by_slot()).all()
        assert (st["temp_of_slot"][32 * w:32 * w + 32] == o.perm()[0]).all()
        assert (E[32 * w:32 * w + 32] == o.energy()).all()
    g.destroy()


@pytest.mark.parametrize("L,nT,R,sweeps,words", [
    (16, 24, 8192, 12, (0, 100, 255)),      # four times config 4: 512 resident blocks on 148 SMs (several waves)
    (32, 32, 2048, 3, (0, 37, 63)),         # eight times config 5: the streaming kernel runs word group by word group
    (32, 32, 608, 2, (0, 9, 10, 18)),       # 19 words: two groups of 10 and 9 (first and last word of each)
])
def test_problems_larger_than_the_gpu_on_sampled_words(L, nT, R, sweeps, words):
    """More realization words than the device can hold at once: the launch runs in waves (resident)
    or word group by word group (streaming: words never interact, so each group runs all sweeps
    of the call on its own); sampled words must still follow the oracle bit for bit."""
    pkg, Oracle = _mods()
    from ea_inputs import temperature_ladder
    betas = 1.0 / temperature_ladder(nT, 0.8, 2.0)
    g = pkg.EA(L, nT, R, betas, 44)
    kernel = g.get_kernel()
    g.sweep(sweeps, 1)
    st = g.get_state()
    E = g.energy()
    for w in words:
        o = Oracle(L, nT, 32, betas, 44, r0=32 * w)
        o.sweep(sweeps, 1)
        assert (_word_spins(st, w, L) == o.spins_by_slot()).all(), (kernel, w)
        assert (st["temp_of_slot"][32 * w:32 * w + 32] == o.perm()[0]).all()
        assert (E[32 * w:32 * w + 32] == o.energy()).all()
    print("kernel used:", kernel)
    assert kernel == (2 if L == 16 else 4)
    g.destroy()
