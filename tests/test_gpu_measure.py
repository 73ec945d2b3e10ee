"""GPU parity of the measurement series: coupling export, two-copy
set-up, integer moments of overlap and energy, Binder ratio -- CUDA path through the C ABI
against the CPU oracle on the same seeded inputs.  Integers bit-exact; the Binder ratio (the
one double-valued observable) within 1e-12 relative (north_star)."""
import numpy as np
import pytest

from ea_inputs import random_couplings, temperature_ladder

pytestmark = pytest.mark.gpu


def _mods():
    import __graft_entry__ as ge
    ge.build()
    import paper_1311_5582_b200 as pkg
    from oracle import Oracle, binder_ratio
    return pkg, Oracle, binder_ratio


def _moments_as_ints(m):
    """binding layout -> Python-int arrays like the oracle's."""
    q4 = m["q4"][..., 0].astype(object) + m["q4"][..., 1].astype(object) * (1 << 64)
    return {"n": m["n"], "q1": m["q1"].astype(object), "q2": m["q2"].astype(object), "q4": q4,
            "e1": m["e1"].astype(object), "e2": m["e2"].astype(object)}


def _compare(g, acc, binder_ratio):
    m = _moments_as_ints(g.get_moments())
    assert m["n"] == acc["n"]
    for k in ("q1", "q2", "q4", "e1", "e2"):
        assert (m[k] == acc[k]).all(), k
    assert (g.get_correlation().astype(object) == acc["corr"]).all(), "plane correlations"
    from oracle import correlation_length
    gx, ox = g.get_correlation_length(), correlation_length(acc, g.L)
    assert (np.isnan(gx) == np.isnan(ox)).all(), (gx, ox)
    okx = ~np.isnan(ox)
    assert (np.abs(gx[okx] - ox[okx]) <= 1e-12 * np.abs(ox[okx])).all(), (gx, ox)
    if "trips" in acc:
        assert (g.get_round_trips().astype(np.int64) == acc["trips"]).all(), "round trips"
    gb, ob = g.get_binder(), binder_ratio(acc)
    assert (np.isnan(gb) == np.isnan(ob)).all()
    ok = ~np.isnan(ob)
    assert (np.abs(gb[ok] - ob[ok]) <= 1e-12 * np.abs(ob[ok])).all(), (gb, ob)


@pytest.mark.parametrize("L,nT,R,kernel,wp,n_meas,between,swap", [
    (4, 5, 70, 1, [[0, 1], [1, 2], [2, -1], [0, 0]], 5, 3, 2),      # generic, ragged R, odd n_T
    (8, 8, 128, 2, [[0, 2], [1, 3], [3, -1]], 6, 4, 1),              # resident
    (16, 6, 64, 2, [[0, 1]], 3, 2, 1),                               # resident, L = 16
    (16, 4, 64, 3, [[0, 1], [1, -1]], 2, 2, 1),                      # tiled
    (32, 4, 64, 4, [[0, 1]], 2, 1, 1),                               # stream
    (6, 3, 40, 0, [[0, 1], [1, 0]], 4, 1, 0),                        # no PT, L = 6
    (12, 3, 64, 0, [[0, 1], [1, -1]], 2, 2, 1),                      # L = 12: 8 threads per plane, 36 planes
    (64, 2, 64, 0, [[0, 1]], 1, 1, 1),                               # L = 64: correlations without staging
    (4, 64, 64, 0, [[1, 0]], 2, 1, 1),                               # 64 temperatures: eight gather groups
])
def test_moments_and_binder_match_oracle(L, nT, R, kernel, wp, n_meas, between, swap):
    pkg, Oracle, binder_ratio = _mods()
    betas = 1.0 / temperature_ladder(nT, 0.8, 2.0)
    g = pkg.EA(L, nT, R, betas, 31, kernel=kernel)
    o = Oracle(L, nT, R, betas, 31)
    if R % 64 == 0:
        g.pair_couplings()
        o.pair_couplings()
        assert (g.get_couplings() == o.couplings()).all()
        assert (g.energy() == o.energy()).all()
    g.measure_begin(wp)
    g.measure(n_meas, between, swap)
    acc = o.measure(n_meas, between, swap, wp)
    _compare(g, acc, binder_ratio)
    # continue the same series, with a different cadence
    g.measure(2, 1, swap)
    acc = o.measure(2, 1, swap, wp, acc)
    _compare(g, acc, binder_ratio)
    # state after a measurement series is the plain trajectory
    assert (g.energy() == o.energy()).all()
    assert (g.get_state()["temp_of_slot"] == o.perm()[0]).all()
    # a new series starts from zero
    g.measure_begin(wp[:1])
    m = g.get_moments()
    assert m["n"] == 0 and not m["q2"].any() and not m["e2"].any()
    assert np.isnan(g.get_binder()).all()
    g.destroy()


def test_get_couplings_round_trip_and_seeded_values():
    pkg, Oracle, _ = _mods()
    L, nT, R = 6, 2, 45
    betas = np.array([1.0, 0.5])
    g = pkg.EA(L, nT, R, betas, 9)
    o = Oracle(L, nT, R, betas, 9)
    assert (g.get_couplings() == o.couplings()).all()        # seeded couplings
    J = random_couplings(R, L ** 3, seed=77)
    g.set_couplings(J)
    assert (g.get_couplings() == J).all()
    g.destroy()


def test_measure_zero_sweeps_between_repeats_the_same_sample():
    pkg, Oracle, binder_ratio = _mods()
    L, nT, R = 4, 3, 64
    betas = np.array([1.5, 1.0, 0.5])
    g = pkg.EA(L, nT, R, betas, 2)
    o = Oracle(L, nT, R, betas, 2)
    g.measure_begin([[0, 1]])
    g.measure(3, 0, 1)
    acc = o.measure(3, 0, 1, [[0, 1]])
    _compare(g, acc, binder_ratio)
    Q = g.overlap([[b, 32 + b] for b in range(32)])          # per-pair kernel against the word kernel
    m = g.get_moments()
    assert (m["q1"][0] == 3 * Q.astype(np.int64)).all()
    g.destroy()


def test_measure_errors_leave_state_unchanged():
    pkg, _, _ = _mods()
    g = pkg.EA(4, 2, 32, np.array([1.0, 0.5]), 1)
    with pytest.raises(pkg.EAError) as e:
        g.measure(1, 1, 1)                                   # no series yet
    assert e.value.code == -1
    with pytest.raises(pkg.EAError):
        g.measure_begin([[0, 1]])                            # W = 1: word 1 does not exist
    with pytest.raises(pkg.EAError):
        g.measure_begin([[-1, 0]])
    with pytest.raises(pkg.EAError):
        g.pair_couplings()                                   # R = 32 is not a multiple of 64
    g.measure_begin([[0, -1]])
    with pytest.raises(pkg.EAError) as e:
        g.measure(2, 2 ** 31, 1)                             # sweep counter would overflow
    assert e.value.code == -4
    st = g.get_state()
    assert st["sweeps"] == 0 and g.get_moments()["n"] == 0
    g.destroy()


def test_round_trips_match_oracle_and_the_transposition_network():
    pkg, Oracle, binder_ratio = _mods()
    # a ladder narrow enough for replicas to travel, measured after every sweep
    L, nT, R = 4, 6, 70
    betas = 1.0 / temperature_ladder(nT, 1.6, 2.4)
    g = pkg.EA(L, nT, R, betas, 12)
    o = Oracle(L, nT, R, betas, 12)
    g.measure_begin([])
    g.measure(300, 1, 1)
    acc = o.measure(300, 1, 1, [])
    trips = g.get_round_trips().astype(np.int64)
    assert (trips == acc["trips"]).all() and trips.sum() > 0
    assert np.isnan(g.get_binder()).all()                    # a series without pairs
    g.destroy()
    # equal betas: every swap accepted, 61 rounds of the odd-even transposition network
    g = pkg.EA(2, 6, 3, np.full(6, 0.7), 9, kernel=1)
    o = Oracle(2, 6, 3, np.full(6, 0.7), 9)
    g.measure_begin([])
    g.measure(61, 1, 1)
    assert (g.get_round_trips().astype(np.int64) == o.measure(61, 1, 1, [])["trips"]).all()
    g.destroy()


def test_binder_convergence_example_runs_and_orders_temperatures():
    """The Fig. 21 example in a short version: with PT the cold Binder ratio of the
    late window is large, the hot one small, and g falls with temperature."""
    _mods()
    from paper_1311_5582_b200.examples.binder_convergence import run
    windows, g = run(L=4, pairs=256, n_temps=8, max_log2=11, min_log2=8, swap_interval=1)
    assert windows == [(256, 512), (512, 1024), (1024, 2048)] and g.shape == (3, 8)
    assert np.isfinite(g).all() and (g <= 1.0).all()
    assert g[-1, 0] > 0.8 and g[-1, -1] < 0.5
    assert (np.diff(g[-1]) < 0.02).all()


def test_shard_measurements_and_field_equal_the_full_run():
    """A handle that simulates words 1..2 of a larger problem (first_realization = 32) gives those
    words' moments, correlations, round trips and field trajectory of the full run."""
    pkg, Oracle, _ = _mods()
    L, nT, R = 8, 6, 128
    betas = 1.0 / temperature_ladder(nT, 1.2, 2.4)
    full = pkg.EA(L, nT, R, betas, 9)
    part = pkg.EA(L, nT, 64, betas, 9, first_realization=32)
    for x in (full, part):
        x.set_field(1)
        x.sweep(3, 1)
        x.set_field(0)
    full.measure_begin([[1, 2], [2, -1]])
    part.measure_begin([[0, 1], [1, -1]])
    full.measure(40, 1, 1)
    part.measure(40, 1, 1)
    mf, mp = full.get_moments(), part.get_moments()
    for k in ("q1", "q2", "q4"):
        assert (mf[k] == mp[k]).all(), k
    assert (mf["e1"][32:96] == mp["e1"]).all() and (mf["e2"][32:96] == mp["e2"]).all()
    assert (full.get_correlation() == part.get_correlation()).all()
    assert (full.get_round_trips()[32:96] == part.get_round_trips()).all()
    assert full.get_round_trips()[32:96].sum() > 0
    ck = part.get_state()
    again = pkg.EA(L, nT, 64, betas, 9, first_realization=32)
    again.set_state(ck)
    again.sweep(5, 1); part.sweep(5, 1); full.sweep(5, 1)
    assert (again.get_state()["spin_words"] == part.get_state()["spin_words"]).all()
    assert (full.get_state()["spin_words"][:, 1:3] == part.get_state()["spin_words"]).all()
    for x in (full, part, again):
        x.destroy()


def test_c_example_runs_from_plain_c(tmp_path):
    """The C ABI from a C program (no Python in the process): builds, runs, prints a physical table:
    E/N near the +-J ground-state energy (about -1.79) at T = 0.5 and a Binder ratio that falls with T."""
    import subprocess
    from pathlib import Path
    pkg, _, _ = _mods()
    root = Path(__file__).resolve().parents[1]
    exe = tmp_path / "ea_demo"
    lib_dir = pkg.library_path().parent
    subprocess.check_call(["gcc", "-std=c99", str(root / "paper_1311_5582_b200" / "examples" / "ea_demo.c"),
                           "-I", str(root / "include"), "-L", str(lib_dir), "-lea_b200", "-lm",
                           f"-Wl,-rpath,{lib_dir}", "-o", str(exe)])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr
    rows = [[float(x) for x in line.split()] for line in out.stdout.splitlines()[1:]]
    assert len(rows) == 16 and abs(rows[0][0] - 0.5) < 1e-3 and abs(rows[-1][0] - 2.0) < 1e-3
    assert -1.80 < rows[0][1] < -1.74 and rows[0][2] > 0.85 and rows[-1][2] < 0.3
