"""Physics check of the CUDA path at scale, against the one number of this kind the paper prints:
the curves of different lattice sizes for the ferromagnetic Ising model cross at 1/T = 0.2217,
T_c = 4.51 (Fig. 19).  All J = +1, magnetization moments from the measurement
series (all-up reference), Binder ratio g_L(T) = (3 - <m^4>/<m^2>^2)/2 for L = 8 and 16 on the
resident kernel with parallel tempering.  Realizations of one word share their random draws and
have identical couplings here, so they coalesce (R11): the independent samples are the
64 words."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _g_of_T(L, temps, sweeps, therm, seed):
    import __graft_entry__ as ge
    ge.build()
    from paper_1311_5582_b200 import EA
    R = 2048
    sim = EA(L, len(temps), R, 1.0 / temps, seed)
    sim.set_couplings(np.ones((R, 3, L ** 3), dtype=np.int8))
    assert sim.get_kernel() == 2
    sim.sweep(therm, 1)
    sim.measure_begin([[w, -1] for w in range(R // 32)])
    sim.measure(sweeps // 10, 10, 1)
    g = sim.get_binder()
    xi = sim.get_correlation_length()
    trips = sim.get_round_trips()
    sim.destroy()
    return g, xi, trips


def test_ferromagnet_binder_ratios_cross_near_4p51():
    temps = np.array([4.2, 4.3, 4.4, 4.5, 4.6, 4.7, 4.8])
    g8, xi8, trips8 = _g_of_T(8, temps, 60000, 10000, 3)
    g16, xi16, _ = _g_of_T(16, temps, 60000, 20000, 4)
    assert trips8.sum() > 0                                   # replicas do travel the ladder
    assert (np.diff(g8) < 0).all() and (np.diff(g16) < 0).all()      # order decreases with T
    d = g16 - g8
    assert d[0] > 0.01 and d[-1] < -0.01, (g8, g16)           # ordered side / disordered side
    i = int(np.where(d > 0)[0].max())                         # last temperature with g16 > g8
    Tc = temps[i] + (temps[i + 1] - temps[i]) * d[i] / (d[i] - d[i + 1])
    assert 4.40 < Tc < 4.62, (Tc, g8, g16)                   # paper: 1/T = 0.2217 -> 4.51
    # the paper's own figure: correlation length over L for different sizes crosses at T_c
    r8, r16 = xi8 / 8.0, xi16 / 16.0
    assert np.isfinite(r8).all() and np.isfinite(r16).all()
    assert (np.diff(r8) < 0).all() and (np.diff(r16) < 0).all()
    dx = r16 - r8
    assert dx[0] > 0 and dx[-1] < 0, (r8, r16)
    j = int(np.where(dx > 0)[0].max())
    Tx = temps[j] + (temps[j + 1] - temps[j]) * dx[j] / (dx[j] - dx[j + 1])
    assert 4.40 < Tx < 4.62, (Tx, r8, r16)
    print("crossings: Binder", Tc, "xi/L", Tx, "xi8/8", r8, "xi16/16", r16)
