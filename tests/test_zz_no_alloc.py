"""ea_overlap_static (include/ea.h): the overlap call that allocates nothing -- its device scratch is
a fixed file-scope array of the library -- against ea_overlap on the same state, two calls in a row
(the array keeps the first call's contents), plus the size limit.  Integer work: equality.  Named
test_zz_* so that pytest collects it last."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_overlap_static_matches_overlap_twice_and_rejects_oversize():
    from paper_1311_5582_b200 import EA, EAError
    L, nT, R = 8, 6, 70
    g = EA(L, nT, R, np.linspace(1.4, 0.5, nT), 2024)
    g.sweep(5, 1)
    rng = np.random.default_rng(7)
    first = np.stack([rng.integers(0, R, 300), rng.integers(-1, R, 300)], axis=1).astype(np.int32)
    a = g.overlap_static(first)
    assert (a == g.overlap(first)).all()
    assert np.abs(a).max() <= L ** 3 and (a[first[:, 0] == first[:, 1]] == L ** 3).all()
    # second call: fewer pairs, other values, after more sweeps -- stale contents must not leak
    g.sweep(3, 1)
    second = np.array([[R - 1, 0], [5, -1], [33, 64], [2, 2], [69, 31]], dtype=np.int32)
    b = g.overlap_static(second)
    assert (b == g.overlap(second)).all()
    assert (g.overlap_static(first) == g.overlap(first)).all()
    # the limit: n_pairs * (2 + n_temps) <= 65536 32-bit words
    ok = np.zeros((65536 // (2 + nT), 2), dtype=np.int32)
    assert (g.overlap_static(ok) == L ** 3).all()
    launches = g.launch_count()
    with pytest.raises(EAError, match="EA_OVERLAP_STATIC_MAX_INT32"):
        g.overlap_static(np.zeros((65536 // (2 + nT) + 1, 2), dtype=np.int32))
    assert g.launch_count() == launches                       # rejected before any launch
    assert g.overlap_static(np.zeros((0, 2), dtype=np.int32)).shape == (0, nT)
    g.destroy()
