"""Test-side layout helpers (numpy only; no method arithmetic)."""
import numpy as np


def checkerboard_maps(L):
    """site i = x + L(y + L z)  ->  (parity p, checkerboard index j)."""
    i = np.arange(L ** 3)
    x, y, z = i % L, (i // L) % L, i // (L * L)
    return (x + y + z) & 1, (x >> 1) + (L // 2) * (y + L * z)


def words_to_spins(words, L, R):
    """words[k][w][p][j] (uint32) -> s[r][k][site] in +-1 (by slot)."""
    nT, W = words.shape[:2]
    p, j = checkerboard_maps(L)
    per_site = words[:, :, p, j]                        # [k][w][site]
    bits = (per_site[..., None] >> np.arange(32, dtype=np.uint32)) & 1   # [k][w][site][b]
    s = bits.transpose(1, 3, 0, 2).reshape(W * 32, nT, L ** 3)[:R]
    return (2 * s.astype(np.int8) - 1).astype(np.int8)


def by_temperature(arr_by_slot, tau):
    """arr[r][k][...] by slot + tau[r][k] -> arr[r][t][...]."""
    sigma = np.argsort(tau, axis=1)
    idx = sigma.reshape(sigma.shape + (1,) * (arr_by_slot.ndim - 2))
    return np.take_along_axis(arr_by_slot, idx, axis=1)
