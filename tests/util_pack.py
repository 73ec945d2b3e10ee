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


def spins_to_words(s, L):
    """s[r][k][site] in +-1 (by slot) -> words[k][w][p][j] (uint32), padding bits 0."""
    R, nT, N = s.shape
    W = (R + 31) // 32
    p, j = checkerboard_maps(L)
    bits = np.zeros((W * 32, nT, N), dtype=np.uint32)
    bits[:R] = (s > 0)
    bits = bits.reshape(W, 32, nT, N)
    per_site = (bits << np.arange(32, dtype=np.uint32)[None, :, None, None]).sum(axis=1, dtype=np.uint32)  # [w][k][site]
    words = np.zeros((nT, W, 2, N // 2), dtype=np.uint32)
    words[:, :, p, j] = per_site.transpose(1, 0, 2)
    return words


def word_digest(spin_words_w, tau_w, E_w):
    """sha256 over one realization word: spin_words[:, w] ([nT][2][N/2] uint32), temp_of_slot and
    energy_by_slot of its 32 realizations ([32][nT])."""
    import hashlib
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(spin_words_w, dtype=np.uint32).tobytes())
    h.update(np.ascontiguousarray(tau_w, dtype=np.uint8).tobytes())
    h.update(np.ascontiguousarray(E_w, dtype=np.int32).tobytes())
    return h.hexdigest()
