"""ctypes loader for oracle/ea_oracle.c (the CPU oracle; test infrastructure only).

Argument marshalling only: every step of the method is in ea_oracle.c, where
each function cites the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from fractions import Fraction
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ea_oracle.c"
_LIB = _HERE / "libea_oracle.so"
_lib = None


def build_oracle(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain C, -O2, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off",
             "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build_oracle()
    lib = C.CDLL(str(_LIB))
    vp, i32, i64, u64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint64
    lib.eao_create.restype = vp
    lib.eao_create.argtypes = [i32, i32, i32, vp, u64, i32]
    lib.eao_destroy.argtypes = [vp]
    lib.eao_set_check.argtypes = [vp, i32]
    lib.eao_check_failures.restype = i64
    lib.eao_check_failures.argtypes = [vp]
    lib.eao_set_couplings.restype = i32
    lib.eao_set_couplings.argtypes = [vp, vp]
    lib.eao_set_spins.restype = i32
    lib.eao_set_spins.argtypes = [vp, vp]
    lib.eao_set_tables.argtypes = [vp, vp, vp]
    lib.eao_get_tables.argtypes = [vp, vp, vp]
    lib.eao_sweep.restype = i32
    lib.eao_sweep.argtypes = [vp, i64, i32]
    lib.eao_energy.argtypes = [vp, vp]
    lib.eao_overlap.restype = i32
    lib.eao_overlap.argtypes = [vp, vp, i32, vp]
    lib.eao_get_spins.argtypes = [vp, vp]
    lib.eao_get_spins_by_slot.argtypes = [vp, vp]
    lib.eao_get_couplings.argtypes = [vp, vp]
    lib.eao_get_perm.argtypes = [vp, vp, vp]
    lib.eao_get_energy_by_slot.argtypes = [vp, vp]
    lib.eao_get_counters.argtypes = [vp, vp, vp, vp]
    lib.eao_energy_from_scratch.restype = C.c_int32
    lib.eao_energy_from_scratch.argtypes = [vp, i32, i32]
    lib.eao_n_sat.restype = i32
    lib.eao_n_sat.argtypes = [vp, i32, i32, i32]
    lib.eao_philox4x32_10.argtypes = [C.c_uint32] * 6 + [vp]
    lib.eao_set_state.restype = i32
    lib.eao_set_state.argtypes = [vp, vp, vp, u64, u64]
    lib.eao_set_field.restype = i32
    lib.eao_set_field.argtypes = [vp, i32]
    lib.eao_seed_couplings.restype = i32
    lib.eao_seed_couplings.argtypes = [vp, C.c_double]
    lib.eao_set_draw_mode.restype = i32
    lib.eao_set_draw_mode.argtypes = [vp, i32]
    lib.eao_get_draw_mode.restype = i32
    lib.eao_get_draw_mode.argtypes = [vp]
    lib.eao_set_swap_mode.restype = i32
    lib.eao_set_swap_mode.argtypes = [vp, i32]
    lib.eao_get_swap_mode.restype = i32
    lib.eao_get_swap_mode.argtypes = [vp]
    lib.eao_get_field.restype = i32
    lib.eao_get_field.argtypes = [vp]
    lib.eao_get_field_tables.restype = i32
    lib.eao_get_field_tables.argtypes = [vp, vp, vp]
    _lib = lib
    return lib


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    out = (C.c_uint32 * 4)()
    _load().eao_philox4x32_10(c0, c1, c2, c3, k0, k1, out)
    return tuple(int(v) for v in out)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    """One EA problem on the CPU: L^3 sites, R realizations, n_temps replicas each."""

    def __init__(self, L, n_temps, R, betas, seed, r0=0, check=False):
        self.lib = _load()
        self.L, self.nT, self.R, self.N = int(L), int(n_temps), int(R), int(L) ** 3
        b = np.ascontiguousarray(betas, dtype=np.float64)
        assert b.shape == (self.nT,)
        self.h = self.lib.eao_create(self.L, self.nT, self.R, _ptr(b), int(seed), int(r0))
        if not self.h:
            raise ValueError("eao_create rejected the arguments")
        if check:
            self.lib.eao_set_check(self.h, 1)

    def close(self):
        if getattr(self, "h", None):
            self.lib.eao_destroy(self.h)
            self.h = None

    __del__ = close

    def set_check(self, on=True):
        self.lib.eao_set_check(self.h, int(on))

    def check_failures(self) -> int:
        return int(self.lib.eao_check_failures(self.h))

    def set_couplings(self, J):
        J = np.ascontiguousarray(J, dtype=np.int8)
        assert J.shape == (self.R, 3, self.N)
        return self.lib.eao_set_couplings(self.h, _ptr(J))

    def set_spins(self, s):
        s = np.ascontiguousarray(s, dtype=np.int8)
        assert s.shape == (self.R, self.nT, self.N)
        return self.lib.eao_set_spins(self.h, _ptr(s))

    def tables(self):
        acc = np.zeros((self.nT, 7), dtype=np.uint64)
        swp = np.zeros((max(self.nT - 1, 1), 3 * self.N + 1), dtype=np.uint64)
        self.lib.eao_get_tables(self.h, _ptr(acc), _ptr(swp))
        return acc, swp[: self.nT - 1]

    def set_tables(self, acc, swp):
        acc = np.ascontiguousarray(acc, dtype=np.uint64)
        swp = np.ascontiguousarray(swp, dtype=np.uint64)
        assert acc.shape == (self.nT, 7) and swp.shape == (self.nT - 1, 3 * self.N + 1)
        self.lib.eao_set_tables(self.h, _ptr(acc), _ptr(swp))

    def set_state(self, spins_by_slot, tau, sweeps, swap_rounds):
        """Resume from a checkpoint: s[r][slot][site], tau[r][slot], the two counters."""
        s = np.ascontiguousarray(spins_by_slot, dtype=np.int8)
        t = np.ascontiguousarray(tau, dtype=np.int32)
        assert s.shape == (self.R, self.nT, self.N) and t.shape == (self.R, self.nT)
        rc = self.lib.eao_set_state(self.h, _ptr(s), _ptr(t), int(sweeps), int(swap_rounds))
        if rc != 0:
            raise ValueError(f"eao_set_state -> {rc}")

    def seed_couplings(self, p_plus):
        """+-J couplings with bond concentration p_plus = P(J = +1), from the Philox seed (R25)."""
        if self.lib.eao_seed_couplings(self.h, float(p_plus)) != 0:
            raise ValueError("p_plus must lie in [0, 1]")

    def set_draw_mode(self, mode):
        """0: one draw per (site, word, slot) (default); 1: one per (site, realization, slot) --
        the paper's own coding, bits of a word = temperature replicas (R24)."""
        if self.lib.eao_set_draw_mode(self.h, int(mode)) != 0:
            raise ValueError("draw mode must be 0 or 1")

    def draw_mode(self) -> int:
        return int(self.lib.eao_get_draw_mode(self.h))

    def set_swap_mode(self, mode):
        """0: an accepted swap exchanges temperature indices (default); 1: it exchanges the two
        lattices and their energies, temperatures stay with the slots (R26)."""
        if self.lib.eao_set_swap_mode(self.h, int(mode)) != 0:
            raise ValueError("swap mode must be 0 or 1")

    def swap_mode(self) -> int:
        return int(self.lib.eao_get_swap_mode(self.h))

    def set_field(self, h):
        """Constant external field h of Eq. 1 (integer); energies are recomputed."""
        rc = self.lib.eao_set_field(self.h, int(h))
        if rc != 0:
            raise ValueError(f"eao_set_field -> {rc}")

    def field(self) -> int:
        return int(self.lib.eao_get_field(self.h))

    def field_tables(self):
        """(accf [nT][7][2], swpf [nT-1][2 (3+|h|) N + 1]) for h != 0."""
        Mf = (3 + abs(self.field())) * self.N
        accf = np.zeros((self.nT, 7, 2), dtype=np.uint64)
        swpf = np.zeros((max(self.nT - 1, 1), 2 * Mf + 1), dtype=np.uint64)
        if self.lib.eao_get_field_tables(self.h, _ptr(accf), _ptr(swpf)) != 0:
            raise ValueError("no field tables at h = 0")
        return accf, swpf[: self.nT - 1]

    def sweep(self, n_sweeps, swap_interval):
        rc = self.lib.eao_sweep(self.h, int(n_sweeps), int(swap_interval))
        if rc != 0:
            raise ValueError(f"eao_sweep -> {rc}")

    def energy(self):
        E = np.zeros((self.R, self.nT), dtype=np.int32)
        self.lib.eao_energy(self.h, _ptr(E))
        return E

    def energy_by_slot(self):
        E = np.zeros((self.R, self.nT), dtype=np.int32)
        self.lib.eao_get_energy_by_slot(self.h, _ptr(E))
        return E

    def energy_from_scratch(self, r, k) -> int:
        return int(self.lib.eao_energy_from_scratch(self.h, int(r), int(k)))

    def n_sat(self, k, r, site) -> int:
        return int(self.lib.eao_n_sat(self.h, int(k), int(r), int(site)))

    def overlap(self, pairs):
        pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        Q = np.zeros((len(pairs), self.nT), dtype=np.int32)
        rc = self.lib.eao_overlap(self.h, _ptr(pairs), len(pairs), _ptr(Q))
        if rc != 0:
            raise ValueError("bad pair")
        return Q

    def spins(self):
        s = np.zeros((self.R, self.nT, self.N), dtype=np.int8)
        self.lib.eao_get_spins(self.h, _ptr(s))
        return s

    def spins_by_slot(self):
        s = np.zeros((self.R, self.nT, self.N), dtype=np.int8)
        self.lib.eao_get_spins_by_slot(self.h, _ptr(s))
        return s

    def couplings(self):
        J = np.zeros((self.R, 3, self.N), dtype=np.int8)
        self.lib.eao_get_couplings(self.h, _ptr(J))
        return J

    def perm(self):
        tau = np.zeros((self.R, self.nT), dtype=np.int32)
        sigma = np.zeros((self.R, self.nT), dtype=np.int32)
        self.lib.eao_get_perm(self.h, _ptr(tau), _ptr(sigma))
        return tau, sigma

    def counters(self):
        g, n = C.c_uint64(), C.c_uint64()
        st = (C.c_int64 * 4)()
        self.lib.eao_get_counters(self.h, C.byref(g), C.byref(n), st)
        return {"sweeps": g.value, "swap_rounds": n.value, "attempts": st[0], "accepted": st[1],
                "swap_attempts": st[2], "swap_accepted": st[3]}


    # ------------------------------------------------------------------ measurement
    def pair_couplings(self):
        """Two-copy set-up: realizations R/2.. get the couplings of 0..R/2-1 (the spins and
        the random draws of the two halves stay different because they sit in different
        words, R11).  The overlap between the copies r and r + R/2 is the
        spin-glass order parameter q whose Binder ratio the paper plots (Fig. 20)."""
        half = self.R // 2
        assert self.R % 64 == 0, "R/2 must be a multiple of 32 (copies in different words)"
        J = self.couplings()
        J[half:] = J[:half]
        return self.set_couplings(J)

    def realization_pairs(self, word_pairs):
        """Word pair (wa, wb) -> the 32 realization pairs (32 wa + b, 32 wb + b); wb = -1 is the
        all-up reference.  Entries that touch a padding bit (index >= R) are None."""
        out = []
        for wa, wb in np.asarray(word_pairs, dtype=np.int64).reshape(-1, 2):
            row = []
            for b in range(32):
                ra, rb = 32 * int(wa) + b, (32 * int(wb) + b if wb >= 0 else -1)
                row.append((ra, rb) if ra < self.R and rb < self.R else None)
            out.append(row)
        return out

    def measure(self, n_meas, sweeps_between, swap_interval, word_pairs, acc=None):
        """n_meas times: sweep(sweeps_between, swap_interval), then one measurement of the
        overlaps q of `word_pairs` and of the energies E, by temperature index.  Accumulates
        exact integer sums (Python ints): n, sum q, sum q^2, sum q^4 as [pair][bit][t] and
        sum E, sum E^2 as [r][t].  Returns (and, if given, continues) the accumulator dict."""
        rp = self.realization_pairs(word_pairs)
        P = len(rp)
        if acc is None:
            z = lambda *shape: np.zeros(shape, dtype=object) + 0
            acc = {"n": 0, "q1": z(P, 32, self.nT), "q2": z(P, 32, self.nT), "q4": z(P, 32, self.nT),
                   "e1": z(self.R, self.nT), "e2": z(self.R, self.nT), "corr": z(P, 32, self.nT, self.L)}
        flat = [(p, b, pr) for p in range(P) for b, pr in enumerate(rp[p]) if pr is not None]
        pairs = np.array([pr for _, _, pr in flat], dtype=np.int32).reshape(-1, 2)
        for _ in range(int(n_meas)):
            self.sweep(sweeps_between, swap_interval)
            Q = self.overlap(pairs) if len(flat) else np.zeros((0, self.nT), dtype=np.int32)
            E = self.energy()
            if len(flat):
                s = self.spins()                     # [r][t][site], by temperature index
                for p, b, (ra, rb) in flat:
                    for t in range(self.nT):
                        qf = s[ra, t].astype(np.int64) * (s[rb, t].astype(np.int64) if rb >= 0 else 1)
                        c = plane_correlation(qf, self.L)
                        for d in range(self.L):
                            acc["corr"][p, b, t, d] += int(c[d])
            for (p, b, _), qrow in zip(flat, Q):
                for t in range(self.nT):
                    q = int(qrow[t])
                    acc["q1"][p, b, t] += q
                    acc["q2"][p, b, t] += q * q
                    acc["q4"][p, b, t] += q * q * q * q
            for r in range(self.R):
                for t in range(self.nT):
                    e = int(E[r, t])
                    acc["e1"][r, t] += e
                    acc["e2"][r, t] += e * e
            acc["n"] += 1
            round_trip_update(acc.setdefault("label", np.zeros((self.R, self.nT), dtype=np.int8)),
                              acc.setdefault("trips", np.zeros(self.R, dtype=np.int64)), self.perm()[0])
        acc["valid"] = np.array([[pr is not None for pr in row] for row in rp], dtype=bool).reshape(P, 32)
        return acc


def plane_correlation(q_field, L):
    """C(d) = sum over the three axes mu and the planes p of S_mu(p) S_mu((p + d) mod L), where
    S_mu(p) = sum of the local overlaps q_i = s_i^a s_i^b over the plane (coordinate mu of i) = p.
    q_field[site], site = x + L (y + L z).  These plane sums are all the wave-vector dependent
    susceptibility along the axes needs (R23); sum_d C(d) = 3 q^2."""
    f = np.asarray(q_field, dtype=np.int64).reshape(L, L, L)         # [z][y][x]
    C = np.zeros(L, dtype=np.int64)
    for axes in ((0, 1), (0, 2), (1, 2)):                             # planes of fixed x, y, z
        S = f.sum(axis=axes)
        for d in range(L):
            C[d] += int((S * np.roll(S, -d)).sum())                   # roll(S, -d)[p] = S[(p + d) mod L]
    return C


def correlation_length(acc, L):
    """Second-moment correlation length by temperature index (the quantity of the paper's
    Fig. 19, which prints no formula; R23):
      chi(k) = [<|q~(k)|^2>] / N averaged over the three axes = sum_d cos(k d) [<C(d)>] / (3 N),
      xi = sqrt(chi(0) / chi(k_min) - 1) / (2 sin(k_min / 2)),  k_min = 2 pi / L.
    Exact integer sums, the cosines in double; NaN where chi(k_min) <= 1e-12 chi(0), where
    chi(0) < chi(k_min), or where nothing was measured."""
    import math
    valid = acc["valid"]
    nT = acc["corr"].shape[2]
    xi = np.full(nT, np.nan)
    if acc["n"] == 0 or not valid.any():
        return xi
    for t in range(nT):
        Cd = [sum(int(v) for v in acc["corr"][valid, t, d]) for d in range(L)]
        chi0 = float(sum(Cd))
        chik = sum(math.cos(2.0 * math.pi * d / L) * float(Cd[d]) for d in range(L))
        if chik > 1e-12 * chi0 and chi0 >= chik:     # chi(k_min) = 0 up to rounding: undefined
            xi[t] = math.sqrt(chi0 / chik - 1.0) / (2.0 * math.sin(math.pi / L))
    return xi


def round_trip_update(label, trips, tau):
    """Round trips of the replicas in temperature space (the diagnostic behind "the choice of
    temperatures is crucial"), observed at measurement times.  tau[r][k] = temperature
    index of the replica in slot k.  label[r][k]: 0 = has not touched an end yet, 1 = was last at
    temperature index 0, 2 = was last at index nT-1.  A replica that comes back to index 0 after
    having been at nT-1 completes one round trip of its realization (R22)."""
    R, nT = tau.shape
    for r in range(R):
        for k in range(nT):
            t = int(tau[r, k])
            if t == 0:
                if label[r, k] == 2:
                    trips[r] += 1
                label[r, k] = 1
            elif t == nT - 1:
                label[r, k] = 2


def binder_ratio(acc):
    """Binder ratio of the overlap by temperature index, g = (3 - [<q^4>] / [<q^2>]^2) / 2:
    <.> = time average of one realization pair, [.] = average over the valid pairs (disorder
    average).  The paper plots it (Fig. 20) without printing the formula; this is
    the standard definition of its reference [63] (R20).  Exact rational arithmetic,
    rounded to double once at the end.  NaN where [<q^2>] = 0."""
    n = acc["n"]
    valid = acc["valid"]
    M = int(valid.sum())
    nT = acc["q2"].shape[2]
    g = np.full(nT, np.nan)
    for t in range(nT):
        s2 = sum(int(v) for v in acc["q2"][valid, t])
        s4 = sum(int(v) for v in acc["q4"][valid, t])
        if n == 0 or M == 0 or s2 == 0:
            continue
        q2 = Fraction(s2, n * M)
        q4 = Fraction(s4, n * M)
        g[t] = float((3 - q4 / (q2 * q2)) / 2)
    return g
