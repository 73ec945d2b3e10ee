"""ctypes binding with the same names as include/ea.h."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libea_b200.so"
_lib = None

EA_KERNEL_AUTO, EA_KERNEL_GENERIC, EA_KERNEL_RESIDENT, EA_KERNEL_TILED, EA_KERNEL_STREAM, EA_KERNEL_REPLICA = 0, 1, 2, 3, 4, 5
EA_KERNEL_GENERIC_STEPWISE = 6
EA_LAYOUT_REALIZATION_BITS, EA_LAYOUT_REPLICA_BITS = 0, 1
EA_SWAP_PERMUTE, EA_SWAP_MOVE = 0, 1

_SYMBOLS = [
    "ea_create", "ea_workspace_bytes", "ea_create_ex", "ea_destroy", "ea_set_couplings",
    "ea_set_spins", "ea_set_tables", "ea_get_tables", "ea_sweep", "ea_synchronize", "ea_energy",
    "ea_overlap", "ea_get_spins", "ea_get_state", "ea_set_kernel", "ea_get_kernel",
    "ea_launch_count", "ea_last_error", "ea_measure_int_peak",
    "ea_get_couplings", "ea_pair_couplings", "ea_measure_begin", "ea_measure", "ea_get_moments",
    "ea_get_binder", "ea_set_field", "ea_get_field", "ea_get_field_tables",
    "ea_get_round_trips", "ea_get_correlation", "ea_get_correlation_length", "ea_set_state",
    "ea_set_layout", "ea_get_layout", "ea_seed_couplings", "ea_set_swap_mode", "ea_get_swap_mode",
    "ea_overlap_static",
]


class EAError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"ea error {code}: {msg}")
        self.code = code


def library_path() -> Path:
    return _LIB_PATH


def exported_symbols():
    return list(_SYMBOLS)


def lib():
    """Load libea_b200.so; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError(f"{_LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; "
                          f"g.build()'` (nvcc, sm_100a); there is no CPU fallback")
    l = C.CDLL(str(_LIB_PATH))
    vp, i32, i64, u64, sz = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_size_t
    l.ea_create.restype = vp
    l.ea_create.argtypes = [i32, i32, i32, vp, u64]
    l.ea_workspace_bytes.restype = sz
    l.ea_workspace_bytes.argtypes = [i32, i32, i32]
    l.ea_create_ex.restype = vp
    l.ea_create_ex.argtypes = [i32, i32, i32, vp, u64, vp, sz, vp, i32]
    l.ea_destroy.restype = None
    l.ea_destroy.argtypes = [vp]
    for name, args in (("ea_set_couplings", [vp, vp]), ("ea_set_spins", [vp, vp]),
                       ("ea_set_tables", [vp, vp, vp]), ("ea_get_tables", [vp, vp, vp]),
                       ("ea_sweep", [vp, i64, i32]), ("ea_synchronize", [vp]),
                       ("ea_energy", [vp, vp]), ("ea_overlap", [vp, vp, i32, vp]),
                       ("ea_overlap_static", [vp, vp, i32, vp]),
                       ("ea_get_spins", [vp, vp]), ("ea_get_state", [vp, vp, vp, vp, vp, vp]),
                       ("ea_set_kernel", [vp, i32]), ("ea_get_kernel", [vp]),
                       ("ea_get_couplings", [vp, vp]), ("ea_pair_couplings", [vp]),
                       ("ea_measure_begin", [vp, vp, i32]), ("ea_measure", [vp, i64, i64, i32]),
                       ("ea_get_moments", [vp, vp, vp, vp, vp, vp, vp]), ("ea_get_binder", [vp, vp]),
                       ("ea_set_field", [vp, i32]), ("ea_get_field", [vp]),
                       ("ea_get_field_tables", [vp, vp, vp]), ("ea_get_round_trips", [vp, vp]),
                       ("ea_get_correlation", [vp, vp]), ("ea_get_correlation_length", [vp, vp]),
                       ("ea_set_layout", [vp, i32]), ("ea_get_layout", [vp]),
                       ("ea_set_swap_mode", [vp, i32]), ("ea_get_swap_mode", [vp])):
        f = getattr(l, name)
        f.restype = i32
        f.argtypes = args
    l.ea_seed_couplings.restype = i32
    l.ea_seed_couplings.argtypes = [vp, C.c_double]
    l.ea_set_state.restype = i32
    l.ea_set_state.argtypes = [vp, vp, vp, u64, u64]
    l.ea_launch_count.restype = i64
    l.ea_launch_count.argtypes = [vp]
    l.ea_last_error.restype = C.c_char_p
    l.ea_last_error.argtypes = [vp]
    l.ea_measure_int_peak.restype = i32
    l.ea_measure_int_peak.argtypes = [vp, vp]
    _lib = l
    return l


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class EA:
    """One simulation handle.  Methods mirror the C calls (ea_<name>)."""

    def __init__(self, L, n_temps, n_realizations, betas, seed, first_realization=0,
                 torch_workspace=True, kernel=EA_KERNEL_AUTO):
        self._l = lib()
        self.L, self.nT, self.R = int(L), int(n_temps), int(n_realizations)
        self.N, self.W = self.L ** 3, (self.R + 31) // 32
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.shape != (self.nT,):
            raise ValueError("betas must have n_temps entries")
        self._ws = None
        ws_ptr, ws_bytes, stream = None, 0, None
        if torch_workspace:
            import torch
            if not torch.cuda.is_available():
                raise EAError(-3, "no CUDA device (there is no CPU fallback)")
            ws_bytes = int(self._l.ea_workspace_bytes(self.L, self.nT, self.R))
            if ws_bytes:
                self._ws = torch.empty(ws_bytes + 256, dtype=torch.uint8, device="cuda")
                ws_ptr = (self._ws.data_ptr() + 255) & ~255
                stream = torch.cuda.current_stream().cuda_stream
        self.h = self._l.ea_create_ex(self.L, self.nT, self.R, _p(b), int(seed), ws_ptr, ws_bytes,
                                      stream, int(first_realization))
        if not self.h:
            raise EAError(-1, self._l.ea_last_error(None).decode())
        if kernel != EA_KERNEL_AUTO:
            self.set_kernel(kernel)

    def _chk(self, rc):
        if rc != 0:
            raise EAError(rc, self._l.ea_last_error(self.h).decode())

    def destroy(self):
        if getattr(self, "h", None):
            self._l.ea_destroy(self.h)
            self.h = None
            self._ws = None

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def set_couplings(self, J):
        J = np.ascontiguousarray(J, dtype=np.int8)
        assert J.shape == (self.R, 3, self.N)
        self._chk(self._l.ea_set_couplings(self.h, _p(J)))

    def set_spins(self, s):
        s = np.ascontiguousarray(s, dtype=np.int8)
        assert s.shape == (self.R, self.nT, self.N)
        self._chk(self._l.ea_set_spins(self.h, _p(s)))

    def set_tables(self, acc, swp):
        acc = np.ascontiguousarray(acc, dtype=np.uint64)
        swp = np.ascontiguousarray(swp, dtype=np.uint64)
        assert acc.shape == (self.nT, 7) and swp.shape == (max(self.nT - 1, 0), 3 * self.N + 1)
        self._chk(self._l.ea_set_tables(self.h, _p(acc), _p(swp)))

    def get_tables(self):
        acc = np.zeros((self.nT, 7), dtype=np.uint64)
        swp = np.zeros((max(self.nT - 1, 0), 3 * self.N + 1), dtype=np.uint64)
        self._chk(self._l.ea_get_tables(self.h, _p(acc), _p(swp)))
        return acc, swp

    def sweep(self, n_sweeps, swap_interval):
        self._chk(self._l.ea_sweep(self.h, int(n_sweeps), int(swap_interval)))

    def synchronize(self):
        self._chk(self._l.ea_synchronize(self.h))

    def energy(self):
        E = np.zeros((self.R, self.nT), dtype=np.int32)
        self._chk(self._l.ea_energy(self.h, _p(E)))
        return E

    def overlap(self, pairs):
        pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        Q = np.zeros((len(pairs), self.nT), dtype=np.int32)
        self._chk(self._l.ea_overlap(self.h, _p(pairs), len(pairs), _p(Q)))
        return Q

    def overlap_static(self, pairs):
        """ea_overlap through the library's fixed device array: no allocation in the call (ea.h)."""
        pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        Q = np.zeros((len(pairs), self.nT), dtype=np.int32)
        self._chk(self._l.ea_overlap_static(self.h, _p(pairs), len(pairs), _p(Q)))
        return Q

    def get_spins(self):
        s = np.zeros((self.R, self.nT, self.N), dtype=np.int8)
        self._chk(self._l.ea_get_spins(self.h, _p(s)))
        return s

    def get_state(self, spins=True):
        words = np.zeros((self.nT, self.W, 2, self.N // 2), dtype=np.uint32) if spins else None
        tau = np.zeros((self.R, self.nT), dtype=np.uint8)
        E = np.zeros((self.R, self.nT), dtype=np.int32)
        g, n = C.c_uint64(), C.c_uint64()
        self._chk(self._l.ea_get_state(self.h, _p(words), _p(tau), _p(E), C.byref(g), C.byref(n)))
        return {"spin_words": words, "temp_of_slot": tau, "energy_by_slot": E,
                "sweeps": g.value, "swap_rounds": n.value}

    def get_couplings(self):
        J = np.zeros((self.R, 3, self.N), dtype=np.int8)
        self._chk(self._l.ea_get_couplings(self.h, _p(J)))
        return J

    def pair_couplings(self):
        self._chk(self._l.ea_pair_couplings(self.h))

    def measure_begin(self, word_pairs):
        wp = np.ascontiguousarray(word_pairs, dtype=np.int32).reshape(-1, 2)
        self._n_wp = len(wp)
        self._chk(self._l.ea_measure_begin(self.h, _p(wp), len(wp)))

    def measure(self, n_meas, sweeps_between, swap_interval):
        self._chk(self._l.ea_measure(self.h, int(n_meas), int(sweeps_between), int(swap_interval)))

    def get_moments(self):
        """The integer accumulators as they are stored: q4 is [P][32][n_temps][2] = (low, high)."""
        P = self._n_wp
        n = C.c_uint64()
        q1 = np.zeros((P, 32, self.nT), dtype=np.int64)
        q2 = np.zeros((P, 32, self.nT), dtype=np.uint64)
        q4 = np.zeros((P, 32, self.nT, 2), dtype=np.uint64)
        e1 = np.zeros((self.R, self.nT), dtype=np.int64)
        e2 = np.zeros((self.R, self.nT), dtype=np.uint64)
        self._chk(self._l.ea_get_moments(self.h, C.byref(n), _p(q1), _p(q2), _p(q4), _p(e1), _p(e2)))
        return {"n": n.value, "q1": q1, "q2": q2, "q4": q4, "e1": e1, "e2": e2}

    def get_correlation(self):
        C_ = np.zeros((self._n_wp, 32, self.nT, self.L), dtype=np.int64)
        self._chk(self._l.ea_get_correlation(self.h, _p(C_)))
        return C_

    def get_correlation_length(self):
        xi = np.zeros(self.nT, dtype=np.float64)
        self._chk(self._l.ea_get_correlation_length(self.h, _p(xi)))
        return xi

    def get_round_trips(self):
        trips = np.zeros(self.R, dtype=np.uint64)
        self._chk(self._l.ea_get_round_trips(self.h, _p(trips)))
        return trips

    def get_binder(self):
        g = np.zeros(self.nT, dtype=np.float64)
        self._chk(self._l.ea_get_binder(self.h, _p(g)))
        return g

    def set_field(self, field):
        self._chk(self._l.ea_set_field(self.h, int(field)))

    def get_field(self):
        return int(self._l.ea_get_field(self.h))

    def get_field_tables(self):
        Mf = (3 + abs(self.get_field())) * self.N
        accf = np.zeros((self.nT, 7, 2), dtype=np.uint64)
        swpf = np.zeros((max(self.nT - 1, 0), 2 * Mf + 1), dtype=np.uint64)
        self._chk(self._l.ea_get_field_tables(self.h, _p(accf), _p(swpf)))
        return accf, swpf

    def set_state(self, state):
        """Resume from the dict get_state() returned (on a handle with the same shape, betas, seed)."""
        words = np.ascontiguousarray(state["spin_words"], dtype=np.uint32)
        tau = np.ascontiguousarray(state["temp_of_slot"], dtype=np.uint8)
        assert words.shape == (self.nT, self.W, 2, self.N // 2) and tau.shape == (self.R, self.nT)
        self._chk(self._l.ea_set_state(self.h, _p(words), _p(tau), int(state["sweeps"]), int(state["swap_rounds"])))

    def set_kernel(self, kernel):
        self._chk(self._l.ea_set_kernel(self.h, int(kernel)))

    def get_kernel(self):
        return int(self._l.ea_get_kernel(self.h))

    def seed_couplings(self, p_plus):
        self._chk(self._l.ea_seed_couplings(self.h, float(p_plus)))

    def set_layout(self, layout):
        self._chk(self._l.ea_set_layout(self.h, int(layout)))

    def get_layout(self):
        return int(self._l.ea_get_layout(self.h))

    def set_swap_mode(self, mode):
        self._chk(self._l.ea_set_swap_mode(self.h, int(mode)))

    def get_swap_mode(self):
        return int(self._l.ea_get_swap_mode(self.h))

    def launch_count(self):
        return int(self._l.ea_launch_count(self.h))


def measure_int_peak(stream=None):
    """ea_measure_int_peak: dict of measured integer issue rates (lane-ops/s)."""
    out = (C.c_double * 4)()
    rc = lib().ea_measure_int_peak(stream, out)
    if rc != 0:
        raise EAError(rc, "ea_measure_int_peak failed")
    return {"lop3": out[0], "imad": out[1], "mix": out[2], "sms": int(out[3])}
