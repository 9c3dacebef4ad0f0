"""ctypes access to the CPU oracle (oracle/ea_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing under paper_1403_4560_b200/ imports it, and it
imports nothing from there.  Argument marshalling only; all arithmetic is in the C file.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

PMJ, GAUSS = 0, 1
NK, REC, NMOM = 12, 25, 66

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i32, u64, dbl = C.c_void_p, C.c_int, C.c_uint64, C.c_double
        L.ea_create.restype = vp
        L.ea_create.argtypes = [i32, i32, i32, dbl, i32, i32, vp, i32, u64, i32]
        for name, args, res in [
            ("ea_destroy", [vp], None),
            ("ea_sweep", [vp, i32], None),
            ("ea_pt_exchange", [vp], None),
            ("ea_measure", [vp, vp], None),
            ("ea_run", [vp, i32, i32, i32], None),
            ("ea_run_series", [vp, i32, i32, vp, vp, vp], None),
            ("ea_n_pairs", [vp], i32),
            ("ea_get_spins", [vp, vp], None),
            ("ea_set_spins", [vp, vp], None),
            ("ea_get_couplings", [vp, vp], None),
            ("ea_set_couplings_pm", [vp, vp], None),
            ("ea_get_energies", [vp, vp, vp], None),
            ("ea_recompute_energies", [vp, vp, vp], None),
            ("ea_hamiltonian", [vp, i32, i32], dbl),
            ("ea_energy_pt", [vp, i32, i32], dbl),
            ("ea_get_thresholds", [vp, vp], None),
            ("ea_get_moments", [vp, vp, vp], None),
            ("ea_get_counters", [vp, vp, vp], None),
            ("ea_get_pt_stats", [vp, vp, vp], None),
            ("ea_enable_pq", [vp, i32], i32),
            ("ea_get_pq", [vp, vp], None),
            ("ea_enable_log_binning", [vp, i32], i32),
            ("ea_get_window_moments", [vp, i32, vp, vp], None),
            ("ea_philox4x32_10", [vp, vp, vp], None),
            ("ea_dlog", [dbl], dbl),
            ("ea_dsincos2pi", [dbl, vp, vp], None),
            ("ea_dexp64", [dbl], u64),
            ("ea_dexp32", [C.c_float], u64),
        ]:
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = res
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().ea_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def dlog(u):
    return lib().ea_dlog(float(u))


def dsincos2pi(u):
    c = C.c_double()
    s = C.c_double()
    lib().ea_dsincos2pi(float(u), C.byref(c), C.byref(s))
    return c.value, s.value


def dexp64(y):
    return int(lib().ea_dexp64(float(y)))


def dexp32(y):
    return int(lib().ea_dexp32(float(np.float32(y))))


class Oracle:
    """One disorder sample with all its replicas x temperature slots."""

    def __init__(self, L, h, n_replicas, temps, kind=PMJ, seed=1, sample=0):
        if isinstance(L, int):
            L = (L, L, L)
        self.Lx, self.Ly, self.Lz = (int(v) for v in L)
        self.N = self.Lx * self.Ly * self.Lz
        self.R = int(n_replicas)
        self.temps = np.ascontiguousarray(temps, dtype=np.float64)
        self.NT = int(self.temps.size)
        self.kind = int(kind)
        self.sample = int(sample)
        self.h = float(h)
        self._h = lib().ea_create(self.Lx, self.Ly, self.Lz, self.h, self.R, self.NT, _p(self.temps),
                                  self.kind, int(seed), self.sample)
        if not self._h:
            raise ValueError("ea_create rejected the arguments")
        self.n_pairs = lib().ea_n_pairs(self._h)

    def close(self):
        if self._h:
            lib().ea_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sweep(self, n=1):
        lib().ea_sweep(self._h, int(n))

    def pt_exchange(self):
        lib().ea_pt_exchange(self._h)

    def measure(self, want=True):
        if not want:
            lib().ea_measure(self._h, None)
            return None
        out = np.zeros((self.NT, self.n_pairs, REC), dtype=np.float64)
        lib().ea_measure(self._h, _p(out))
        return out

    def run(self, n_sweeps, pt_every=0, meas_every=0):
        lib().ea_run(self._h, int(n_sweeps), int(pt_every), int(meas_every))

    def run_series(self, n_sweeps, pt_every=0):
        U = np.zeros((n_sweeps, self.R, self.NT), dtype=np.int64)
        M = np.zeros((n_sweeps, self.R, self.NT), dtype=np.int32)
        Q = np.zeros((n_sweeps, self.NT), dtype=np.int32)
        lib().ea_run_series(self._h, int(n_sweeps), int(pt_every), _p(U), _p(M), _p(Q))
        return U, M, Q

    def spins(self):
        out = np.zeros((self.R, self.NT, self.N), dtype=np.int8)
        lib().ea_get_spins(self._h, _p(out))
        return out

    def set_spins(self, s):
        s = np.ascontiguousarray(s, dtype=np.int8).reshape(self.R, self.NT, self.N)
        lib().ea_set_spins(self._h, _p(s))

    def couplings(self):
        out = np.zeros((3, self.N), dtype=np.float32)
        lib().ea_get_couplings(self._h, _p(out))
        return out

    def set_couplings_pm(self, J):
        J = np.ascontiguousarray(J, dtype=np.int8).reshape(3, self.N)
        lib().ea_set_couplings_pm(self._h, _p(J))

    def energies(self):
        U = np.zeros((self.R, self.NT), dtype=np.int64)
        M = np.zeros((self.R, self.NT), dtype=np.int32)
        lib().ea_get_energies(self._h, _p(U), _p(M))
        return U, M

    def recomputed_energies(self):
        U = np.zeros((self.R, self.NT), dtype=np.int64)
        M = np.zeros((self.R, self.NT), dtype=np.int32)
        lib().ea_recompute_energies(self._h, _p(U), _p(M))
        return U, M

    def hamiltonian(self, a, t):
        return lib().ea_hamiltonian(self._h, int(a), int(t))

    def energy_pt(self, a, t):
        return lib().ea_energy_pt(self._h, int(a), int(t))

    def thresholds(self):
        out = np.zeros((self.NT, 7, 2), dtype=np.uint64)
        lib().ea_get_thresholds(self._h, _p(out))
        return out

    def moments(self):
        out = np.zeros((self.NT, NMOM), dtype=np.float64)
        n = C.c_int64()
        lib().ea_get_moments(self._h, _p(out), C.byref(n))
        return out, n.value

    def counters(self):
        a, b = C.c_uint64(), C.c_uint64()
        lib().ea_get_counters(self._h, C.byref(a), C.byref(b))
        return a.value, b.value

    def enable_pq(self, n_bins=None):
        self.pq_bins = self.N + 1 if n_bins is None else int(n_bins)
        if lib().ea_enable_pq(self._h, self.pq_bins) != 0:
            raise ValueError("ea_enable_pq rejected n_bins")

    def pq(self):
        out = np.zeros((self.NT, self.pq_bins), dtype=np.uint64)
        lib().ea_get_pq(self._h, _p(out))
        return out

    def enable_log_binning(self, n_windows):
        self.n_windows = int(n_windows)
        if lib().ea_enable_log_binning(self._h, self.n_windows) != 0:
            raise ValueError("ea_enable_log_binning rejected n_windows")

    def window_moments(self, k):
        out = np.zeros((self.NT, NMOM), dtype=np.float64)
        n = C.c_int64()
        lib().ea_get_window_moments(self._h, int(k), _p(out), C.byref(n))
        return out, n.value

    def pt_stats(self):
        a, b = C.c_uint64(), C.c_uint64()
        lib().ea_get_pt_stats(self._h, C.byref(a), C.byref(b))
        return a.value, b.value
