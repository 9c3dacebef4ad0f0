"""ctypes binding of libsg_b200 (include/sg.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of paper_1403_4560_b200/csrc; PyTorch supplies the
device workspace tensor and the CUDA stream.  There is no CPU fallback: if the library has not been
built (python -m paper_1403_4560_b200.build or __graft_entry__.build()) the import raises.
"""
import ctypes as C
import os

import numpy as np

PMJ, GAUSS, PMJ_TPACK = 0, 1, 2
NK, REC, NMOM = 12, 25, 66
OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ESTATE = 0, -1, -2, -3, -4, -5
PATH_AUTO, PATH_GENERIC = 0, 1
NOALLOC_MAX_SYSTEMS = 65536
ACCEPT_GENERAL, ACCEPT_CARRY_CHAIN, ACCEPT_BINARY_SEARCH = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libsg_b200.so")

EXPORTS = {
    # name: (restype, argtypes)
    "sg_workspace_bytes": (C.c_size_t, [C.c_int] * 5),
    "sg_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_int,
                            C.c_int, C.c_uint64, C.c_void_p, C.c_size_t, C.c_void_p]),
    "sg_set_first_sample": (C.c_int, [C.c_void_p, C.c_int64]),
    "sg_reset": (C.c_int, [C.c_void_p]),
    "sg_sweep": (C.c_int, [C.c_void_p, C.c_int]),
    "sg_pt_exchange": (C.c_int, [C.c_void_p]),
    "sg_measure": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_run": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "sg_synchronize": (C.c_int, [C.c_void_p]),
    "sg_destroy": (C.c_int, [C.c_void_p]),
    "sg_get_spins": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_set_spins": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_get_couplings": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_get_spins_range": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "sg_set_spins_range": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "sg_get_couplings_range": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "sg_get_energies": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "sg_get_thresholds": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_get_moments": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "sg_get_counters": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "sg_get_launch_count": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_set_counters": (C.c_int, [C.c_void_p, C.c_uint64, C.c_uint64]),
    "sg_set_moments": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64]),
    "sg_last_error": (C.c_char_p, [C.c_void_p]),
    "sg_debug_fail_launch": (C.c_int, [C.c_void_p, C.c_int]),
    "sg_get_accept_variant": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_set_kernel_path": (C.c_int, [C.c_void_p, C.c_int]),
    "sg_get_state_hash": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_get_state_hash_noalloc": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_get_energies_cached": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "sg_get_pt_stats": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "sg_enable_pq": (C.c_int, [C.c_void_p, C.c_int]),
    "sg_get_pq": (C.c_int, [C.c_void_p, C.c_void_p]),
    "sg_enable_log_binning": (C.c_int, [C.c_void_p, C.c_int]),
    "sg_get_window_moments": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]),
}

if not os.path.exists(LIB_PATH):
    raise ImportError("libsg_b200.so is not built (%s); run `python -m paper_1403_4560_b200.build` — "
                      "there is no CPU fallback" % LIB_PATH)
_lib = C.CDLL(LIB_PATH)
for _name, (_res, _args) in EXPORTS.items():
    _fn = getattr(_lib, _name)
    _fn.restype = _res
    _fn.argtypes = _args


class SgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libsg_b200 error %d: %s" % (code, msg))
        self.code = code


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def sg_workspace_bytes(L, n_samples, n_replicas, n_temps, coupling_kind):
    return int(_lib.sg_workspace_bytes(L, n_samples, n_replicas, n_temps, coupling_kind))


class Simulation:
    """One sg_ctx.  `workspace`: a torch CUDA uint8 tensor (allocated here with torch if None);
    `stream`: a torch.cuda.Stream (current stream if None)."""

    def __init__(self, L, h, n_samples, n_replicas, temps, coupling_kind=PMJ, seed=1, workspace=None,
                 stream=None, device=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libsg_b200 needs a CUDA device; there is no CPU fallback")
        self.L, self.N = int(L), int(L) ** 3
        self.h = float(h)
        self.n_samples, self.R = int(n_samples), int(n_replicas)
        self.temps = np.ascontiguousarray(temps, dtype=np.float64)
        self.NT = int(self.temps.size)
        self.kind = int(coupling_kind)
        self.n_pairs = self.R * (self.R - 1) // 2
        self.pq_bins, self.n_windows = 1, 0
        self._h = C.c_void_p()
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        need = sg_workspace_bytes(self.L, self.n_samples, self.R, self.NT, self.kind)
        if need == 0:
            raise SgError(EINVAL, "invalid parameters (sg_workspace_bytes returned 0)")
        with torch.cuda.device(self.device):
            if workspace is None:
                workspace = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            self.workspace = workspace
            ptr = workspace.data_ptr()
            aligned = (ptr + 255) // 256 * 256
            avail = workspace.numel() - (aligned - ptr)
            self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
            rc = _lib.sg_create(C.byref(self._h), self.L, self.h, self.n_samples, self.R, _p(self.temps), self.NT,
                                self.kind, int(seed), C.c_void_p(aligned), avail, C.c_void_p(self.stream.cuda_stream))
        if rc != OK:
            self._h = C.c_void_p()
            raise SgError(rc, (_lib.sg_last_error(None) or b"").decode())

    # -- helpers
    def _check(self, rc):
        if rc != OK:
            raise SgError(rc, (_lib.sg_last_error(self._h) or b"").decode())

    def close(self):
        if self._h:
            _lib.sg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the path
    def sg_set_first_sample(self, first_sample):
        self._check(_lib.sg_set_first_sample(self._h, int(first_sample)))

    def sg_reset(self):
        self._check(_lib.sg_reset(self._h))

    def sg_sweep(self, n=1):
        self._check(_lib.sg_sweep(self._h, int(n)))

    def sg_pt_exchange(self):
        self._check(_lib.sg_pt_exchange(self._h))

    def sg_measure(self, want=True):
        if not want:
            self._check(_lib.sg_measure(self._h, None))
            return None
        out = np.empty((self.n_samples, self.NT, self.n_pairs, REC), dtype=np.float64)
        self._check(_lib.sg_measure(self._h, _p(out)))
        return out

    def sg_run(self, n_sweeps, pt_every=0, meas_every=0):
        self._check(_lib.sg_run(self._h, int(n_sweeps), int(pt_every), int(meas_every)))

    def sg_synchronize(self):
        self._check(_lib.sg_synchronize(self._h))

    # -- introspection
    def sg_get_spins(self, s0=None, ns=None):
        if s0 is None:
            s0, ns = 0, self.n_samples
        out = np.empty((ns, self.R, self.NT, self.N), dtype=np.int8)
        self._check(_lib.sg_get_spins_range(self._h, int(s0), int(ns), _p(out)))
        return out

    def sg_set_spins(self, spins, s0=0):
        spins = np.ascontiguousarray(spins, dtype=np.int8)
        ns = spins.size // (self.R * self.NT * self.N)
        self._check(_lib.sg_set_spins_range(self._h, int(s0), int(ns), _p(spins)))

    def sg_get_couplings(self, s0=None, ns=None):
        if s0 is None:
            s0, ns = 0, self.n_samples
        out = np.empty((ns, 3, self.N), dtype=np.float32)
        self._check(_lib.sg_get_couplings_range(self._h, int(s0), int(ns), _p(out)))
        return out

    def sg_get_energies(self):
        U = np.empty((self.n_samples, self.R, self.NT), dtype=np.int64)
        M = np.empty((self.n_samples, self.R, self.NT), dtype=np.int32)
        self._check(_lib.sg_get_energies(self._h, _p(U), _p(M)))
        return U, M

    def sg_get_energies_cached(self):
        """The kernels' own (U, M) (raises SgError(ESTATE) if they are not up to date with the state)."""
        U = np.empty((self.n_samples, self.R, self.NT), dtype=np.int64)
        M = np.empty((self.n_samples, self.R, self.NT), dtype=np.int32)
        self._check(_lib.sg_get_energies_cached(self._h, _p(U), _p(M)))
        return U, M

    def sg_get_energies_cached_into(self, U, M):
        """Fill caller-owned (e.g. pinned) int64 / int32 host arrays of shape [n_samples][R][NT]."""
        self._check(_lib.sg_get_energies_cached(self._h, C.c_void_p(U.ctypes.data), C.c_void_p(M.ctypes.data)))

    def sg_set_kernel_path(self, path):
        self._check(_lib.sg_set_kernel_path(self._h, int(path)))

    def sg_get_state_hash(self):
        nw = (self.n_samples + 31) // 32 if self.kind != GAUSS else self.n_samples
        out = np.empty((nw, self.R, self.NT), dtype=np.uint64)
        self._check(_lib.sg_get_state_hash(self._h, _p(out)))
        return out

    def sg_get_state_hash_noalloc(self):
        """sg_get_state_hash for callers that must not allocate device memory (include/sg.h): same values, staged in the
        library's fixed 512 KiB device array; raises SgError(EINVAL) beyond NOALLOC_MAX_SYSTEMS systems."""
        nw = (self.n_samples + 31) // 32 if self.kind != GAUSS else self.n_samples
        out = np.empty((nw, self.R, self.NT), dtype=np.uint64)
        self._check(_lib.sg_get_state_hash_noalloc(self._h, _p(out)))
        return out

    def sg_get_pt_stats(self):
        """(proposed, accepted) per adjacent slot pair, summed over samples and replicas."""
        prop = np.zeros(max(self.NT - 1, 0), dtype=np.uint64)
        acc = np.zeros(max(self.NT - 1, 0), dtype=np.uint64)
        self._check(_lib.sg_get_pt_stats(self._h, _p(prop), _p(acc)))
        return prop, acc

    def sg_enable_pq(self, n_bins=None):
        n_bins = self.N + 1 if n_bins is None else int(n_bins)
        self._check(_lib.sg_enable_pq(self._h, n_bins))
        self.pq_bins = n_bins                   # only once the library has accepted it

    def sg_get_pq(self):
        out = np.empty((self.n_samples, self.NT, self.pq_bins), dtype=np.uint32)
        self._check(_lib.sg_get_pq(self._h, _p(out)))
        return out

    def sg_enable_log_binning(self, n_windows):
        self._check(_lib.sg_enable_log_binning(self._h, int(n_windows)))
        self.n_windows = int(n_windows)         # only once the library has accepted it

    def sg_get_window_moments(self, k):
        out = np.empty((self.n_samples, self.NT, NMOM), dtype=np.float64)
        n = C.c_int64()
        self._check(_lib.sg_get_window_moments(self._h, int(k), _p(out), C.byref(n)))
        return out, n.value

    def sg_get_thresholds(self):
        out = np.empty((self.NT, 7, 2), dtype=np.uint64)
        self._check(_lib.sg_get_thresholds(self._h, _p(out)))
        return out

    def sg_get_moments(self, want=True):
        n = C.c_int64()
        out = None
        if want:
            out = np.empty((self.n_samples, self.NT, NMOM), dtype=np.float64)
            self._check(_lib.sg_get_moments(self._h, _p(out), C.byref(n)))
        else:
            self._check(_lib.sg_get_moments(self._h, None, C.byref(n)))
        return out, n.value

    def sg_get_moments_into(self, out):
        """Fill a caller-owned (e.g. pinned) host buffer; returns n_meas."""
        n = C.c_int64()
        self._check(_lib.sg_get_moments(self._h, C.c_void_p(out.ctypes.data if hasattr(out, "ctypes") else out.data_ptr()),
                                        C.byref(n)))
        return n.value

    def sg_get_accept_variant(self):
        v = C.c_int()
        self._check(_lib.sg_get_accept_variant(self._h, C.byref(v)))
        return v.value

    def sg_debug_fail_launch(self, countdown):
        self._check(_lib.sg_debug_fail_launch(self._h, int(countdown)))

    def sg_get_counters(self):
        a, b = C.c_uint64(), C.c_uint64()
        self._check(_lib.sg_get_counters(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def sg_set_counters(self, sweeps_done, exchanges_done):
        self._check(_lib.sg_set_counters(self._h, int(sweeps_done), int(exchanges_done)))

    def sg_set_moments(self, moments, n_meas):
        m = np.ascontiguousarray(moments, dtype=np.float64)
        if m.shape != (self.n_samples, self.NT, NMOM):
            raise ValueError("sg_set_moments: expected shape %r" % ((self.n_samples, self.NT, NMOM),))
        self._check(_lib.sg_set_moments(self._h, _p(m), int(n_meas)))

    def sg_get_launch_count(self):
        a = C.c_uint64()
        self._check(_lib.sg_get_launch_count(self._h, C.byref(a)))
        return a.value
