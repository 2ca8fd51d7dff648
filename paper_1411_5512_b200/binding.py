"""ctypes binding of libea_b200.so -- argument marshalling only; every step runs in the CUDA kernels.

Function names are those of include/ea.h.  PyTorch is used for device memory (the workspace tensor handed to
`ea_create_ex`) and streams, nothing else.  There is NO fallback: if the shared library is missing or has no
CUDA device to run on, calls raise `EAError` / `OSError`.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libea_b200.so")

EA_OK, EA_ERR_INVALID, EA_ERR_CUDA, EA_ERR_NOMEM, EA_ERR_STATE = range(5)
EA_KERNEL_AUTO, EA_KERNEL_SCALAR, EA_KERNEL_VEC2, EA_KERNEL_ROWS, EA_KERNEL_RESIDENT, EA_KERNEL_FOLD, EA_KERNEL_ROWS_PERSISTENT, \
    EA_KERNEL_SMALL = range(8)
KERNEL_NAMES = {"auto": 0, "scalar": 1, "vec2": 2, "rows": 3, "resident": 4, "rows_persistent": 6, "small": 7}
LANES = 64
C4_STATIC_MAX_VECTORS = 1024  # EA_C4_STATIC_MAX_VECTORS (include/ea.h)


class ea_params(C.Structure):
    _fields_ = [("L", C.c_int32), ("n_samples", C.c_int32), ("n_replicas", C.c_int32), ("n_slots", C.c_int32),
                ("p", C.c_double), ("T", C.c_double), ("seed", C.c_uint64), ("device", C.c_int32),
                ("kernel", C.c_int32), ("stream", C.c_void_p), ("d_workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t)]


class EAError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("ea status %d: %s" % (status, msg))
        self.status = status


# name -> (restype, argtypes); the -m "not gpu" suite checks that every symbol of include/ea.h is here and exported
_vp, _i, _u64, _dbl = C.c_void_p, C.c_int, C.c_uint64, C.c_double
SIGNATURES = {
    "ea_workspace_bytes": (C.c_size_t, [_i, _i, _i]),
    "ea_create": (_i, [_i, _dbl, _dbl, _i, _u64, C.POINTER(_vp)]),
    "ea_create_ex": (_i, [C.POINTER(ea_params), C.POINTER(_vp)]),
    "ea_workspace_bytes_ex": (C.c_size_t, [_i, _i, _i, _i]),
    "ea_destroy": (_i, [_vp]),
    "ea_sweep": (_i, [_vp, _u64]),
    "ea_half_sweep": (_i, [_vp, _i]),
    "ea_get_time": (_i, [_vp, C.POINTER(_u64)]),
    "ea_set_time": (_i, [_vp, _u64]),
    "ea_set_temperature": (_i, [_vp, _dbl]),
    "ea_get_thresholds": (_i, [_vp, C.POINTER(_u64)]),
    "ea_set_dynamics": (_i, [_vp, _i]),
    "ea_get_dynamics": (_i, [_vp, C.POINTER(_i)]),
    "ea_get_thresholds_heatbath": (_i, [_vp, C.POINTER(_u64)]),
    "ea_set_kernel": (_i, [_vp, _i]),
    "ea_set_concurrency_hint": (_i, [_vp, _i]),
    "ea_get_kernel": (_i, [_vp, C.POINTER(_i)]),
    "ea_synchronize": (_i, [_vp]),
    "ea_get_launch_count": (_i, [_vp, C.POINTER(_u64)]),
    "ea_snapshot": (_i, [_vp, _i]),
    "ea_autocorr": (_i, [_vp, _i, _vp, _vp]),
    "ea_c4": (_i, [_vp, _i, _vp, _vp, _vp]),
    "ea_c4_vectors": (_i, [_vp, C.c_int64, _vp, _vp]),
    "ea_c4_vectors_static": (_i, [_vp, C.c_int64, _vp, _vp]),
    "ea_c4_shells": (_i, [_vp, _i, _vp, _vp]),
    "ea_c4_curve": (_i, [_vp, _vp, _i, _i, C.c_int64, _i, C.POINTER(_i), _vp, _vp, _vp]),
    "ea_integral_estimator": (_i, [_i, _vp, _vp, _vp, _i, _vp]),
    "ea_energy": (_i, [_vp, _vp]),
    "ea_magnetisation": (_i, [_vp, _vp]),
    "ea_measure": (_i, [_vp, _i, _i, _vp, _vp, _vp, _vp, _vp]),
    "ea_get_spins": (_i, [_vp, _vp]),
    "ea_set_spins": (_i, [_vp, _vp]),
    "ea_get_bonds": (_i, [_vp, _vp]),
    "ea_set_bonds": (_i, [_vp, _vp]),
    "ea_get_snapshot": (_i, [_vp, _i, _vp]),
    "ea_batch_create": (_i, [_vp, _i, C.POINTER(_vp)]),
    "ea_batch_sweep": (_i, [_vp, _u64]),
    "ea_batch_destroy": (_i, [_vp]),
    "ea_selftest_host": (_i, []),
    "ea_selftest_pipes": (_i, [_i, C.POINTER(_dbl)]),
    "ea_philox_selftest": (_i, [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]),
    "ea_strerror": (C.c_char_p, [_i]),
    "ea_last_error": (C.c_char_p, [_vp]),
    "ea_version": (C.c_char_p, []),
}

_lib = None


def lib():
    """Load libea_b200.so (built by `python -m paper_1411_5512_b200.build`).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OSError("libea_b200.so is not built (run `python -m paper_1411_5512_b200.build`); "
                          "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _ptr(a):
    """Host pointer of a numpy array or a torch CPU tensor (contiguous)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.device.type == "cpu" and a.is_contiguous()  # torch tensor (possibly pinned)
    return a.data_ptr()


class Sim:
    """One batch of 64 samples on an L^3 lattice on the GPU.  Methods mirror the C entry points."""

    def __init__(self, L, p, T, n_replicas=1, seed=0, n_slots=2, kernel="auto", device=None, stream=None,
                 torch_workspace=True, n_samples=LANES, workspace=None):
        """workspace: (device pointer, owner) of caller-placed device memory of >= workspace_bytes(...) bytes,
        256-byte aligned; `owner` is kept alive with the sim.  Default: a torch tensor (torch_workspace=True) or
        the library's own cudaMalloc (torch_workspace=False)."""
        self._h = _vp()
        self.L, self.N, self.n_replicas, self.n_slots = int(L), int(L) ** 3, int(n_replicas), int(n_slots)
        self.n_samples = int(n_samples)
        prm = ea_params()
        prm.L, prm.n_samples, prm.n_replicas, prm.n_slots = int(L), int(n_samples), int(n_replicas), int(n_slots)
        prm.p, prm.T, prm.seed = float(p), float(T), int(seed)
        prm.kernel = KERNEL_NAMES[kernel] if isinstance(kernel, str) else int(kernel)
        prm.device = -1 if device is None else int(device)
        self._ws = None
        self._stream = stream
        if stream is not None:  # a torch.cuda.Stream: the library launches on it
            prm.stream = stream.cuda_stream
        nbytes = lib().ea_workspace_bytes_ex(int(L), int(n_samples), int(n_replicas), int(n_slots))
        if workspace is not None:
            ptr, self._ws = workspace
            if int(ptr) % 256:
                raise EAError(EA_ERR_INVALID, "workspace pointer must be 256-byte aligned")
            prm.d_workspace, prm.workspace_bytes = int(ptr), nbytes
        elif torch_workspace and nbytes:
            import torch  # device memory only
            if not torch.cuda.is_available():
                raise EAError(EA_ERR_CUDA, "no CUDA device (there is no CPU fallback)")
            dev = torch.device("cuda", torch.cuda.current_device() if device is None else int(device))
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
            base = self._ws.data_ptr()
            prm.d_workspace = (base + 255) & ~255
            prm.workspace_bytes = nbytes
            # the block may be recycled from a tensor that work queued on torch's current stream still uses, while
            # the library writes it on its own stream: order the two once, here
            torch.cuda.current_stream(dev).synchronize()
        st = lib().ea_create_ex(C.byref(prm), C.byref(self._h))
        if st != EA_OK:
            self._h = _vp()
            raise EAError(st, lib().ea_strerror(st).decode() + " (ea_create_ex)")

    @property
    def lane_mask(self):
        """64-lane mask of the samples this sim carries (n_samples < 64: reading C-M)."""
        M = self.n_samples
        if M == LANES:
            return 0xFFFFFFFFFFFFFFFF
        if self.n_replicas == 2:
            h = (1 << (M // 2)) - 1
            return h | (h << 32)
        return (1 << M) - 1

    # -- plumbing -----------------------------------------------------------------------------------
    def _ck(self, st):
        if st != EA_OK:
            raise EAError(st, lib().ea_last_error(self._h).decode() or lib().ea_strerror(st).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().ea_destroy(self._h)
            self._h = _vp()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- dynamics -------------------------------------------------------------------------------------
    def sweep(self, n=1):
        if int(n) < 0:
            raise ValueError("sweep count must be >= 0 (got %d)" % int(n))  # would wrap to 2^64 - |n| in the C ABI
        self._ck(lib().ea_sweep(self._h, int(n)))

    def half_sweep(self, parity):
        self._ck(lib().ea_half_sweep(self._h, int(parity)))

    def synchronize(self):
        self._ck(lib().ea_synchronize(self._h))

    @property
    def launch_count(self):
        n = _u64()
        self._ck(lib().ea_get_launch_count(self._h, C.byref(n)))
        return n.value

    @property
    def time(self):
        t = _u64()
        self._ck(lib().ea_get_time(self._h, C.byref(t)))
        return t.value

    @time.setter
    def time(self, t):
        self._ck(lib().ea_set_time(self._h, int(t)))

    def set_temperature(self, T):
        self._ck(lib().ea_set_temperature(self._h, float(T)))

    @property
    def thresholds(self):
        thr = (_u64 * 3)()
        self._ck(lib().ea_get_thresholds(self._h, thr))
        return np.array(list(thr), dtype=np.uint64)

    def set_dynamics(self, dynamics):
        """"metropolis" (the paper's, Eq. 9) or "heatbath" (reading C-HB)."""
        code = {"metropolis": 0, "heatbath": 1}[dynamics] if isinstance(dynamics, str) else int(dynamics)
        self._ck(lib().ea_set_dynamics(self._h, code))

    @property
    def thresholds_heatbath(self):
        thr = (C.c_uint64 * 7)()
        self._ck(lib().ea_get_thresholds_heatbath(self._h, thr))
        return np.array(list(thr), dtype=np.uint64)

    @property
    def kernel(self):
        k = _i()
        self._ck(lib().ea_get_kernel(self._h, C.byref(k)))
        return k.value

    @kernel.setter
    def kernel(self, k):
        self._ck(lib().ea_set_kernel(self._h, KERNEL_NAMES[k] if isinstance(k, str) else int(k)))

    def set_concurrency_hint(self, n_concurrent_sims):
        """How many sims the caller advances at the same time on this device (never changes a result)."""
        self._ck(lib().ea_set_concurrency_hint(self._h, int(n_concurrent_sims)))

    # -- observables ----------------------------------------------------------------------------------
    def snapshot(self, slot):
        self._ck(lib().ea_snapshot(self._h, int(slot)))

    def autocorr(self, slot, with_C=False):
        A = np.zeros(LANES, dtype=np.int64)
        Cn = np.zeros(LANES, dtype=np.float64) if with_C else None
        self._ck(lib().ea_autocorr(self._h, int(slot), _ptr(A), _ptr(Cn)))
        return (A, Cn) if with_C else A

    def c4(self, r_max, with_q=False, with_avg=False):
        B = np.zeros((3, r_max + 1, 32), dtype=np.int64)
        q = np.zeros(32, dtype=np.int64) if with_q else None
        avg = np.zeros(r_max + 1, dtype=np.float64) if with_avg else None
        self._ck(lib().ea_c4(self._h, int(r_max), _ptr(B), _ptr(q), _ptr(avg)))
        out = (B,) + ((q,) if with_q else ()) + ((avg,) if with_avg else ())
        return out if len(out) > 1 else B

    def c4_vectors(self, vectors):
        """B[v, b] = sum_i q_i q_{i + r_v} for lattice vectors r_v = vectors[v] = (dx, dy, dz)."""
        v = np.ascontiguousarray(vectors, dtype=np.int32).reshape(-1, 3)
        B = np.zeros((v.shape[0], 32), dtype=np.int64)
        self._ck(lib().ea_c4_vectors(self._h, v.shape[0], _ptr(v), _ptr(B)))
        return B

    def c4_vectors_static(self, vectors):
        """c4_vectors for at most C4_STATIC_MAX_VECTORS vectors without any allocation in the library (static device scratch)."""
        v = np.ascontiguousarray(vectors, dtype=np.int32).reshape(-1, 3)
        B = np.zeros((v.shape[0], 32), dtype=np.int64)
        self._ck(lib().ea_c4_vectors_static(self._h, v.shape[0], _ptr(v), _ptr(B)))
        return B

    def c4_shells(self, r_max):
        """(S, mult): shell sums of B over the cube |component| <= r_max by squared length d2 = 0..3 r_max^2."""
        n_bins = 3 * r_max * r_max + 1
        S = np.zeros((n_bins, 32), dtype=np.int64)
        mult = np.zeros(n_bins, dtype=np.int64)
        self._ck(lib().ea_c4_shells(self._h, int(r_max), _ptr(S), _ptr(mult)))
        return S, mult

    def energy(self):
        E = np.zeros(LANES, dtype=np.int64)
        self._ck(lib().ea_energy(self._h, _ptr(E)))
        return E

    def magnetisation(self):
        M = np.zeros(LANES, dtype=np.int64)
        self._ck(lib().ea_magnetisation(self._h, _ptr(M)))
        return M

    def measure(self, slot=None, r_max=None, energy=True, magnetisation=True):
        """One measure point in one call (ea_measure): dict with A (if slot is given), B and q (if r_max is given; 2 replicas),
        E, M -- the same integers as the separate calls."""
        out = {}
        A = np.zeros(LANES, dtype=np.int64) if slot is not None else None
        B = np.zeros((3, int(r_max) + 1, LANES // 2), dtype=np.int64) if r_max is not None else None
        q = np.zeros(LANES // 2, dtype=np.int64) if r_max is not None else None
        E = np.zeros(LANES, dtype=np.int64) if energy else None
        M = np.zeros(LANES, dtype=np.int64) if magnetisation else None
        nul = C.c_void_p(None)
        self._ck(lib().ea_measure(self._h, -1 if slot is None else int(slot), 0 if r_max is None else int(r_max),
                                  nul if A is None else _ptr(A), nul if B is None else _ptr(B), nul if q is None else _ptr(q),
                                  nul if E is None else _ptr(E), nul if M is None else _ptr(M)))
        for k, v in (("A", A), ("B", B), ("q", q), ("E", E), ("M", M)):
            if v is not None:
                out[k] = v
        return out

    # -- canonical packed I/O -----------------------------------------------------------------------------
    def get_spins(self, out=None):
        w = np.zeros(self.N, dtype=np.uint64) if out is None else out
        self._ck(lib().ea_get_spins(self._h, _ptr(w)))
        return w

    def set_spins(self, words):
        if isinstance(words, np.ndarray):
            words = np.ascontiguousarray(words, dtype=np.uint64)
            assert words.shape == (self.N,)
        self._ck(lib().ea_set_spins(self._h, _ptr(words)))

    def get_bonds(self, out=None):
        w = np.zeros(3 * self.N, dtype=np.uint64) if out is None else out
        self._ck(lib().ea_get_bonds(self._h, _ptr(w)))
        return w

    def set_bonds(self, words):
        if isinstance(words, np.ndarray):
            words = np.ascontiguousarray(words, dtype=np.uint64)
            assert words.shape == (3 * self.N,)
        self._ck(lib().ea_set_bonds(self._h, _ptr(words)))

    def get_snapshot(self, slot):
        w = np.zeros(self.N, dtype=np.uint64)
        self._ck(lib().ea_get_snapshot(self._h, int(slot), _ptr(w)))
        return w


class Batch:
    """K small sims (L = 16, 32, 64) advanced by one launch per colour (ea_batch_*).  The members stay usable."""

    def __init__(self, sims):
        self.sims = list(sims)
        arr = (_vp * len(self.sims))(*[s._h for s in self.sims])
        self._h = _vp()
        st = lib().ea_batch_create(arr, len(self.sims), C.byref(self._h))
        if st != EA_OK:
            self._h = _vp()
            raise EAError(st, lib().ea_strerror(st).decode() + " (ea_batch_create)")

    def sweep(self, n=1):
        if int(n) < 0:
            raise ValueError("sweep count must be >= 0")
        st = lib().ea_batch_sweep(self._h, int(n))
        if st != EA_OK:
            raise EAError(st, lib().ea_last_error(self.sims[0]._h).decode())

    def close(self):
        if self._h:
            lib().ea_batch_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def c4_curve(S, mult, N, r_lim):
    """Shell sums -> (r, c, e): radius, sample-mean C_4 and its standard error (host arithmetic in the library)."""
    S = np.ascontiguousarray(S, dtype=np.int64)
    mult = np.ascontiguousarray(mult, dtype=np.int64)
    n_bins, n_samples = S.shape
    r, c, e = (np.zeros(n_bins, dtype=np.float64) for _ in range(3))
    n = C.c_int(0)
    st = lib().ea_c4_curve(_ptr(S), _ptr(mult), n_bins, n_samples, int(N), int(r_lim), C.byref(n), _ptr(r), _ptr(c), _ptr(e))
    if st != 0:
        raise EAError(st, "ea_c4_curve: invalid argument")
    return r[:n.value].copy(), c[:n.value].copy(), e[:n.value].copy()


def integral_estimator(r, c, e, k):
    """(I_k, I_{k+1}, xi_k, r_cut) of Eq. 5-6 with the 3-sigma cut-off of PAPER.md:116."""
    r, c, e = (np.ascontiguousarray(a, dtype=np.float64) for a in (r, c, e))
    out = np.zeros(4, dtype=np.float64)
    st = lib().ea_integral_estimator(len(r), _ptr(r), _ptr(c), _ptr(e), int(k), _ptr(out))
    if st != 0:
        raise EAError(st, "ea_integral_estimator: invalid argument")
    return tuple(float(x) for x in out)


def workspace_bytes(L, n_replicas=1, n_slots=2, n_samples=LANES):
    return int(lib().ea_workspace_bytes_ex(int(L), int(n_samples), int(n_replicas), int(n_slots)))


def selftest_pipes(device=None):
    """Measured issue rates (ea_selftest_pipes): dict of warp instructions per second and the SM clock."""
    out = (_dbl * 8)()
    st = lib().ea_selftest_pipes(-1 if device is None else int(device), out)
    if st != EA_OK:
        raise EAError(st, "ea_selftest_pipes: " + lib().ea_strerror(st).decode())
    return {"lop3_warp_inst_per_s": out[0], "imad_wide_warp_inst_per_s": out[1], "popc_warp_inst_per_s": out[2],
            "lop3_with_imad_wide_warp_inst_per_s": out[3], "sm_mhz": out[4], "n_sm": int(out[5]),
            "lop3_with_imad_warp_inst_per_s": out[6]}


def philox_selftest(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    st = lib().ea_philox_selftest(c, k, o)
    if st != EA_OK:
        raise EAError(st, "ea_philox_selftest")
    return [int(x) for x in o]


def version():
    return lib().ea_version().decode()
