"""CPU oracle for the +-J Edwards-Anderson checkerboard sweep (TEST INFRASTRUCTURE).

Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference`
legs may import this package.  It never imports the CUDA path
(`paper_1411_5512_b200`) and the CUDA path never imports it.

`Oracle` is a thin ctypes view of oracle/ea_oracle.c; every piece of arithmetic lives in
the C file, next to the PAPER.md passage it follows.
"""
import ctypes as C

import numpy as np

from . import build as _build

LANES = 64
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, i32, i64, u64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_double
        pu32, pu64, pi64 = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_int64)
        sig = {
            "oracle_philox4x32_10": (None, [pu32, pu32, pu32]),
            "oracle_thresholds": (None, [dbl, pu64]),
            "oracle_thresholds_heatbath": (None, [dbl, pu64]),
            "oracle_accept_heatbath": (i32, [pu64, i32, C.c_uint32]),
            "oracle_set_dynamics": (i32, [vp, i32]),
            "oracle_bond_threshold": (u64, [dbl]),
            "oracle_accept": (i32, [pu64, i32, C.c_uint32]),
            "oracle_shift": (i64, [i32, i64, i32, i32]),
            "oracle_neighbour": (i64, [i32, i64, i32, i32]),
            "oracle_local_sum": (i32, [vp, i32, i64]),
            "oracle_create": (vp, [i32, dbl, dbl, i32, u64, i32]),
            "oracle_destroy": (None, [vp]),
            "oracle_set_temperature": (None, [vp, dbl]),
            "oracle_get_thresholds": (None, [vp, pu64]),
            "oracle_get_time": (u64, [vp]),
            "oracle_set_time": (None, [vp, u64]),
            "oracle_set_order": (None, [vp, i32]),
            "oracle_set_threads": (None, [i32]),
            "oracle_get_max_threads": (i32, []),
            "oracle_spin_bytes": (C.POINTER(C.c_int8), [vp]),
            "oracle_bond_bytes": (C.POINTER(C.c_int8), [vp]),
            "oracle_dE_accum": (pi64, [vp]),
            "oracle_half_sweep": (None, [vp, i32]),
            "oracle_sweep": (None, [vp, u64]),
            "oracle_energy": (None, [vp, pi64]),
            "oracle_magnetisation": (None, [vp, pi64]),
            "oracle_snapshot": (i32, [vp, i32]),
            "oracle_autocorr": (i32, [vp, i32, pi64]),
            "oracle_overlap": (i32, [vp, pi64]),
            "oracle_c4_one": (i32, [vp, i32, i32, pi64]),
            "oracle_c4": (i32, [vp, i32, pi64]),
            "oracle_c4_vector": (i32, [vp, i32, i32, i32, pi64]),
            "oracle_c4_shells": (i32, [vp, i32, pi64, pi64]),
            "oracle_get_spins": (None, [vp, pu64]),
            "oracle_set_spins": (None, [vp, pu64]),
            "oracle_get_bonds": (None, [vp, pu64]),
            "oracle_set_bonds": (None, [vp, pu64]),
            "oracle_get_snapshot": (None, [vp, i32, pu64]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def thresholds(T):
    thr = np.zeros(3, dtype=np.uint64)
    lib().oracle_thresholds(float(T), _p(thr, C.c_uint64))
    return thr


def thresholds_heatbath(T):
    """thr[n_u] = floor(2^32 / (1 + exp((12 - 4 n_u) / T)) + 0.5), n_u = 0..6 (reading C-HB)."""
    thr = np.zeros(7, dtype=np.uint64)
    lib().oracle_thresholds_heatbath(float(T), _p(thr, C.c_uint64))
    return thr


def accept_heatbath(thr, local_sum, r):
    t = np.ascontiguousarray(thr, dtype=np.uint64)
    return bool(lib().oracle_accept_heatbath(_p(t, C.c_uint64), int(local_sum), int(r)))


def bond_threshold(p):
    return int(lib().oracle_bond_threshold(float(p)))


def accept(thr, local_sum, r):
    thr = np.asarray(thr, dtype=np.uint64)
    return bool(lib().oracle_accept(_p(thr, C.c_uint64), int(local_sum), int(r)))


def set_threads(n):
    lib().oracle_set_threads(int(n))


def max_threads():
    return int(lib().oracle_get_max_threads())


class Oracle:
    """One batch of 64 samples on an L^3 lattice, stepped by the C oracle."""

    def __init__(self, L, p, T, n_replicas=1, seed=0, n_slots=2):
        self._h = lib().oracle_create(int(L), float(p), float(T), int(n_replicas), int(seed), int(n_slots))
        if not self._h:
            raise ValueError("oracle_create rejected the parameters")
        self.L, self.N, self.n_replicas, self.n_slots = int(L), int(L) ** 3, int(n_replicas), int(n_slots)

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    # --- dynamics -------------------------------------------------------------------
    def sweep(self, n=1):
        lib().oracle_sweep(self._h, int(n))

    def half_sweep(self, parity):
        lib().oracle_half_sweep(self._h, int(parity))

    def set_order(self, order):
        lib().oracle_set_order(self._h, int(order))

    def set_temperature(self, T):
        lib().oracle_set_temperature(self._h, float(T))

    def set_dynamics(self, dynamics):
        """"metropolis" (Eq. 9, the paper's) or "heatbath" (reading C-HB)."""
        code = {"metropolis": 0, "heatbath": 1}[dynamics]
        if lib().oracle_set_dynamics(self._h, code):
            raise ValueError("bad dynamics")

    @property
    def thresholds(self):
        thr = np.zeros(3, dtype=np.uint64)
        lib().oracle_get_thresholds(self._h, _p(thr, C.c_uint64))
        return thr

    @property
    def time(self):
        return int(lib().oracle_get_time(self._h))

    @time.setter
    def time(self, t):
        lib().oracle_set_time(self._h, int(t))

    def local_sum(self, lane, site):
        return int(lib().oracle_local_sum(self._h, int(lane), int(site)))

    # --- raw +-1 byte views (numpy pins) ----------------------------------------------
    def spin_bytes(self):
        """View int8 [64][N] of +-1 (no copy)."""
        ptr = lib().oracle_spin_bytes(self._h)
        return np.ctypeslib.as_array(ptr, shape=(LANES, self.N))

    def bond_bytes(self):
        """View int8 [64][3][N] of +-1 (no copy)."""
        ptr = lib().oracle_bond_bytes(self._h)
        return np.ctypeslib.as_array(ptr, shape=(LANES, 3, self.N))

    def dE_accum(self):
        ptr = lib().oracle_dE_accum(self._h)
        return np.ctypeslib.as_array(ptr, shape=(LANES,)).copy()

    # --- observables ------------------------------------------------------------------
    def energy(self):
        E = np.zeros(LANES, dtype=np.int64)
        lib().oracle_energy(self._h, _p(E, C.c_int64))
        return E

    def magnetisation(self):
        M = np.zeros(LANES, dtype=np.int64)
        lib().oracle_magnetisation(self._h, _p(M, C.c_int64))
        return M

    def snapshot(self, slot):
        if lib().oracle_snapshot(self._h, int(slot)):
            raise ValueError("bad slot")

    def autocorr(self, slot):
        A = np.zeros(LANES, dtype=np.int64)
        if lib().oracle_autocorr(self._h, int(slot), _p(A, C.c_int64)):
            raise ValueError("bad or unset slot")
        return A

    def overlap(self):
        q = np.zeros(32, dtype=np.int64)
        if lib().oracle_overlap(self._h, _p(q, C.c_int64)):
            raise ValueError("overlap needs n_replicas == 2")
        return q

    def c4_one(self, d, r):
        B = np.zeros(32, dtype=np.int64)
        if lib().oracle_c4_one(self._h, int(d), int(r), _p(B, C.c_int64)):
            raise ValueError("bad c4 arguments")
        return B

    def c4(self, r_max):
        B = np.zeros((3, r_max + 1, 32), dtype=np.int64)
        if lib().oracle_c4(self._h, int(r_max), _p(B, C.c_int64)):
            raise ValueError("bad c4 arguments")
        return B

    def c4_vector(self, dx, dy, dz):
        """B_b(r) = sum_i q_i q_{i+r} for the lattice vector r = (dx, dy, dz) (Eq. 3; reading C-S8v)."""
        B = np.zeros(32, dtype=np.int64)
        if lib().oracle_c4_vector(self._h, int(dx), int(dy), int(dz), _p(B, C.c_int64)):
            raise ValueError("c4_vector needs n_replicas == 2")
        return B

    def c4_shells(self, r_max):
        """(S, mult): S[d2, b] = sum of B_b(r) over all vectors with |r|^2 = d2 and components in
        [-r_max, r_max]; mult[d2] = their number; d2 = 0..3 r_max^2."""
        n_bins = 3 * r_max * r_max + 1
        S = np.zeros((n_bins, 32), dtype=np.int64)
        mult = np.zeros(n_bins, dtype=np.int64)
        if lib().oracle_c4_shells(self._h, int(r_max), _p(S, C.c_int64), _p(mult, C.c_int64)):
            raise ValueError("bad c4_shells arguments")
        return S, mult

    # --- canonical packed words ---------------------------------------------------------
    def get_spins(self):
        w = np.zeros(self.N, dtype=np.uint64)
        lib().oracle_get_spins(self._h, _p(w, C.c_uint64))
        return w

    def set_spins(self, words):
        w = np.ascontiguousarray(words, dtype=np.uint64)
        assert w.shape == (self.N,)
        lib().oracle_set_spins(self._h, _p(w, C.c_uint64))

    def get_bonds(self):
        w = np.zeros(3 * self.N, dtype=np.uint64)
        lib().oracle_get_bonds(self._h, _p(w, C.c_uint64))
        return w

    def set_bonds(self, words):
        w = np.ascontiguousarray(words, dtype=np.uint64)
        assert w.shape == (3 * self.N,)
        lib().oracle_set_bonds(self._h, _p(w, C.c_uint64))

    def get_snapshot(self, slot):
        w = np.zeros(self.N, dtype=np.uint64)
        lib().oracle_get_snapshot(self._h, int(slot), _p(w, C.c_uint64))
        return w


# ----------------------------------------------------------------------------------------------------
# Integral estimator of the coherence length (Eq. 5-6; procedure PAPER.md:116).
# Plain fp64, in the paper's order; reading C-S12:
#   curve   : points (r_j, c_j, e_j), r ascending from r_0 = 0, c = sample mean of C_4, e = its standard error
#             over the disorder samples, restricted to r <= r_lim (Eq. 5 integrates to L/2)
#   cut-off : the integrals run "up to the point, where the value of C_4 first becomes smaller than three times
#             its error" (:116): j* = first j >= 1 with c_j < 3 e_j, points 0 .. j*-1 are used (all if none)
#   rule    : trapezoid on the (non-uniform) r grid:  I_k = sum_j (r_j^k c_j + r_{j+1}^k c_{j+1}) (r_{j+1} - r_j) / 2
#   the paper then adds the tail of its fitted function (4); fits are out of scope, so NO tail is added
#   xi_k = I_{k+1} / I_k
# ----------------------------------------------------------------------------------------------------
def c4_curve(S, mult, N, r_lim):
    """Shell sums -> (r, c, e).  c_b(d2) = S[d2, b] / (mult[d2] N) per disorder sample b; c = mean over b;
    e = sqrt(sum_b (c_b - c)^2 / (n (n - 1)))."""
    S = np.asarray(S, dtype=np.int64)
    mult = np.asarray(mult, dtype=np.int64)
    r, c, e = [], [], []
    n = S.shape[1]
    for d2 in range(S.shape[0]):
        if mult[d2] == 0 or d2 > r_lim * r_lim:
            continue
        cb = S[d2].astype(np.float64) / (float(mult[d2]) * float(N))
        mean = float(np.sum(cb)) / n
        var = float(np.sum((cb - mean) ** 2)) / (n * (n - 1))
        r.append(float(np.sqrt(float(d2))))
        c.append(mean)
        e.append(float(np.sqrt(var)))
    return np.array(r), np.array(c), np.array(e)


def integral_estimator(r, c, e, k):
    """(I_k, I_{k+1}, xi_k, r_cut) of Eq. 5-6 with the 3-sigma cut-off and the trapezoid rule stated above."""
    r = np.asarray(r, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    e = np.asarray(e, dtype=np.float64)
    n_use = len(r)
    for j in range(1, len(r)):
        if c[j] < 3.0 * e[j]:
            n_use = j
            break
    I = [0.0, 0.0]
    for m, kk in enumerate((k, k + 1)):
        acc = 0.0
        for j in range(n_use - 1):
            acc += 0.5 * (r[j] ** kk * c[j] + r[j + 1] ** kk * c[j + 1]) * (r[j + 1] - r[j])
        I[m] = acc
    xi = I[1] / I[0] if I[0] != 0.0 else float("nan")
    return I[0], I[1], xi, float(r[n_use - 1])
