"""ctypes front-end of the CPU oracle (oracle/cg_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports paper_1407_5026_b200 (the CUDA path).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cg_oracle.c")
_HDR = os.path.join(_HERE, "cg_oracle.h")
_LIB = os.path.join(_HERE, "libcgo.so")

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-std=c11",
          "-D_POSIX_C_SOURCE=200809L", "-Wall", "-Wextra", "-shared", "-fPIC"]


def build(force=False):
    """Compile the oracle with gcc (plain C, FMA contraction off)."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u64, u32, i64, dbl, vp = C.c_uint64, C.c_uint32, C.c_int64, C.c_double, C.c_void_p
        P = C.POINTER
        sig = {
            "cgo_philox4x32_10": (None, [P(u32), P(u32), P(u32)]),
            "cgo_pr_split": (None, [u64, u32, P(u64), P(u32)]),
            "cgo_init": (C.c_int, [P(vp), C.c_int, dbl, dbl, dbl, dbl, u64, u32]),
            "cgo_init3": (C.c_int, [P(vp), C.c_int, dbl, dbl, dbl, dbl, u64, u32]),
            "cgo_get_dz": (C.c_int, [vp, vp]),
            "cgo_dimension": (C.c_int, [vp]),
            "cgo_free": (None, [vp]),
            "cgo_run": (C.c_int, [vp, u64]),
            "cgo_get_state": (C.c_int, [vp, vp, vp, P(dbl), P(i64)]),
            "cgo_get_counters": (C.c_int, [vp, P(u64), P(u64), P(u64), P(u64)]),
            "cgo_enable_hop_log": (C.c_int, [vp, C.c_int]),
            "cgo_get_hops": (C.c_int, [vp, u64, u64, vp, vp, vp]),
            "cgo_recompute_eps": (C.c_int, [vp, vp, P(dbl)]),
            "cgo_num_displacements": (i64, [vp]),
            "cgo_get_tables": (C.c_int, [vp, vp, vp, vp, vp, P(dbl), P(dbl)]),
            "cgo_invr_sites": (dbl, [vp, u32, u32]),
            "cgo_get_phi": (C.c_int, [vp, vp]),
            "cgo_decode_attempt": (C.c_int, [vp, u64, P(u32), P(u32), P(i64), P(dbl), P(dbl)]),
            "cgo_set_state": (C.c_int, [vp, vp, u64]),
            "cgo_set_phi": (C.c_int, [vp, vp]),
            "cgo_set_fixed_A": (C.c_int, [vp, dbl]),
            "cgo_apply_hops": (C.c_int, [vp, u64, vp, vp]),
            "cgo_near_ties": (u64, [vp]),
            "cgo_exp_evaluations": (u64, [vp]),
            "cgo_update_seconds": (dbl, [vp]),
            "cgo_normal_of_hop": (dbl, [vp, u64]),
            "cgo_get_time_stochastic": (C.c_int, [vp, P(dbl)]),
            "cgo_dos": (C.c_int, [vp, dbl, dbl, u32, vp, P(u64)]),
            "cgo_get_series": (C.c_int, [vp, u64, u64, vp, vp]),
            "cgo_sigma0": (C.c_int, [vp, P(dbl)]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().cgo_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def pr_split(m, M):
    p, q = C.c_uint64(), C.c_uint32()
    lib().cgo_pr_split(int(m), int(M), C.byref(p), C.byref(q))
    return p.value, q.value


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    """cgo_init / cgo_run / cgo_get_state with the same shape as the CUDA binding."""

    def __init__(self, L, W=1.0, xi=1.0, T=0.05, E=0.0, seed=1, M=1, hop_log=True, dim=2):
        self._h = C.c_void_p()
        assert dim in (2, 3)
        init = lib().cgo_init if dim == 2 else lib().cgo_init3
        rc = init(C.byref(self._h), int(L), float(W), float(xi), float(T), float(E), int(seed), int(M))
        if rc != 0:
            raise ValueError("cgo_init%s failed with code %d" % ("" if dim == 2 else "3", rc))
        self.L, self.N, self.M, self.dim = int(L), int(L) ** dim, int(M), dim
        if hop_log:
            lib().cgo_enable_hop_log(self._h, 1)

    def close(self):
        if self._h:
            lib().cgo_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            raise RuntimeError("oracle call failed with code %d" % rc)

    def run(self, n_hops):
        self._check(lib().cgo_run(self._h, int(n_hops)))

    def state(self):
        n = np.empty(self.N, np.int8)
        eps = np.empty(self.N, np.float64)
        t, dP = C.c_double(), C.c_int64()
        self._check(lib().cgo_get_state(self._h, _ptr(n), _ptr(eps), C.byref(t), C.byref(dP)))
        return n, eps, t.value, dP.value

    def counters(self):
        a, pe, it, h = C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_uint64()
        self._check(lib().cgo_get_counters(self._h, C.byref(a), C.byref(pe), C.byref(it), C.byref(h)))
        return {"attempts": a.value, "proposals_evaluated": pe.value,
                "iterations": it.value, "hops": h.value}

    def hops(self, first=0, count=None):
        if count is None:
            count = self.counters()["hops"] - first
        a = np.empty(count, np.uint64)
        i = np.empty(count, np.uint32)
        j = np.empty(count, np.uint32)
        self._check(lib().cgo_get_hops(self._h, int(first), int(count), _ptr(a), _ptr(i), _ptr(j)))
        return a, i, j

    def recompute_eps(self):
        eps = np.empty(self.N, np.float64)
        dev = C.c_double()
        self._check(lib().cgo_recompute_eps(self._h, _ptr(eps), C.byref(dev)))
        return eps, dev.value

    def tables(self):
        K = lib().cgo_num_displacements(self._h)
        dz = np.empty(K, np.int32)
        dy = np.empty(K, np.int32)
        dx = np.empty(K, np.int32)
        cdf = np.empty(K, np.float64)
        invr = np.empty(K, np.float64)
        S, G = C.c_double(), C.c_double()
        self._check(lib().cgo_get_tables(self._h, _ptr(dy), _ptr(dx), _ptr(cdf), _ptr(invr),
                                         C.byref(S), C.byref(G)))
        self._check(lib().cgo_get_dz(self._h, _ptr(dz)))
        return {"K": K, "dz": dz, "dy": dy, "dx": dx, "cdf": cdf, "invr_k": invr, "S": S.value,
                "Gamma": G.value}

    def invr_sites(self, a, b):
        return lib().cgo_invr_sites(self._h, int(a), int(b))

    def phi(self):
        phi = np.empty(self.N, np.float64)
        self._check(lib().cgo_get_phi(self._h, _ptr(phi)))
        return phi

    def decode_attempt(self, a):
        i, j, k = C.c_uint32(), C.c_uint32(), C.c_int64()
        ud, ua = C.c_double(), C.c_double()
        self._check(lib().cgo_decode_attempt(self._h, int(a), C.byref(i), C.byref(j), C.byref(k),
                                             C.byref(ud), C.byref(ua)))
        return i.value, j.value, k.value, ud.value, ua.value

    def set_state(self, n, next_attempt=0):
        n = np.ascontiguousarray(n, np.int8)
        assert n.size == self.N
        self._check(lib().cgo_set_state(self._h, _ptr(n), int(next_attempt)))

    def set_phi(self, phi):
        phi = np.ascontiguousarray(phi, np.float64)
        assert phi.size == self.N
        self._check(lib().cgo_set_phi(self._h, _ptr(phi)))

    def set_fixed_A(self, A):
        self._check(lib().cgo_set_fixed_A(self._h, float(A)))

    def apply_hops(self, i, j):
        i = np.ascontiguousarray(i, np.uint32)
        j = np.ascontiguousarray(j, np.uint32)
        assert i.size == j.size
        self._check(lib().cgo_apply_hops(self._h, int(i.size), _ptr(i), _ptr(j)))

    def near_ties(self):
        return lib().cgo_near_ties(self._h)

    def exp_evaluations(self):
        return lib().cgo_exp_evaluations(self._h)

    def update_seconds(self):
        return lib().cgo_update_seconds(self._h)

    # ---- observables (O11-O14 in cg_oracle.h)
    def normal_of_hop(self, h):
        return lib().cgo_normal_of_hop(self._h, int(h))

    def time_stochastic(self):
        t = C.c_double()
        self._check(lib().cgo_get_time_stochastic(self._h, C.byref(t)))
        return t.value

    def dos(self, lo, width, nbins):
        hist = np.zeros(nbins, np.uint64)
        out = C.c_uint64()
        self._check(lib().cgo_dos(self._h, float(lo), float(width), int(nbins), _ptr(hist), C.byref(out)))
        return hist, out.value

    def series(self, first=0, count=None):
        if count is None:
            count = self.counters()["hops"] - first
        t = np.empty(count, np.float64)
        P = np.empty(count, np.int64)
        self._check(lib().cgo_get_series(self._h, int(first), int(count), _ptr(t), _ptr(P)))
        return t, P

    def sigma0(self):
        v = C.c_double()
        self._check(lib().cgo_sigma0(self._h, C.byref(v)))
        return v.value
