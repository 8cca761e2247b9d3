"""Thin ctypes binding of libcg.so (include/cg.h).  Argument marshalling only.

PyTorch supplies device memory (the workspace and hop-log tensors) and the CUDA
stream; every step of the hot path runs in the library's kernels.  There is no CPU
fallback: if the library or a CUDA device is missing, construction raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcg.so")
_lib = None

CG_OK, CG_EINVAL, CG_ENOMEM, CG_ECUDA, CG_EUNSUPPORTED, CG_EDEVICE = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "cg_init", "cg_workspace_bytes", "cg_init_ws", "cg_init3", "cg_workspace_bytes3", "cg_init3_ws",
    "cg_run", "cg_run_many", "cg_get_state", "cg_set_state",
    "cg_get_time_stochastic", "cg_get_normals", "cg_get_dos", "cg_get_dos_noalloc", "cg_get_series", "cg_get_sigma0",
    "cg_get_counters", "cg_enable_hop_log", "cg_get_hops", "cg_recompute_eps", "cg_apply_hops",
    "cg_set_update_kernel", "cg_get_table_sizes", "cg_get_tables", "cg_get_table_dz", "cg_get_phi", "cg_set_launch", "cg_get_launch", "cg_get_kernel",
    "cg_set_tuning", "cg_get_tuning", "cg_get_labels_per_thread", "cg_set_phase_timers", "cg_get_phase_cycles", "cg_get_exchange_cycles", "cg_bench_l2", "cg_free", "cg_strerror",
    "cg_last_error",
]


class CgError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("libcg: %s (code %d)" % (text, code))
        self.code = code


def lib():
    """Load libcg.so (built in-tree by paper_1407_5026_b200/build.py); never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("libcg.so is not built; run `python -m paper_1407_5026_b200.build` "
                          "or __graft_entry__.build()")
    L = C.CDLL(_LIB_PATH)
    u64, u32, i64, dbl, vp, sz, ci = (C.c_uint64, C.c_uint32, C.c_int64, C.c_double, C.c_void_p,
                                      C.c_size_t, C.c_int)
    P = C.POINTER
    sig = {
        "cg_init": (ci, [P(vp), ci, dbl, dbl, dbl, dbl, u64, u32]),
        "cg_workspace_bytes": (sz, [ci, u32]),
        "cg_init_ws": (ci, [P(vp), ci, dbl, dbl, dbl, dbl, u64, u32, vp, sz, vp]),
        "cg_init3": (ci, [P(vp), ci, dbl, dbl, dbl, dbl, u64, u32]),
        "cg_workspace_bytes3": (sz, [ci, u32]),
        "cg_init3_ws": (ci, [P(vp), ci, dbl, dbl, dbl, dbl, u64, u32, vp, sz, vp]),
        "cg_run": (ci, [vp, u64]),
        "cg_run_many": (ci, [P(vp), ci, u64]),
        "cg_get_state": (ci, [vp, vp, vp, P(dbl), P(i64)]),
        "cg_set_state": (ci, [vp, vp, vp, u64, u64, i64]),
        "cg_get_counters": (ci, [vp, P(u64), P(u64), P(u64), P(u64)]),
        "cg_enable_hop_log": (ci, [vp, u64, vp, sz]),
        "cg_get_hops": (ci, [vp, u64, u64, vp, vp, vp]),
        "cg_recompute_eps": (ci, [vp, P(dbl)]),
        "cg_get_time_stochastic": (ci, [vp, P(dbl)]),
        "cg_get_normals": (ci, [vp, u64, u64, vp]),
        "cg_get_dos": (ci, [vp, dbl, dbl, u32, vp, P(u64)]),
        "cg_get_dos_noalloc": (ci, [vp, dbl, dbl, u32, vp, P(u64)]),
        "cg_get_series": (ci, [vp, u64, u64, vp, vp]),
        "cg_get_sigma0": (ci, [vp, P(dbl)]),
        "cg_apply_hops": (ci, [vp, u64, vp, vp, P(C.c_float)]),
        "cg_set_update_kernel": (ci, [vp, ci]),
        "cg_get_table_sizes": (ci, [vp, P(i64), P(i64)]),
        "cg_get_tables": (ci, [vp, vp, vp, vp, vp, P(dbl), P(dbl)]),
        "cg_get_table_dz": (ci, [vp, vp]),
        "cg_get_phi": (ci, [vp, vp]),
        "cg_set_launch": (ci, [vp, ci, ci]),
        "cg_get_launch": (ci, [vp, P(ci), P(ci), P(ci)]),
        "cg_get_kernel": (ci, [vp, P(ci)]),
        "cg_set_tuning": (ci, [vp, ci, ci]),
        "cg_get_tuning": (ci, [vp, P(ci), P(ci)]),
        "cg_get_labels_per_thread": (ci, [vp, P(ci)]),
        "cg_get_exchange_cycles": (ci, [vp, vp]),
        "cg_set_phase_timers": (ci, [vp, ci]),
        "cg_get_phase_cycles": (ci, [vp, P(u64), P(u64), P(u64), P(u64), P(u64), ci]),
        "cg_bench_l2": (ci, [sz, ci, ci, ci, ci, ci, ci, P(dbl)]),
        "cg_free": (None, [vp]),
        "cg_strerror": (C.c_char_p, [ci]),
        "cg_last_error": (C.c_char_p, [vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


L2_MODES = {"rmw": 0, "read": 1, "write": 2}


def bench_l2(nbytes, reps=1000, trials=10, mode="rmw", ctas_per_sm=2, threads=512, vec_bytes=16):
    """cg_bench_l2: GB/s of L1-bypassing accesses over a resident buffer (read-modify-write counts both ways)."""
    out = C.c_double()
    rc = lib().cg_bench_l2(int(nbytes), int(reps), int(trials), L2_MODES[mode], int(ctas_per_sm), int(threads),
                           int(vec_bytes), C.byref(out))
    if rc != 0:
        raise CgError(rc, lib().cg_strerror(rc).decode())
    return out.value


def run_many(sims, n_accepted_hops):
    """cg_run_many: every sim of `sims` advances by n_accepted_hops in ONE persistent launch."""
    sims = list(sims)
    arr = (C.c_void_p * len(sims))(*[g._h for g in sims])
    with sims[0]._torch.cuda.device(sims[0].device):
        rc = lib().cg_run_many(arr, len(sims), int(n_accepted_hops))
    if rc != 0:
        text = lib().cg_last_error(sims[0]._h).decode() or lib().cg_strerror(rc).decode()
        raise CgError(rc, text)


class CoulombGlass:
    """cg_init / cg_run / cg_get_state on cuda:`device`."""

    def __init__(self, L, W=1.0, xi=1.0, T=0.05, E=0.0, seed=1, M=1024, hop_log=0, device=0,
                 stream=None, dim=2):
        import torch  # device memory and streams only
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1407_5026_b200 needs a CUDA device (no CPU fallback)")
        self._lib = lib()
        self._torch = torch
        self.device = torch.device("cuda", device)
        if dim not in (2, 3):
            raise ValueError("dim must be 2 (cg_init) or 3 (cg_init3)")
        self.L, self.N, self.M, self.dim = int(L), int(L) ** dim, int(M), dim
        self._h = C.c_void_p()
        ws_bytes = self._lib.cg_workspace_bytes if dim == 2 else self._lib.cg_workspace_bytes3
        init_ws = self._lib.cg_init_ws if dim == 2 else self._lib.cg_init3_ws
        with torch.cuda.device(self.device):
            nbytes = ws_bytes(self.L, self.M)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            # +256 so the base can be rounded up to the 256-byte alignment cg_init_ws asks for
            self._ws = torch.empty(max(nbytes, 1) + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) & ~255
            rc = init_ws(C.byref(self._h), self.L, float(W), float(xi), float(T), float(E),
                         int(seed), self.M, C.c_void_p(base), nbytes, C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            self._h = C.c_void_p()
            raise CgError(rc, self._lib.cg_strerror(rc).decode())
        self._log = None
        if hop_log:
            self.enable_hop_log(hop_log)

    # -- lifetime -------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._lib.cg_free(self._h)
            self._h = C.c_void_p()
            self._ws = None
            self._log = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != 0:
            text = self._lib.cg_strerror(rc).decode()
            if rc in (CG_ECUDA, CG_EDEVICE):
                text += ": " + self._lib.cg_last_error(self._h).decode()
            raise CgError(rc, text)

    # -- the three calls of the problem statement -----------------------------------------
    def run(self, n_accepted_hops):
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_run(self._h, int(n_accepted_hops)))

    def state(self):
        """-> (n[N] int8, eps[N] float64, t in tau0, dP)."""
        n = np.empty(self.N, np.int8)
        eps = np.empty(self.N, np.float64)
        t, dP = C.c_double(), C.c_int64()
        self._check(self._lib.cg_get_state(self._h, _ptr(n), _ptr(eps), C.byref(t), C.byref(dP)))
        return n, eps, t.value, dP.value

    def state_into(self, n, eps):
        """cg_get_state into caller-provided host arrays (e.g. pinned); -> (t, dP)."""
        t, dP = C.c_double(), C.c_int64()
        self._check(self._lib.cg_get_state(self._h, C.c_void_p(n.ctypes.data), C.c_void_p(eps.ctypes.data),
                                           C.byref(t), C.byref(dP)))
        return t.value, dP.value

    def set_state(self, n, eps, attempts, hops, dP):
        n = np.ascontiguousarray(n, np.int8)
        eps = np.ascontiguousarray(eps, np.float64)
        assert n.size == self.N and eps.size == self.N
        self._check(self._lib.cg_set_state(self._h, _ptr(n), _ptr(eps), int(attempts), int(hops), int(dP)))

    # -- diagnostics ------------------------------------------------------------------------
    def counters(self):
        a, pe, it, h = C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_uint64()
        self._check(self._lib.cg_get_counters(self._h, C.byref(a), C.byref(pe), C.byref(it), C.byref(h)))
        return {"attempts": a.value, "proposals_evaluated": pe.value, "iterations": it.value,
                "hops": h.value}

    def enable_hop_log(self, capacity):
        torch = self._torch
        capacity = int(capacity)
        self._log = torch.empty(16 * capacity + 8, dtype=torch.uint8, device=self.device) if capacity else None
        ptr = (self._log.data_ptr() + 7) & ~7 if capacity else 0
        with torch.cuda.device(self.device):
            self._check(self._lib.cg_enable_hop_log(self._h, capacity, C.c_void_p(ptr), 16 * capacity))
        self._log_cap, self._log_base = capacity, self.counters()["hops"]

    def hops(self, first=0, count=None):
        if count is None:
            count = self.logged_hops() - first
        a = np.empty(count, np.uint64)
        i = np.empty(count, np.uint32)
        j = np.empty(count, np.uint32)
        self._check(self._lib.cg_get_hops(self._h, int(first), int(count), _ptr(a), _ptr(i), _ptr(j)))
        return a, i, j

    def logged_hops(self):
        """Hops executed since the log was enabled, bounded by its capacity."""
        if self._log is None:
            return 0
        return min(self.counters()["hops"] - self._log_base, self._log_cap)

    # ---- observables (include/cg.h "Observables"): argument marshalling only
    def time_stochastic(self):
        t = C.c_double()
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_get_time_stochastic(self._h, C.byref(t)))
        return t.value

    def normals(self, first_hop, count):
        z = np.empty(int(count), np.float64)
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_get_normals(self._h, int(first_hop), int(count), _ptr(z)))
        return z

    def dos(self, lo, width, nbins):
        hist = np.zeros(int(nbins), np.uint64)
        outside = C.c_uint64()
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_get_dos(self._h, float(lo), float(width), int(nbins), _ptr(hist),
                                             C.byref(outside)))
        return hist, outside.value

    def dos_noalloc(self, lo, width, nbins, hist=None):
        """cg_get_dos_noalloc: the same counts; the kernel's scratch is a static device array of the library."""
        if hist is None:
            hist = np.zeros(int(nbins), np.uint64)
        outside = C.c_uint64()
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_get_dos_noalloc(self._h, float(lo), float(width), int(nbins), _ptr(hist),
                                                     C.byref(outside)))
        return hist, outside.value

    def series(self, first=0, count=None):
        if count is None:
            count = self.logged_hops() - first
        t = np.empty(int(count), np.float64)
        P = np.empty(int(count), np.int64)
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_get_series(self._h, int(first), int(count), _ptr(t), _ptr(P)))
        return t, P

    def sigma0(self):
        v = C.c_double()
        self._check(self._lib.cg_get_sigma0(self._h, C.byref(v)))
        return v.value

    def recompute_eps(self):
        dev = C.c_double()
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_recompute_eps(self._h, C.byref(dev)))
        return dev.value

    def apply_hops(self, i, j, kernel=None):
        """Scripted hops through the update kernel alone; -> device milliseconds of the launch.
        kernel: None/"auto", "gathers" or "staged" (cg_set_update_kernel)."""
        self._check(self._lib.cg_set_update_kernel(self._h, {None: 0, "auto": 0, "gathers": 1, "staged": 2}[kernel]))
        i = np.ascontiguousarray(i, np.uint32)
        j = np.ascontiguousarray(j, np.uint32)
        assert i.size == j.size
        ms = C.c_float()
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_apply_hops(self._h, int(i.size), _ptr(i), _ptr(j), C.byref(ms)))
        return ms.value

    def tables(self):
        K, KL = C.c_int64(), C.c_int64()
        self._check(self._lib.cg_get_table_sizes(self._h, C.byref(K), C.byref(KL)))
        n = KL.value
        dy = np.empty(n, np.int32); dx = np.empty(n, np.int32)
        cdf = np.empty(n, np.float64); invr = np.empty(n, np.float64)
        S, G = C.c_double(), C.c_double()
        self._check(self._lib.cg_get_tables(self._h, _ptr(dy), _ptr(dx), _ptr(cdf), _ptr(invr),
                                            C.byref(S), C.byref(G)))
        dz = np.empty(n, np.int32)
        self._check(self._lib.cg_get_table_dz(self._h, _ptr(dz)))
        return {"K": K.value, "K_live": n, "dz": dz, "dy": dy, "dx": dx, "cdf": cdf, "invr_k": invr,
                "S": S.value, "Gamma": G.value}

    def phi(self):
        phi = np.empty(self.N, np.float64)
        self._check(self._lib.cg_get_phi(self._h, _ptr(phi)))
        return phi

    def set_launch(self, n_ctas=0, threads=0):
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_set_launch(self._h, int(n_ctas), int(threads)))

    def launch(self):
        a, b, c = C.c_int(), C.c_int(), C.c_int()
        self._check(self._lib.cg_get_launch(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return {"n_ctas": a.value, "threads": b.value, "smem_bytes": c.value}

    def set_tuning(self, snapshot_interval=0, cluster_size=0):
        """cg_set_tuning: eps write-through every H hops, CTAs per thread-block cluster (0: unchanged)."""
        with self._torch.cuda.device(self.device):
            self._check(self._lib.cg_set_tuning(self._h, int(snapshot_interval), int(cluster_size)))

    def tuning(self):
        a, b = C.c_int(), C.c_int()
        self._check(self._lib.cg_get_tuning(self._h, C.byref(a), C.byref(b)))
        return {"snapshot_interval": a.value, "cluster_size": b.value}

    def exchange_cycles(self):
        """cg_get_exchange_cycles: where the exchange warps (all CTAs) spent their cycles, timed build."""
        a = np.zeros(6, np.uint64)
        self._check(self._lib.cg_get_exchange_cycles(self._h, _ptr(a)))
        return dict(zip(("recycle", "gate", "own_workers", "scan", "publish", "warps"), (int(v) for v in a)))

    def kernel(self):
        """'single' (cg_pr_single: one CTA, state in shared memory) or 'dataflow' (cg_pr_persistent)."""
        k = C.c_int()
        self._check(self._lib.cg_get_kernel(self._h, C.byref(k)))
        return "single" if k.value == 1 else "dataflow"

    def labels_per_thread(self):
        k = C.c_int()
        self._check(self._lib.cg_get_labels_per_thread(self._h, C.byref(k)))
        return k.value

    def set_phase_timers(self, on=True):
        self._check(self._lib.cg_set_phase_timers(self._h, 1 if on else 0))

    def phase_cycles(self, reset=False):
        """cg_get_phase_cycles: W_R / W_U of PAPER.md:106 from the persistent kernel itself (SM cycles)."""
        t, w, u, p, n = C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_uint64()
        self._check(self._lib.cg_get_phase_cycles(self._h, C.byref(t), C.byref(w), C.byref(u), C.byref(p),
                                                  C.byref(n), 1 if reset else 0))
        return {"total": t.value, "wait": w.value, "update": u.value, "propose": p.value, "warps": n.value}
