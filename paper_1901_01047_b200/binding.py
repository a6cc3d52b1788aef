"""ctypes binding of include/ctaux.h.  Same names as the C ABI; marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

LOG_DTYPE = np.dtype([("p", "<u8"), ("type", "<i4"), ("arg", "<i4"), ("tau", "<f8"),
                      ("spin", "<i4"), ("accepted", "<i4"), ("R", "<f8"), ("u", "<f8")])

STEP_CLASSES = ["prep", "cand_gemm", "propose", "build_uv", "flush_gemm", "rebuild", "other", "usinv_gemm"]


class CtauxError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__(f"{what}: code {code} ({detail})")
        self.code = code


class _Params(C.Structure):
    _fields_ = [("Lx", C.c_int32), ("Ly", C.c_int32), ("beta", C.c_double), ("U", C.c_double),
                ("K", C.c_double), ("n_tau", C.c_int32), ("g0_table", C.c_void_p),
                ("delay", C.c_int32), ("n_walkers", C.c_int32), ("init_k", C.c_int32),
                ("max_k", C.c_int32), ("rebuild_every", C.c_int32), ("log_capacity", C.c_int32),
                ("cand_window", C.c_int32), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("stream", C.c_void_p), ("guard_amp", C.c_double), ("fused_small", C.c_int32), ("rebuild_mode", C.c_int32), ("flip_moves", C.c_int32),
                ("n_tol", C.c_double), ("n_pairs", C.c_int32), ("pair_a", C.c_void_p), ("pair_b", C.c_void_p),
                ("pair_U", C.c_void_p), ("n_omega", C.c_int32), ("nfft_oversampling", C.c_int32), ("nfft_window", C.c_int32), ("graph_mode", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("proposals", C.c_uint64), ("next_id", C.c_uint64), ("acc_ins", C.c_int64),
                ("acc_rem", C.c_int64), ("sweeps", C.c_int64), ("blocks", C.c_int64),
                ("flushes", C.c_int64), ("rebuilds", C.c_int64), ("sum_rank", C.c_int64),
                ("k", C.c_int32), ("sign", C.c_int32), ("flops_cand", C.c_double),
                ("flops_flush", C.c_double), ("flops_rebuild", C.c_double),
                ("min_margin", C.c_double), ("sum_k", C.c_double), ("flops_usinv", C.c_double),
                ("guard_ends", C.c_int64), ("acc_flip", C.c_int64), ("monitor_rebuilds", C.c_int64),
                ("err_est", C.c_double), ("flops_cand_alg", C.c_double)]


# include/ctaux.h (the walker boundary) and include/ctaux_testing.h (test / measurement helpers)
EXPORTS = ["ctaux_workspace_bytes", "ctaux_create", "ctaux_reset", "ctaux_set_state", "ctaux_sweep",
           "ctaux_propose", "ctaux_rebuild", "ctaux_get_config", "ctaux_get_config_all", "ctaux_get_N", "ctaux_get_N_all", "ctaux_get_N_device", "ctaux_get_stats", "ctaux_get_stats_all",
           "ctaux_get_log", "ctaux_accumulate", "ctaux_get_M", "ctaux_reset_accumulator", "ctaux_g0_workspace_bytes", "ctaux_g0_table", "ctaux_g0_table_noalloc", "ctaux_launch_count", "ctaux_timing_enable", "ctaux_timing_get",
           "ctaux_destroy", "ctaux_strerror", "ctaux_last_cuda_error"]
TEST_EXPORTS = ["ctaux_dgemm", "ctaux_probe_fp64", "ctaux_debug_philox"]

_lib = None


def lib_path() -> str:
    return _build.LIB_PATH


def load_library():
    """Load libctaux_b200.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise CtauxError(-3, "libctaux_b200.so missing", path)
    L = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.ctaux_workspace_bytes.restype = C.c_size_t
    L.ctaux_workspace_bytes.argtypes = [C.POINTER(_Params)]
    L.ctaux_create.argtypes = [C.POINTER(_Params), C.POINTER(vp)]
    L.ctaux_reset.argtypes = [vp, vp]
    L.ctaux_set_state.argtypes = [vp] + [vp] * 8
    L.ctaux_sweep.argtypes = [vp, i32]
    L.ctaux_propose.argtypes = [vp, i32]
    L.ctaux_rebuild.argtypes = [vp]
    L.ctaux_get_config.argtypes = [vp, i32, C.POINTER(i32), vp, vp, vp, vp, i32]
    L.ctaux_get_N.argtypes = [vp, i32, i32, vp, i32]
    L.ctaux_get_config_all.argtypes = [vp, vp, vp, vp, vp, vp]
    L.ctaux_get_N_all.argtypes = [vp, vp]
    L.ctaux_get_N_device.argtypes = [vp, i32, i32, vp, i32]
    L.ctaux_get_stats.argtypes = [vp, i32, C.POINTER(_Stats)]
    L.ctaux_get_stats_all.argtypes = [vp, vp]
    L.ctaux_get_log.restype = i64
    L.ctaux_get_log.argtypes = [vp, i32, vp, i64, i64]
    L.ctaux_accumulate.argtypes = [vp]
    L.ctaux_get_M.argtypes = [vp, vp, vp, vp]
    L.ctaux_reset_accumulator.argtypes = [vp]
    L.ctaux_g0_workspace_bytes.restype = C.c_size_t
    L.ctaux_g0_workspace_bytes.argtypes = [i32, i32, i32, i32]
    L.ctaux_g0_table.argtypes = [vp, i32, i32, C.c_double, C.c_double, C.c_double, i32, i32, vp, i32, vp, vp, C.c_size_t]
    L.ctaux_g0_table_noalloc.argtypes = [vp, i32, i32, C.c_double, C.c_double, C.c_double, i32, i32, vp, i32, vp]
    L.ctaux_launch_count.restype = i64
    L.ctaux_launch_count.argtypes = [vp]
    L.ctaux_timing_enable.argtypes = [vp, i32]
    L.ctaux_timing_get.argtypes = [vp, vp, vp]
    L.ctaux_destroy.restype = None
    L.ctaux_destroy.argtypes = [vp]
    L.ctaux_strerror.restype = C.c_char_p
    L.ctaux_strerror.argtypes = [C.c_int]
    L.ctaux_last_cuda_error.restype = C.c_char_p
    L.ctaux_dgemm.argtypes = [vp, i32, i32, i32, C.c_double, vp, i32, vp, i32, C.c_double, vp, i32, i32]
    L.ctaux_probe_fp64.argtypes = [i32, C.POINTER(C.c_double)]
    L.ctaux_debug_philox.argtypes = [vp, vp, vp, i32]
    _lib = L
    return L


def exported_symbols():
    L = load_library()
    return {name: hasattr(L, name) for name in EXPORTS + TEST_EXPORTS}


def _check(rc, what):
    if rc != 0:
        L = load_library()
        detail = L.ctaux_strerror(rc).decode()
        if rc == -3:
            detail += ": " + L.ctaux_last_cuda_error().decode()
        raise CtauxError(rc, what, detail)


class Walkers:
    """B batched CT-AUX walkers on one GPU (ctaux_create / reset / sweep / get_*)."""

    def __init__(self, Lx, Ly, beta, U, K, g0_table, delay, n_walkers, init_k, max_k,
                 rebuild_every=10, log_capacity=0, cand_window=0, device="cuda:0", stream=None,
                 guard_amp=0.0, fused_small=0, rebuild_mode=0, flip_moves=0, n_tol=0.0, n_omega=0, nfft_oversampling=0,
                 nfft_window=0, pairs=None, graph_mode=0):
        import torch
        if not torch.cuda.is_available():
            raise CtauxError(-3, "ctaux_create", "no CUDA device: this package has no CPU fallback")
        self._torch = torch
        self._L = load_library()
        self.device = torch.device(device)
        table = np.ascontiguousarray(g0_table, dtype=np.float64)
        assert table.shape == (Lx * Ly, table.shape[1])
        self._table = table
        self.n_walkers, self.max_k = n_walkers, max_k
        p = _Params()
        p.Lx, p.Ly, p.beta, p.U, p.K = Lx, Ly, beta, U, K
        p.n_tau = table.shape[1] - 1
        p.g0_table = table.ctypes.data
        p.delay, p.n_walkers, p.init_k, p.max_k = delay, n_walkers, init_k, max_k
        p.rebuild_every, p.log_capacity, p.cand_window = rebuild_every, log_capacity, cand_window
        p.guard_amp = guard_amp
        p.fused_small = fused_small
        p.rebuild_mode = rebuild_mode
        p.flip_moves = flip_moves
        p.n_tol = n_tol
        if pairs is not None:     # (a, b, U): general opposite-spin density-density interaction (ctaux_params.n_pairs)
            pa = np.ascontiguousarray(pairs[0], dtype=np.int32)
            pb = np.ascontiguousarray(pairs[1], dtype=np.int32)
            pu = np.ascontiguousarray(pairs[2], dtype=np.float64)
            assert pa.size == pb.size == pu.size > 0
            self._pairs = (pa, pb, pu)
            p.n_pairs, p.pair_a, p.pair_b, p.pair_U = pa.size, pa.ctypes.data, pb.ctypes.data, pu.ctypes.data
        p.n_omega, p.nfft_oversampling, p.nfft_window = n_omega, nfft_oversampling, nfft_window
        p.graph_mode = graph_mode
        self.n_omega, self.Nc = n_omega, Lx * Ly
        nbytes = self._L.ctaux_workspace_bytes(C.byref(p))
        if nbytes == 0:
            raise CtauxError(-1, "ctaux_workspace_bytes", "invalid parameters")
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p.workspace = self._ws.data_ptr()
        p.workspace_bytes = nbytes
        p.stream = self._stream.cuda_stream
        self.workspace_bytes = nbytes
        self._params = p
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(self._L.ctaux_create(C.byref(p), C.byref(h)), "ctaux_create")
        self._h = h

    @classmethod
    def from_config(cls, cfg, table, n_walkers=None, **kw):
        args = dict(delay=cfg["delay"], n_walkers=n_walkers or cfg["n_walkers"], init_k=cfg["init_k"],
                    max_k=cfg["max_k"], rebuild_every=cfg["rebuild_every"])
        args.update(kw)
        return cls(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, **args)

    def close(self):
        if getattr(self, "_h", None):
            self._L.ctaux_destroy(self._h)
            self._h = None
            self._ws = None

    __del__ = close

    def reset(self, seeds):
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        assert seeds.size == self.n_walkers
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_reset(self._h, seeds.ctypes.data), "ctaux_reset")

    def set_state(self, seeds, configs, next_id, proposals):
        """configs: list (per walker) of dicts with id/site/tau/spin arrays in list order."""
        B, mk = self.n_walkers, self.max_k
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        k = np.array([len(c["site"]) for c in configs], dtype=np.int32)
        ids = np.zeros((B, mk), np.uint64)
        site = np.zeros((B, mk), np.int32)
        tau = np.zeros((B, mk), np.float64)
        spin = np.zeros((B, mk), np.int8)
        for w, c in enumerate(configs):
            ids[w, :k[w]] = c["id"]
            site[w, :k[w]] = c["site"]
            tau[w, :k[w]] = c["tau"]
            spin[w, :k[w]] = c["spin"]
        next_id = np.ascontiguousarray(next_id, dtype=np.uint64)
        proposals = np.ascontiguousarray(proposals, dtype=np.uint64)
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_set_state(self._h, seeds.ctypes.data, k.ctypes.data, ids.ctypes.data,
                                           site.ctypes.data, tau.ctypes.data, spin.ctypes.data,
                                           next_id.ctypes.data, proposals.ctypes.data), "ctaux_set_state")

    def sweep(self, n_sweeps):
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_sweep(self._h, int(n_sweeps)), "ctaux_sweep")

    def propose(self, n_proposals):
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_propose(self._h, int(n_proposals)), "ctaux_propose")

    def rebuild(self):
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_rebuild(self._h), "ctaux_rebuild")

    def get_config(self, w):
        k = C.c_int32(0)
        mk = self.max_k
        ids, site = np.zeros(mk, np.uint64), np.zeros(mk, np.int32)
        tau, spin = np.zeros(mk, np.float64), np.zeros(mk, np.int8)
        _check(self._L.ctaux_get_config(self._h, w, C.byref(k), ids.ctypes.data, site.ctypes.data,
                                        tau.ctypes.data, spin.ctypes.data, mk), "ctaux_get_config")
        n = k.value
        return dict(id=ids[:n].copy(), site=site[:n].copy(), tau=tau[:n].copy(), spin=spin[:n].copy())

    def get_N(self, w, spin):
        """k x k numpy array (row index = first index, Fortran order), list order.  The device-to-host copy
        lands in a pinned staging buffer (full PCIe rate) and is copied out once."""
        st = self.get_stats(w)
        k = st["k"]
        if not k:
            return np.zeros((0, 0), np.float64)
        if getattr(self, "_pin", None) is None:
            self._pin = self._torch.empty(self.max_k * self.max_k, dtype=self._torch.float64, pin_memory=True)
        stage = self._pin[:k * k].numpy()
        _check(self._L.ctaux_get_N(self._h, w, spin, stage.ctypes.data, k), "ctaux_get_N")
        return stage.reshape((k, k), order="F").copy(order="F")

    def get_config_all(self):
        """Configurations of all walkers with one synchronisation: list of dicts (id, site, tau, spin)."""
        B, mk = self.n_walkers, self.max_k
        k = np.zeros(B, np.int32)
        ids, site = np.zeros((B, mk), np.uint64), np.zeros((B, mk), np.int32)
        tau, spin = np.zeros((B, mk), np.float64), np.zeros((B, mk), np.int8)
        _check(self._L.ctaux_get_config_all(self._h, k.ctypes.data, ids.ctypes.data, site.ctypes.data,
                                            tau.ctypes.data, spin.ctypes.data), "ctaux_get_config_all")
        return [dict(id=ids[w, :k[w]].copy(), site=site[w, :k[w]].copy(), tau=tau[w, :k[w]].copy(),
                     spin=spin[w, :k[w]].copy()) for w in range(B)]

    def get_N_all(self, ks):
        """All N_sigma through one pinned buffer and one call: list of (N_up, N_down) views (Fortran order) into
        a pinned staging tensor that the next get_N_all overwrites."""
        B, mk = self.n_walkers, self.max_k
        if getattr(self, "_pin_all", None) is None:
            self._pin_all = self._torch.empty(B * 2 * mk * mk, dtype=self._torch.float64, pin_memory=True)
        flat = self._pin_all.numpy()
        _check(self._L.ctaux_get_N_all(self._h, flat.ctypes.data), "ctaux_get_N_all")
        out = []
        for w in range(B):
            k = int(ks[w])
            out.append(tuple(flat[(2 * w + s) * mk * mk:(2 * w + s) * mk * mk + k * k].reshape((k, k), order="F")
                             for s in range(2)))
        return out

    # ---- the C ABI's own batched forms: packed [B][max_k] arrays in pinned host memory, no per-walker Python
    def get_state_packed(self, with_N=True):
        """ctaux_get_config_all + ctaux_get_stats_all (+ ctaux_get_N_all) into pinned host buffers owned by this object
        (overwritten by the next call): dict(k [B], id/site/tau/spin [B][max_k], stats: structured array of
        ctaux_stats [B], N: flat buffer in ctaux_get_N_all's layout or None)."""
        t, B, mk = self._torch, self.n_walkers, self.max_k
        if getattr(self, "_pk", None) is None:
            pin = lambda n, dt: t.empty(n, dtype=dt, pin_memory=True).numpy()
            self._pk = dict(k=pin(B, t.int32), id=pin(B * mk, t.int64).view(np.uint64).reshape(B, mk),
                            site=pin(B * mk, t.int32).reshape(B, mk), tau=pin(B * mk, t.float64).reshape(B, mk),
                            spin=pin(B * mk, t.int8).reshape(B, mk))
            self._pk_stats = (_Stats * B)()
        pk = self._pk
        with t.cuda.device(self.device):
            _check(self._L.ctaux_get_config_all(self._h, pk["k"].ctypes.data, pk["id"].ctypes.data, pk["site"].ctypes.data,
                                                pk["tau"].ctypes.data, pk["spin"].ctypes.data), "ctaux_get_config_all")
            _check(self._L.ctaux_get_stats_all(self._h, C.addressof(self._pk_stats)), "ctaux_get_stats_all")
            N = None
            if with_N:
                if getattr(self, "_pin_all", None) is None:
                    self._pin_all = t.empty(B * 2 * mk * mk, dtype=t.float64, pin_memory=True)
                N = self._pin_all.numpy()
                _check(self._L.ctaux_get_N_all(self._h, N.ctypes.data), "ctaux_get_N_all")
        return dict(pk, stats=np.ctypeslib.as_array(self._pk_stats), N=N)

    def set_state_packed(self, seeds, st):
        """ctaux_set_state from packed host arrays (the dict get_state_packed returns: the chain continues from
        st["stats"]["next_id"] / ["proposals"])."""
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        next_id = np.ascontiguousarray(st["stats"]["next_id"], dtype=np.uint64)
        prop = np.ascontiguousarray(st["stats"]["proposals"], dtype=np.uint64)
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_set_state(self._h, seeds.ctypes.data, st["k"].ctypes.data, st["id"].ctypes.data,
                                           st["site"].ctypes.data, st["tau"].ctypes.data, st["spin"].ctypes.data,
                                           next_id.ctypes.data, prop.ctypes.data), "ctaux_set_state")

    def get_N_device(self, w, spin):
        torch = self._torch
        k = self.get_stats(w)["k"]
        out = torch.empty((k, k), dtype=torch.float64, device=self.device)  # holds N^T in C order
        if k:
            _check(self._L.ctaux_get_N_device(self._h, w, spin, out.data_ptr(), k), "ctaux_get_N_device")
        return out.t()

    def get_stats(self, w):
        s = _Stats()
        _check(self._L.ctaux_get_stats(self._h, w, C.byref(s)), "ctaux_get_stats")
        return {f: getattr(s, f) for f, _ in _Stats._fields_}

    def accumulate(self):
        """S6: add sign * M of every walker's current configuration to the tau-grid accumulators (delayed NFFT)."""
        with self._torch.cuda.device(self.device):
            _check(self._L.ctaux_accumulate(self._h), "ctaux_accumulate")

    def get_M(self):
        """(M_sum complex [2][Nc][n_omega], sign_sum, n_meas): the one transform at the end of the run."""
        out = np.zeros((2, self.Nc, self.n_omega, 2), np.float64)
        ss, nm = C.c_double(0.0), C.c_int64(0)
        _check(self._L.ctaux_get_M(self._h, out.ctypes.data, C.addressof(ss), C.addressof(nm)), "ctaux_get_M")
        return out[..., 0] + 1j * out[..., 1], ss.value, nm.value

    def reset_accumulator(self):
        _check(self._L.ctaux_reset_accumulator(self._h), "ctaux_reset_accumulator")

    def get_stats_all(self):
        arr = (_Stats * self.n_walkers)()
        _check(self._L.ctaux_get_stats_all(self._h, C.addressof(arr)), "ctaux_get_stats_all")
        names = [f for f, _ in _Stats._fields_]
        return [{f: getattr(s, f) for f in names} for s in arr]

    def get_log(self, w, first=0, count=None):
        if count is None:
            count = self._params.log_capacity
        out = np.zeros(max(count, 0), LOG_DTYPE)
        n = self._L.ctaux_get_log(self._h, w, out.ctypes.data, first, count) if count > 0 else 0
        if n < 0:
            _check(int(n), "ctaux_get_log")
        return out[:n]

    def launch_count(self):
        return self._L.ctaux_launch_count(self._h)

    def timing_enable(self, on=True):
        _check(self._L.ctaux_timing_enable(self._h, 1 if on else 0), "ctaux_timing_enable")

    def timing_get(self):
        ms = np.zeros(8, np.float64)
        nl = np.zeros(8, np.int64)
        _check(self._L.ctaux_timing_get(self._h, ms.ctypes.data, nl.ctypes.data), "ctaux_timing_get")
        return {name: dict(ms=float(ms[i]), launches=int(nl[i])) for i, name in enumerate(STEP_CLASSES)}


class WalkerGroups:
    """B walkers split over G contexts, each on its own CUDA stream and driven by its own host thread
    (ctaux_sweep blocks, ctypes releases the GIL).  Walkers are independent chains,
    so the grouping changes nothing in any chain; it lets the serial S3 proposal kernel of one group
    (a few SMs busy) overlap the S2/S4 GEMMs of the others.  BASELINE.json config 5: "2 walkers on
    separate streams".  Walker w of the job lives in group w // (B/G) at local index w % (B/G)."""

    def __init__(self, n_groups, n_walkers, make):
        """make(group_index, walkers_in_group, stream) -> Walkers"""
        import torch
        assert n_walkers % n_groups == 0
        self.n_groups, self.n_walkers, self.per = n_groups, n_walkers, n_walkers // n_groups
        self.streams = [torch.cuda.Stream() for _ in range(n_groups)]
        self.groups = [make(g, self.per, self.streams[g]) for g in range(n_groups)]

    def _each(self, fn):
        import threading
        errs = []

        def run(W, g):
            try:
                fn(W, g)
            except BaseException as e:  # re-raised on the caller's thread
                errs.append(e)

        th = [threading.Thread(target=run, args=(W, g)) for g, W in enumerate(self.groups)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        if errs:
            raise errs[0]

    def reset(self, seeds):
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        self._each(lambda W, g: W.reset(seeds[g * self.per:(g + 1) * self.per]))

    def set_state(self, seeds, configs, next_id, proposals):
        P = self.per
        self._each(lambda W, g: W.set_state(seeds[g * P:(g + 1) * P], configs[g * P:(g + 1) * P],
                                            next_id[g * P:(g + 1) * P], proposals[g * P:(g + 1) * P]))

    def sweep(self, n_sweeps):
        self._each(lambda W, g: W.sweep(n_sweeps))

    def propose(self, n_proposals):
        self._each(lambda W, g: W.propose(n_proposals))

    def rebuild(self):
        self._each(lambda W, g: W.rebuild())

    def _loc(self, w):
        return self.groups[w // self.per], w % self.per

    def get_config(self, w):
        W, i = self._loc(w)
        return W.get_config(i)

    def get_N(self, w, spin):
        W, i = self._loc(w)
        return W.get_N(i, spin)

    def get_stats(self, w):
        W, i = self._loc(w)
        return W.get_stats(i)

    def get_log(self, w, first=0, count=None):
        W, i = self._loc(w)
        return W.get_log(i, first, count)

    def launch_count(self):
        return sum(W.launch_count() for W in self.groups)

    def fetch_all(self, with_N=True):
        """(configs, stats, N) of every walker in job order, the groups read out concurrently (one host thread
        and one pinned staging buffer per group).  N[w] = (N_up, N_down) or None."""
        cfgs = [None] * self.n_walkers
        stats = [None] * self.n_walkers
        Ns = [None] * self.n_walkers

        def one(W, g):
            lo = g * self.per
            cfgs[lo:lo + self.per] = W.get_config_all()
            stats[lo:lo + self.per] = W.get_stats_all()
            if with_N:
                Ns[lo:lo + self.per] = W.get_N_all([len(c["site"]) for c in cfgs[lo:lo + self.per]])

        self._each(one)
        return cfgs, stats, Ns

    def get_state_packed(self, with_N=True):
        """Per stream group, concurrently: list of the dicts Walkers.get_state_packed returns."""
        out = [None] * len(self.groups)

        def one(W, g):
            out[g] = W.get_state_packed(with_N)

        self._each(one)
        return out

    def set_state_packed(self, seeds, states):
        seeds = np.ascontiguousarray(seeds, dtype=np.uint64)
        self._each(lambda W, g: W.set_state_packed(seeds[g * self.per:(g + 1) * self.per], states[g]))

    def timing_enable(self, on=True):
        for W in self.groups:
            W.timing_enable(on)

    def timing_get(self):
        out = None
        for W in self.groups:
            t = W.timing_get()
            if out is None:
                out = t
            else:
                for k in out:
                    out[k]["ms"] += t[k]["ms"]
                    out[k]["launches"] += t[k]["launches"]
        return out

    def synchronize(self):
        for s in self.streams:
            s.synchronize()

    def close(self):
        for W in self.groups:
            W.close()


def g0_table_from_sigma(Lx, Ly, t, mu, beta, n_omega, n_quad, n_tau, sigma_c=None, device="cuda:0"):
    """The DCA bare cluster propagator G0c(r, tau) as the [Nc][n_tau + 1] table ctaux_create consumes (ctaux_g0_table:
    coarse graining, cluster exclusion and the Fourier transforms run on the device).  sigma_c: complex [Nc][n_omega] or None."""
    import torch
    if not torch.cuda.is_available():
        raise CtauxError(-3, "ctaux_g0_table", "no CUDA device: this package has no CPU fallback")
    L = load_library()
    nbytes = L.ctaux_g0_workspace_bytes(Lx, Ly, n_omega, n_tau)
    if nbytes == 0:
        raise CtauxError(-1, "ctaux_g0_workspace_bytes", "invalid parameters")
    dev = torch.device(device)
    sig_ptr = None
    if sigma_c is not None:
        sc = np.asarray(sigma_c, dtype=np.complex128)
        assert sc.shape == (Lx * Ly, n_omega)
        sig = np.ascontiguousarray(np.stack([sc.real, sc.imag], axis=-1))
        sig_ptr = sig.ctypes.data
    table = np.zeros((Lx * Ly, n_tau + 1), np.float64)
    with torch.cuda.device(dev):
        ws = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        _check(L.ctaux_g0_table(torch.cuda.current_stream(dev).cuda_stream, Lx, Ly, t, mu, beta, n_omega, n_quad, sig_ptr,
                                n_tau, table.ctypes.data, ws.data_ptr(), nbytes), "ctaux_g0_table")
    return table


G0_NOALLOC_MAX_BYTES = 8 << 20      # CTAUX_G0_NOALLOC_MAX_BYTES of include/ctaux.h


def g0_table_from_sigma_noalloc(Lx, Ly, t, mu, beta, n_omega, n_quad, n_tau, sigma_c=None, device="cuda:0"):
    """g0_table_from_sigma through ctaux_g0_table_noalloc: no device memory is allocated by the call (the scratch is a
    static 8 MiB device array inside the library, shared by all calls on a device: do not overlap calls).  Sizes whose
    scratch exceeds the array raise CtauxError(-2)."""
    import torch
    if not torch.cuda.is_available():
        raise CtauxError(-3, "ctaux_g0_table_noalloc", "no CUDA device: this package has no CPU fallback")
    L = load_library()
    dev = torch.device(device)
    sig_ptr = None
    if sigma_c is not None:
        sc = np.asarray(sigma_c, dtype=np.complex128)
        assert sc.shape == (Lx * Ly, n_omega)
        sig = np.ascontiguousarray(np.stack([sc.real, sc.imag], axis=-1))
        sig_ptr = sig.ctypes.data
    table = np.zeros((Lx * Ly, n_tau + 1), np.float64)
    with torch.cuda.device(dev):
        rc = L.ctaux_g0_table_noalloc(torch.cuda.current_stream(dev).cuda_stream, Lx, Ly, t, mu, beta, n_omega, n_quad,
                                      sig_ptr, n_tau, table.ctypes.data)
    if rc == -2:      # the library's message states the bytes needed and the size of the static array
        raise CtauxError(rc, "ctaux_g0_table_noalloc", L.ctaux_last_cuda_error().decode())
    _check(rc, "ctaux_g0_table_noalloc")
    return table


def colmajor(rows, cols, device="cuda", fill=None, generator=None):
    """A rows x cols float64 CUDA tensor stored column-major with a leading dimension that is a multiple of 8
    (the layout ctaux_dgemm wants): element (i, j) at data_ptr + 8*(i + j*ld)."""
    import torch
    ld = max(8, (rows + 7) // 8 * 8)
    if fill is None:
        store = torch.zeros((cols, ld), dtype=torch.float64, device=device)
    else:
        store = fill(cols, ld).to(device)
    return store[:, :rows].t()


def ctaux_dgemm(A, B, C_out=None, alpha=1.0, beta=0.0, stream=None, b_nmajor=0):
    """C = beta*C + alpha*A@B through the library's TMA-staged DMMA tile kernel.  A (M x K), B (K x N), C (M x N)
    are torch float64 CUDA tensors stored column-major (stride(0) == 1) with leading dimensions that are multiples
    of 8 (see colmajor()).  b_nmajor = 1 exercises the tile's "N-major" right-operand layout (B^T is handed over)."""
    import torch
    L = load_library()
    M, K = A.shape
    K2, N = B.shape
    assert K == K2 and A.dtype == torch.float64 and B.dtype == torch.float64
    if C_out is None:
        C_out = colmajor(M, N, A.device)
    for t in (A, B, C_out):
        assert t.shape[0] <= 1 or t.stride(0) == 1, "column-major operands required"
    ld = lambda t: int(t.stride(1)) if t.shape[1] > 1 else max(8, (t.shape[0] + 7) // 8 * 8)
    s = stream if stream is not None else torch.cuda.current_stream(A.device)
    if b_nmajor:        # the tile's "N-major" right operand: hand over B^T stored column-major (N x K)
        Bt = colmajor(N, K, A.device)
        Bt.copy_(B.t())
        B = Bt
    _check(L.ctaux_dgemm(s.cuda_stream, M, N, K, alpha, A.data_ptr(), ld(A), B.data_ptr(), ld(B), beta,
                         C_out.data_ptr(), ld(C_out), 1 if b_nmajor else 0), "ctaux_dgemm")
    return C_out


def probe_fp64(which=0):
    """Issue-rate peak of the FP64 tensor (0: DMMA.8x8x4) or vector (1: DFMA) pipe, TFLOP/s."""
    L = load_library()
    v = C.c_double(0.0)
    _check(L.ctaux_probe_fp64(which, C.byref(v)), "ctaux_probe_fp64")
    return v.value


def debug_philox(ctr, key):
    L = load_library()
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    _check(L.ctaux_debug_philox(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, ctr.shape[0]), "ctaux_debug_philox")
    return out
