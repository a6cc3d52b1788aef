"""ctypes front end of the CPU oracle (oracle/ctaux_oracle.cpp).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ctaux_oracle.cpp")
_LIB = os.path.join(_HERE, "libctaux_oracle.so")

LOG_DTYPE = np.dtype([("p", "<u8"), ("type", "<i4"), ("arg", "<i4"), ("tau", "<f8"),
                      ("spin", "<i4"), ("accepted", "<i4"), ("R", "<f8"), ("u", "<f8")])

T0, T1 = 0, 1


def build(force: bool = False) -> str:
    """g++ -O3 the oracle into oracle/libctaux_oracle.so (plain C++, no BLAS)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-march=x86-64-v3", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", _LIB]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i32, i64, u64, f64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_double
        L.orc_create.restype = vp
        L.orc_create.argtypes = [i32, i32, f64, f64, f64, i32, vp, u64, i32]
        L.orc_destroy.argtypes = [vp]
        L.orc_reset.argtypes = [vp, i32]
        L.orc_set_mode.argtypes = [vp, i32]
        L.orc_set_flips.argtypes = [vp, i32]
        L.orc_set_pairs.argtypes = [vp, i32, vp, vp, vp]
        L.orc_pair_exp_gamma.argtypes = [vp, i32]
        L.orc_pair_exp_gamma.restype = f64
        L.orc_acc_flip.restype = i64
        L.orc_acc_flip.argtypes = [vp]
        L.orc_set_state.argtypes = [vp, i32, vp, vp, vp, vp, u64, u64]
        L.orc_sweep.argtypes = [vp, i32]
        L.orc_propose.argtypes = [vp, i64]
        for name, rt in [("orc_k", i32), ("orc_sign", i32), ("orc_p", u64), ("orc_next_id", u64),
                         ("orc_acc_ins", i64), ("orc_acc_rem", i64), ("orc_min_margin", f64),
                         ("orc_exp_gamma", f64), ("orc_log_size", i64)]:
            getattr(L, name).restype = rt
            getattr(L, name).argtypes = [vp]
        L.orc_get_config.argtypes = [vp, vp, vp, vp, vp]
        L.orc_get_A.argtypes = [vp, i32, vp]
        L.orc_build_A.argtypes = [vp, i32, i32, vp, vp, vp, vp]
        L.orc_get_N.argtypes = [vp, i32, vp]
        L.orc_get_N.restype = i32
        L.orc_get_N_incremental.argtypes = [vp, i32, vp]
        L.orc_get_N_incremental.restype = i32
        L.orc_logdet.argtypes = [vp, i32, vp]
        L.orc_logdet.restype = f64
        L.orc_g.argtypes = [vp, i32, f64]
        L.orc_g.restype = f64
        L.orc_get_log.argtypes = [vp, vp, i64, i64]
        L.orc_clear_log.argtypes = [vp]
        L.orc_log_entry_bytes.restype = i32
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_unif53.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_unif53.restype = f64
        assert L.orc_log_entry_bytes() == LOG_DTYPE.itemsize
        _lib = L
    return _lib


def philox(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def unif53(a: int, b: int) -> float:
    return lib().orc_unif53(a, b)


class OracleWalker:
    """One Markov chain.  mode=T0 brute force (the definition), mode=T1 rank-1 updates."""

    def __init__(self, Lx, Ly, beta, U, K, table, seed, mode=T0):
        table = np.ascontiguousarray(table, dtype=np.float64)
        Nc = Lx * Ly
        assert table.shape[0] == Nc
        self.M = table.shape[1] - 1
        self.Nc = Nc
        self._h = lib().orc_create(Lx, Ly, beta, U, K, self.M, table.ctypes.data, int(seed), mode)

    @classmethod
    def from_config(cls, cfg, table, seed, mode=T0):
        return cls(cfg["Lx"], cfg["Ly"], cfg["beta"], cfg["U"], cfg["K"], table, seed, mode)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def reset(self, init_k):
        lib().orc_reset(self._h, init_k)

    def set_mode(self, mode):
        lib().orc_set_mode(self._h, mode)

    def set_flips(self, on=True):
        """Enable the auxiliary-spin flip as a third move.  Default: off."""
        lib().orc_set_flips(self._h, 1 if on else 0)

    def set_pairs(self, a, b, U):
        """NEXT-4: general opposite-spin density-density interaction, pairs p = (a_p up, b_p down, U_p); the `site` of a
        vertex (configurations, logs) is then the pair index.  Call before reset / set_state."""
        a = np.ascontiguousarray(a, dtype=np.int32)
        b = np.ascontiguousarray(b, dtype=np.int32)
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert a.size == b.size == U.size
        lib().orc_set_pairs(self._h, a.size, a.ctypes.data, b.ctypes.data, U.ctypes.data)

    def pair_exp_gamma(self, p):
        return lib().orc_pair_exp_gamma(self._h, int(p))

    acc_flip = property(lambda s: lib().orc_acc_flip(s._h))

    def set_state(self, site, tau, spin, ids=None, next_id=None, p=0):
        site = np.ascontiguousarray(site, dtype=np.int32)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        spin = np.ascontiguousarray(spin, dtype=np.int8)
        k = site.size
        if ids is None:
            ids = np.arange(k, dtype=np.uint64)
        ids = np.ascontiguousarray(ids, dtype=np.uint64)
        if next_id is None:
            next_id = int(ids.max()) + 1 if k else 0
        lib().orc_set_state(self._h, k, ids.ctypes.data, site.ctypes.data, tau.ctypes.data,
                            spin.ctypes.data, int(next_id), int(p))

    def sweep(self, n=1):
        lib().orc_sweep(self._h, n)

    def propose(self, n=1):
        lib().orc_propose(self._h, n)

    k = property(lambda s: lib().orc_k(s._h))
    sign = property(lambda s: lib().orc_sign(s._h))
    p = property(lambda s: lib().orc_p(s._h))
    next_id = property(lambda s: lib().orc_next_id(s._h))
    acc_ins = property(lambda s: lib().orc_acc_ins(s._h))
    acc_rem = property(lambda s: lib().orc_acc_rem(s._h))
    min_margin = property(lambda s: lib().orc_min_margin(s._h))
    exp_gamma = property(lambda s: lib().orc_exp_gamma(s._h))

    def config(self):
        k = self.k
        ids = np.zeros(k, np.uint64)
        site = np.zeros(k, np.int32)
        tau = np.zeros(k, np.float64)
        spin = np.zeros(k, np.int8)
        lib().orc_get_config(self._h, ids.ctypes.data, site.ctypes.data, tau.ctypes.data, spin.ctypes.data)
        return dict(id=ids, site=site, tau=tau, spin=spin)

    def A(self, sidx):
        k = self.k
        out = np.zeros((k, k), np.float64)
        lib().orc_get_A(self._h, sidx, out.ctypes.data)
        return out

    def A_of(self, sidx, site, tau, spin):
        """A_sigma of a given vertex list (the walker's own configuration is not touched)."""
        site = np.ascontiguousarray(site, dtype=np.int32)
        tau = np.ascontiguousarray(tau, dtype=np.float64)
        spin = np.ascontiguousarray(spin, dtype=np.int8)
        k = site.size
        out = np.zeros((k, k), np.float64)
        lib().orc_build_A(self._h, sidx, k, site.ctypes.data, tau.ctypes.data, spin.ctypes.data, out.ctypes.data)
        return out

    def N(self, sidx):
        k = self.k
        out = np.zeros((k, k), np.float64)
        rc = lib().orc_get_N(self._h, sidx, out.ctypes.data)
        if rc != 0:
            raise ArithmeticError("singular A")
        return out

    def N_incremental(self, sidx):
        k = self.k
        out = np.zeros((k, k), np.float64)
        rc = lib().orc_get_N_incremental(self._h, sidx, out.ctypes.data)
        if rc != 0:
            raise RuntimeError("no incremental N (mode T0 or nothing proposed yet)")
        return out

    def logdet(self, sidx):
        sg = C.c_int(0)
        la = lib().orc_logdet(self._h, sidx, C.byref(sg))
        return la, sg.value

    def g(self, d, dtau):
        return lib().orc_g(self._h, int(d), float(dtau))

    def log(self):
        n = lib().orc_log_size(self._h)
        out = np.zeros(n, LOG_DTYPE)
        if n:
            lib().orc_get_log(self._h, out.ctypes.data, 0, n)
        return out

    def clear_log(self):
        lib().orc_clear_log(self._h)


def run_walkers(cfg, table, seeds, n_sweeps, mode=T1, init_k=None, threads=None):
    """Run one chain per seed (reset + n_sweeps sweeps), one Python thread per host core
    (ctypes releases the GIL).  Returns the list of OracleWalker objects."""
    init_k = cfg["init_k"] if init_k is None else init_k
    threads = threads or os.cpu_count() or 1

    def one(seed):
        w = OracleWalker.from_config(cfg, table, seed, mode)
        w.reset(init_k)
        w.sweep(n_sweeps)
        return w

    with ThreadPoolExecutor(max_workers=threads) as ex:
        return list(ex.map(one, [int(s) for s in seeds]))


if __name__ == "__main__":
    print(build(force=True))
