"""ctypes wrapper around oracle/direct_sum.c and oracle/bltc_cpu.c (argument marshalling only).

TEST INFRASTRUCTURE, NOT THE PRODUCT -- see oracle/__init__.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "direct_sum.c"), os.path.join(_HERE, "coulomb_sum.c"), os.path.join(_HERE, "bltc_cpu.c")]
_LIB = os.path.join(_HERE, "liboracle.so")
# strict IEEE: no fast-math, no FMA contraction, baseline x86-64 (no -march=native)
_CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", "-Wall"]
# The same sources as a compiler would build them for speed (the "fair" CPU number).  Used ONLY by
# bench.py's cpu_baseline_fast key -- never for parity: fast-math changes the arithmetic.
_LIB_FAST = os.path.join(_HERE, "liboracle_fast.so")
_CFLAGS_FAST = ["-O3", "-march=native", "-ffast-math", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall"]

_lib = None
_lib_fast = None
_dp = C.POINTER(C.c_double)
_ip64 = C.POINTER(C.c_int64)
_ip32 = C.POINTER(C.c_int32)


def build(force: bool = False, fast: bool = False) -> str:
    """Compile the oracle with gcc if the .so is missing or older than its sources.  fast=True: the
    -O3 -march=native -ffast-math build (timing only; -march=native: build it on the machine that runs it)."""
    target, flags = (_LIB_FAST, _CFLAGS_FAST) if fast else (_LIB, _CFLAGS)
    stale = force or not os.path.exists(target) or any(
        os.path.getmtime(s) > os.path.getmtime(target) for s in _SRC)
    if stale:
        cmd = ["gcc", *flags, "-o", target, *_SRC, "-lm"]
        subprocess.run(cmd, check=True, stdout=sys.stderr, stderr=sys.stderr)
    return target


def _load(fast: bool = False):
    global _lib, _lib_fast
    if fast and _lib_fast is not None:
        return _lib_fast
    if not fast and _lib is not None:
        return _lib
    lib = C.CDLL(build(force=fast, fast=fast))      # the fast build is always rebuilt for this host's CPU
    lib.oracle_max_threads.restype = C.c_int
    lib.oracle_last_phase_seconds.argtypes = [_dp]
    lib.oracle_kernel.restype = C.c_double
    lib.oracle_kernel.argtypes = [C.c_int, C.c_double] + [C.c_double] * 6 + [C.POINTER(C.c_int)]
    lib.oracle_direct.restype = C.c_int
    lib.oracle_direct.argtypes = [C.c_int, C.c_int64, _dp, _dp, _dp, _dp,
                                  C.c_int64, _dp, _dp, _dp, _dp, _dp,
                                  C.c_double, C.c_int, C.c_int, _dp]
    lib.oracle_plan_create.restype = C.c_void_p
    lib.oracle_plan_create.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_int64, _dp, _dp, _dp,
                                       C.c_double, C.c_int, C.c_int, C.c_int]
    lib.oracle_plan_destroy.argtypes = [C.c_void_p]
    lib.oracle_plan_set_upward.argtypes = [C.c_void_p, C.c_int]
    lib.oracle_plan_sizes.argtypes = [C.c_void_p, _ip64]
    lib.oracle_plan_export.argtypes = [C.c_void_p, _ip64, _ip64, _ip64, _ip64, _dp, _dp, _ip32, _ip32,
                                       _ip64, _ip64, _ip64, _ip32, _ip64, _ip32]
    lib.oracle_plan_proxy.restype = C.c_int
    lib.oracle_plan_proxy.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp]
    lib.oracle_bltc_eval.restype = C.c_int
    lib.oracle_bltc_eval.argtypes = [C.c_void_p, C.c_int, _dp, _dp, _dp, C.c_double, C.c_int, C.c_int,
                                     C.c_int64, _ip64, _dp, _dp]
    lib.oracle_coulomb_direct.restype = C.c_int
    lib.oracle_coulomb_direct.argtypes = [C.c_int64, _dp, _dp, _dp, _dp, C.c_int64, _dp, _dp, _dp, _dp, _dp,
                                          C.c_double, C.c_int, _dp]
    lib.oracle_bltc_eval_coulomb.restype = C.c_int
    lib.oracle_bltc_eval_coulomb.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_double, C.c_int,
                                             C.c_int64, _ip64, _dp, _dp]
    if fast:
        _lib_fast = lib
    else:
        _lib = lib
    return lib


def n_threads() -> int:
    """Threads the oracle's OpenMP loops use: omp_get_max_threads() of the loaded library."""
    return int(_load().oracle_max_threads())


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def kernel_value(kind, k, t, s):
    lib = _load()
    skip = C.c_int(0)
    v = lib.oracle_kernel(kind, float(k), *[float(v) for v in t], *[float(v) for v in s], C.byref(skip))
    return v, bool(skip.value)


def direct(targets, sources, w, f_src, k, *, f_tgt=None, subtract=True, finalize=True, kind=0):
    """Direct sum (oracle/direct_sum.c).  targets/sources: (x, y, z) tuples or [3][n] arrays.
    f_src: [N] or [n_orb][N]; k scalar or [n_orb].  Returns [M] or [n_orb][M]."""
    lib = _load()
    tx, ptx = _d(targets[0]); ty, pty = _d(targets[1]); tz, ptz = _d(targets[2])
    sx, psx = _d(sources[0]); sy, psy = _d(sources[1]); sz, psz = _d(sources[2])
    w_, pw = _d(w)
    f_src = np.asarray(f_src, dtype=np.float64)
    single = f_src.ndim == 1
    F = np.atleast_2d(f_src)
    K = np.broadcast_to(np.atleast_1d(np.asarray(k, dtype=np.float64)), (F.shape[0],))
    FT = None
    if subtract:
        if f_tgt is None:
            raise ValueError("subtract=True needs f_tgt (f at the targets)")
        FT = np.atleast_2d(np.asarray(f_tgt, dtype=np.float64))
    M, N = tx.shape[0], sx.shape[0]
    out = np.empty((F.shape[0], M))
    for o in range(F.shape[0]):
        fo, pfo = _d(F[o])
        if subtract:
            fto, pfto = _d(FT[o])
        else:
            pfto = None
        oo = np.empty(M)
        rc = lib.oracle_direct(kind, M, ptx, pty, ptz, pfto, N, psx, psy, psz, pw, pfo,
                               float(K[o]), int(subtract), int(finalize), oo.ctypes.data_as(_dp))
        if rc != 0:
            raise ValueError("oracle_direct: bad arguments")
        out[o] = oo
    return out[0] if single else out


def coulomb_direct(targets, sources, w, f_src, *, f_tgt=None, subtract=True, alpha=1.0):
    """Hartree-potential direct sum with Gaussian singularity subtraction (oracle/coulomb_sum.c,
    PAPER.md:197-224 Eq. (19),(23),(24)).  f_src: [N] or [n_f][N].  Returns [M] or [n_f][M]."""
    lib = _load()
    tx, ptx = _d(targets[0]); ty, pty = _d(targets[1]); tz, ptz = _d(targets[2])
    sx, psx = _d(sources[0]); sy, psy = _d(sources[1]); sz, psz = _d(sources[2])
    w_, pw = _d(w)
    f_src = np.asarray(f_src, dtype=np.float64)
    single = f_src.ndim == 1
    F = np.atleast_2d(f_src)
    FT = None
    if subtract:
        if f_tgt is None:
            raise ValueError("subtract=True needs f_tgt (f at the targets)")
        FT = np.atleast_2d(np.asarray(f_tgt, dtype=np.float64))
    M, N = tx.shape[0], sx.shape[0]
    out = np.empty((F.shape[0], M))
    for o in range(F.shape[0]):
        fo, pfo = _d(F[o])
        pfto = None
        if subtract:
            fto, pfto = _d(FT[o])
        oo = np.empty(M)
        rc = lib.oracle_coulomb_direct(M, ptx, pty, ptz, pfto, N, psx, psy, psz, pw, pfo,
                                       float(alpha), int(subtract), oo.ctypes.data_as(_dp))
        if rc != 0:
            raise ValueError("oracle_coulomb_direct: bad arguments")
        out[o] = oo
    return out[0] if single else out


class OraclePlan:
    """Tree + batches + interaction lists of oracle/bltc_cpu.c (Algorithm 3 line 1 and the
    decisions of line 3), and the evaluation (lines 2-3)."""

    def __init__(self, sources, theta, degree, leaf_size, batch_size, targets=None, fast=False,
                 upward_from_children=False):
        """upward_from_children: proxy charges of internal clusters from their children's proxy charges (reading R23,
        SURVEY.md 8(f) NEXT-4) instead of from their own particles (reading R9, the default)."""
        lib = _load(fast)
        self._lib = lib
        self._s = [_d(a) for a in sources]
        self.N = self._s[0][0].shape[0]
        if targets is None:
            self._t = None
            self.M = self.N
            targs = (0, None, None, None)
        else:
            self._t = [_d(a) for a in targets]
            self.M = self._t[0][0].shape[0]
            targs = (self.M, self._t[0][1], self._t[1][1], self._t[2][1])
        self.degree = int(degree)
        self.P = (self.degree + 1) ** 3
        self._h = lib.oracle_plan_create(self.N, self._s[0][1], self._s[1][1], self._s[2][1], *targs,
                                         float(theta), int(degree), int(leaf_size), int(batch_size))
        if not self._h:
            raise ValueError("oracle_plan_create: bad arguments")
        self.upward_from_children = bool(upward_from_children)
        lib.oracle_plan_set_upward(self._h, int(self.upward_from_children))
        s = (C.c_int64 * 8)()
        lib.oracle_plan_sizes(self._h, s)
        (self.n_clusters, self.n_leaves, self.n_batches, self.n_far, self.n_near,
         self.far_evals, self.near_evals, self.shared_batches) = [int(v) for v in s]

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            self._lib.oracle_plan_destroy(h)
            self._h = None

    def export(self):
        nc, nb = self.n_clusters, self.n_batches
        o = dict(
            src_perm=np.empty(self.N, np.int64), tgt_perm=np.empty(self.M, np.int64),
            cl_begin=np.empty(nc, np.int64), cl_end=np.empty(nc, np.int64),
            cl_lo=np.empty((nc, 3)), cl_hi=np.empty((nc, 3)),
            cl_parent=np.empty(nc, np.int32), cl_nchild=np.empty(nc, np.int32),
            b_begin=np.empty(nb, np.int64), b_end=np.empty(nb, np.int64),
            far_ptr=np.empty(nb + 1, np.int64), far_idx=np.empty(self.n_far, np.int32),
            near_ptr=np.empty(nb + 1, np.int64), near_idx=np.empty(self.n_near, np.int32))
        p64 = lambda a: a.ctypes.data_as(_ip64)
        p32 = lambda a: a.ctypes.data_as(_ip32)
        pd = lambda a: a.ctypes.data_as(_dp)
        self._lib.oracle_plan_export(
            self._h, p64(o["src_perm"]), p64(o["tgt_perm"]), p64(o["cl_begin"]), p64(o["cl_end"]),
            pd(o["cl_lo"]), pd(o["cl_hi"]), p32(o["cl_parent"]), p32(o["cl_nchild"]),
            p64(o["b_begin"]), p64(o["b_end"]), p64(o["far_ptr"]), p32(o["far_idx"]),
            p64(o["near_ptr"]), p32(o["near_idx"]))
        return o

    def proxy(self, c, q):
        """(qhat[P], nodes[3][n+1]) of cluster c for caller-order charges q (Eq. (35) right)."""
        q_, pq = _d(q)
        qhat = np.empty(self.P)
        nodes = np.empty((3, self.degree + 1))
        rc = self._lib.oracle_plan_proxy(self._h, int(c), pq, qhat.ctypes.data_as(_dp),
                                         nodes.ctypes.data_as(_dp))
        if rc != 0:
            raise ValueError("bad cluster index")
        return qhat, nodes

    def last_phase_seconds(self):
        """(proxy-charge seconds, batch-sum seconds) of the most recent library call (one field)."""
        t = np.zeros(2)
        self._lib.oracle_last_phase_seconds(t.ctypes.data_as(_dp))
        return float(t[0]), float(t[1])

    def _evaluate(self, call, w, f_src, f_tgt, subtract, batches, return_parts):
        """Shared marshalling of evaluate / evaluate_coulomb: one library call per field, call(o, pw, pfo, pft,
        nsel, psel, pout, pparts) -> rc."""
        w_, pw = _d(w)
        f_src = np.asarray(f_src, dtype=np.float64)
        single = f_src.ndim == 1
        F = np.atleast_2d(f_src)
        FT = None
        if subtract:
            if f_tgt is None:
                if self._t is not None:
                    raise ValueError("subtract with separate targets needs f_tgt")
                FT = F
            else:
                FT = np.atleast_2d(np.asarray(f_tgt, dtype=np.float64))
        if batches is not None:
            sel = np.ascontiguousarray(batches, dtype=np.int64)
            nsel, psel = sel.shape[0], sel.ctypes.data_as(_ip64)
        else:
            nsel, psel = 0, None
        out = np.full((F.shape[0], self.M), np.nan)
        parts = np.full((F.shape[0], 2, self.M), np.nan) if return_parts else None
        for o in range(F.shape[0]):
            fo, pfo = _d(F[o])
            pft = None
            if subtract:
                fto, pft = _d(FT[o])
            oo = np.full(self.M, np.nan)
            pp = np.full((2, self.M), np.nan) if return_parts else None
            rc = call(o, pw, pfo, pft, nsel, psel, oo.ctypes.data_as(_dp),
                      pp.ctypes.data_as(_dp) if return_parts else None)
            if rc != 0:
                raise ValueError("oracle BLTC evaluation: bad arguments")
            out[o] = oo
            if return_parts:
                parts[o] = pp
            ph = self.last_phase_seconds()
            self.phase_seconds = [self.phase_seconds[0] + ph[0], self.phase_seconds[1] + ph[1]] if o else list(ph)
        res = out[0] if single else out
        if return_parts:
            return res, (parts[0] if single else parts)
        return res

    def evaluate(self, w, f_src, k, *, f_tgt=None, subtract=True, finalize=True, kind=0,
                 batches=None, return_parts=False):
        """f_src [N] or [n_orb][N]; returns out [M] or [n_orb][M] in caller order (NaN for
        targets of batches that were not selected)."""
        n_f = np.atleast_2d(np.asarray(f_src)).shape[0]
        K = np.broadcast_to(np.atleast_1d(np.asarray(k, dtype=np.float64)), (n_f,))
        call = lambda o, pw, pfo, pft, nsel, psel, pout, pparts: self._lib.oracle_bltc_eval(
            self._h, kind, pw, pfo, pft, float(K[o]), int(subtract), int(finalize), nsel, psel, pout, pparts)
        return self._evaluate(call, w, f_src, f_tgt, subtract, batches, return_parts)

    def evaluate_coulomb(self, w, f_src, *, f_tgt=None, subtract=True, alpha=1.0, batches=None,
                         return_parts=False):
        """Hartree potential through the treecode (oracle_bltc_eval_coulomb, reading R21)."""
        call = lambda o, pw, pfo, pft, nsel, psel, pout, pparts: self._lib.oracle_bltc_eval_coulomb(
            self._h, pw, pfo, pft, float(alpha), int(subtract), nsel, psel, pout, pparts)
        return self._evaluate(call, w, f_src, f_tgt, subtract, batches, return_parts)
