"""Thin ctypes binding of libbltc (include/bltc.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; nothing is computed here.
Arguments may be torch tensors (CUDA or CPU, float64, contiguous) or numpy float64 arrays; the
library itself decides host vs device from the raw pointer.  There is no CPU fallback: if
libbltc.so cannot be built/loaded, importing the entry points raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

BLTC_OK, BLTC_EINVAL, BLTC_ENOMEM, BLTC_ECUDA, BLTC_ENODEVICE = 0, -1, -2, -3, -4
PHASES = ("gather", "upward", "far", "near", "epilogue")

_dp = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)


class BltcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libbltc error {code}: {msg}")
        self.code = code


class bltc_stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "n_points", "n_clusters", "n_leaves", "n_batches", "n_far", "n_near", "far_evals", "near_evals",
        "n_proxy_clusters", "upward_pairs", "n_far_items", "n_near_items", "partial_len",
        "n_upward_items", "n_upward_reduce", "launches_per_group")] + [
        ("shared_batches", C.c_int32), ("interp_degree", C.c_int32),
        ("theta", C.c_double), ("build_ms", C.c_double), ("upload_ms", C.c_double),
        ("shard_rank", C.c_int32), ("shard_world", C.c_int32)] + [(n, C.c_int64) for n in (
            "shard_batch_begin", "shard_batch_end", "shard_targets", "shard_far_evals", "shard_near_evals")] + [
        ("tree_ms", C.c_double), ("lists_ms", C.c_double), ("decomp_ms", C.c_double), ("create_ms", C.c_double),
        ("built_on_device", C.c_int32), ("upward_from_children", C.c_int32)]


MAX_ORBITAL_TILE = 7          # BLTC_MAX_ORBITAL_TILE of include/bltc.h

EXPORTED = ("bltc_create", "bltc_create_host_plan", "bltc_create_sharded", "bltc_create_host_plan_sharded",
            "bltc_create_with_builder",
            "bltc_get_shard_targets", "bltc_convolve", "direct_convolve", "bltc_convolve_scatter",
            "bltc_convolve_coulomb_scatter",
            "bltc_convolve_coulomb", "direct_convolve_coulomb", "bltc_gi_update", "bltc_gi_update_noalloc", "bltc_destroy",
            "bltc_get_stats", "bltc_export_plan", "bltc_export_proxy", "bltc_set_profiling",
            "bltc_get_phase_ms", "bltc_direct_set_profiling", "bltc_direct_get_kernel_ms",
            "bltc_probe_fp64", "bltc_probe_fp64_form", "bltc_orbital_tiles", "bltc_last_error", "bltc_version")

_lib = None


def lib():
    """Load (building if stale) paper_2003_01833_b200/libbltc.so.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp = C.c_void_p
    L.bltc_last_error.restype = C.c_char_p
    L.bltc_version.restype = C.c_char_p
    L.bltc_create.argtypes = [C.POINTER(vp), vp, vp, vp, C.c_int64, C.c_double, C.c_int, C.c_int, C.c_int]
    L.bltc_create_host_plan.argtypes = L.bltc_create.argtypes
    L.bltc_create_sharded.argtypes = L.bltc_create.argtypes + [C.c_int, C.c_int]
    L.bltc_create_host_plan_sharded.argtypes = L.bltc_create_sharded.argtypes
    L.bltc_create_with_builder.argtypes = L.bltc_create_sharded.argtypes + [C.c_int]
    L.bltc_get_shard_targets.argtypes = [vp, _i64p]
    L.bltc_convolve.argtypes = [vp, _dp, vp, C.c_int, vp, C.c_int, vp]
    L.direct_convolve.argtypes = [vp, vp, C.c_int64, vp, vp, vp, C.c_int64, _dp, C.c_int, vp, C.c_int, vp]
    L.bltc_convolve_coulomb.argtypes = [vp, vp, C.c_int, vp, C.c_int, C.c_double, vp]
    L.bltc_convolve_scatter.argtypes = [vp, _dp, vp, C.c_int, vp, C.POINTER(vp), C.c_int, C.c_int, vp]
    L.bltc_convolve_coulomb_scatter.argtypes = [vp, vp, C.c_int, vp, C.POINTER(vp), C.c_int, C.c_int, C.c_double, vp]
    L.direct_convolve_coulomb.argtypes = [vp, vp, C.c_int64, vp, vp, vp, C.c_int64, C.c_int, vp, C.c_int,
                                          C.c_double, vp]
    L.bltc_gi_update.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int64, C.c_double, vp, vp]
    L.bltc_gi_update_noalloc.argtypes = L.bltc_gi_update.argtypes
    L.bltc_destroy.argtypes = [vp]
    L.bltc_get_stats.argtypes = [vp, C.POINTER(bltc_stats)]
    L.bltc_export_plan.argtypes = [vp, _i64p, _i64p, _i64p, _i64p, _dp, _dp, _i32p, _i32p, _i64p, _i64p,
                                   _i64p, _i32p, _i64p, _i32p]
    L.bltc_export_proxy.argtypes = [vp, _i32p, _dp, _dp, _dp, _i32p]
    L.bltc_set_profiling.argtypes = [vp, C.c_int]
    L.bltc_get_phase_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.bltc_direct_set_profiling.argtypes = [C.c_int]
    L.bltc_direct_get_kernel_ms.argtypes = [C.POINTER(C.c_float)]
    L.bltc_probe_fp64.argtypes = [C.c_int, _dp, vp]
    L.bltc_probe_fp64_form.argtypes = [C.c_int, C.c_int, _dp, vp]
    L.bltc_orbital_tiles.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int]
    for name in EXPORTED:
        f = getattr(L, name)
        if name not in ("bltc_last_error", "bltc_version"):
            f.restype = C.c_int
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise BltcError(rc, lib().bltc_last_error().decode())


def _ptr(a, what, allow_none=False, count=None):
    """Raw address of a float64 contiguous torch tensor / numpy array (keeps no reference).  count: the number of
    doubles the library will read or write there -- a smaller buffer is a ValueError here, not an out-of-bounds
    access inside a kernel."""
    if a is None:
        if allow_none:
            return None
        raise ValueError(f"{what} must not be None")
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"]:
            raise ValueError(f"{what}: need a C-contiguous float64 array")
        if count is not None and a.size < count:
            raise ValueError(f"{what}: need at least {count} elements, got {a.size}")
        return a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor):
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise ValueError(f"{what}: need a contiguous float64 tensor")
        if count is not None and a.numel() < count:
            raise ValueError(f"{what}: need at least {count} elements, got {a.numel()}")
        return a.data_ptr()
    raise TypeError(f"{what}: expected numpy array or torch tensor")


def _stream_ptr(stream):
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return torch.cuda.current_stream().cuda_stream
        return None
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _karray(k, n_orb):
    k = np.ascontiguousarray(np.atleast_1d(np.asarray(k, dtype=np.float64)))
    if k.shape != (n_orb,):
        raise ValueError(f"k must have shape ({n_orb},)")
    return k


class Plan:
    """Handle returned by bltc_create / bltc_create_host_plan."""

    def __init__(self, handle, N):
        self._h = handle
        self.N = N

    def destroy(self):
        if self._h:
            lib().bltc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _create(fn, targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size, *shard):
    h = C.c_void_p()
    _check(fn(C.byref(h), _ptr(targets, "targets", True, 3 * int(N)), _ptr(sources, "sources", False, 3 * int(N)),
              _ptr(weights, "weights", True, int(N)), int(N), float(theta), int(interp_degree),
              int(batch_size), int(leaf_size), *[int(v) for v in shard]))
    return Plan(h, int(N))


def bltc_create_sharded(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size, rank, world):
    """include/bltc.h bltc_create_sharded: rank's slice of the target batches (multi-GPU, no collective)."""
    return _create(lib().bltc_create_sharded, targets, sources, weights, N, theta, interp_degree, batch_size,
                   leaf_size, rank, world)


def bltc_create_host_plan_sharded(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size,
                                  rank, world):
    return _create(lib().bltc_create_host_plan_sharded, targets, sources, weights, N, theta, interp_degree,
                   batch_size, leaf_size, rank, world)


def bltc_get_shard_targets(plan):
    """Caller indices of the targets a (sharded) plan computes, in target tree order."""
    n = bltc_get_stats(plan)["shard_targets"]
    idx = np.empty(n, dtype=np.int64)
    _check(lib().bltc_get_shard_targets(plan._h, idx.ctypes.data_as(_i64p)))
    return idx


def bltc_create(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size):
    """include/bltc.h bltc_create.  targets may be None (targets are the sources)."""
    return _create(lib().bltc_create, targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size)


BUILDER_DEVICE, BUILDER_HOST, UPWARD_FROM_CHILDREN, UPWARD_FROM_PARTICLES = 0, 1, 2, 4


def bltc_create_with_builder(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size,
                             rank=0, world=1, builder=BUILDER_DEVICE):
    """include/bltc.h bltc_create_with_builder: tree and lists by kernels (BUILDER_DEVICE, what bltc_create uses)
    or by the threaded host code (BUILDER_HOST); both give the same plan.  OR UPWARD_FROM_PARTICLES into `builder` for the
    literal upward pass of Alg. 3 line 2 (every cluster from its own particles) instead of the default child -> parent
    pass (UPWARD_FROM_CHILDREN: same proxy charges up to rounding, O(N P) work)."""
    return _create(lib().bltc_create_with_builder, targets, sources, weights, N, theta, interp_degree, batch_size,
                   leaf_size, rank, world, builder)


def bltc_create_host_plan(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size):
    return _create(lib().bltc_create_host_plan, targets, sources, weights, N, theta, interp_degree,
                   batch_size, leaf_size)


def bltc_convolve(plan, k, f, n_orb, out, subtract_singularity=True, stream=None):
    """include/bltc.h bltc_convolve.  f, out: [n_orb][N] device or host buffers."""
    kk = _karray(k, n_orb)
    n = int(n_orb) * plan.N
    _check(lib().bltc_convolve(plan._h, kk.ctypes.data_as(_dp), _ptr(f, "f", False, n), int(n_orb), _ptr(out, "out", False, n),
                               int(bool(subtract_singularity)), _stream_ptr(stream)))
    return out


def _peer_array(peers, n):
    """HOST array of device pointers for the scatter calls: peers are tensors (checked for size) or raw addresses."""
    arr = (C.c_void_p * max(len(peers), 1))()
    for i, p in enumerate(peers):
        arr[i] = int(p) if isinstance(p, int) else _ptr(p, f"peer_outs[{i}]", False, n)
    return arr


def bltc_convolve_scatter(plan, k, f, n_orb, out, peer_outs, subtract_singularity=True, stream=None):
    """include/bltc.h bltc_convolve_scatter: the epilogue also stores into every buffer of peer_outs (tensors or raw
    device addresses, e.g. the other ranks' symmetric-memory buffers)."""
    kk = _karray(k, n_orb)
    n = int(n_orb) * plan.N
    arr = _peer_array(peer_outs, n)
    _check(lib().bltc_convolve_scatter(plan._h, kk.ctypes.data_as(_dp), _ptr(f, "f", False, n), int(n_orb),
                                       _ptr(out, "out", False, n), arr, len(peer_outs), int(bool(subtract_singularity)),
                                       _stream_ptr(stream)))
    return out


def bltc_convolve_coulomb_scatter(plan, f, n_f, out, peer_outs, subtract_singularity=True, alpha=1.0, stream=None):
    n = int(n_f) * plan.N
    arr = _peer_array(peer_outs, n)
    _check(lib().bltc_convolve_coulomb_scatter(plan._h, _ptr(f, "f", False, n), int(n_f), _ptr(out, "out", False, n), arr,
                                               len(peer_outs), int(bool(subtract_singularity)), float(alpha),
                                               _stream_ptr(stream)))
    return out


def direct_convolve(targets, f_targets, M, sources, weights, f_sources, N, k, n_orb, out,
                    subtract_singularity=True, stream=None):
    """include/bltc.h direct_convolve."""
    kk = _karray(k, n_orb)
    M, N, n_orb = int(M), int(N), int(n_orb)
    _check(lib().direct_convolve(_ptr(targets, "targets", False, 3 * M), _ptr(f_targets, "f_targets", True, n_orb * M), M,
                                 _ptr(sources, "sources", False, 3 * N), _ptr(weights, "weights", False, N),
                                 _ptr(f_sources, "f_sources", False, n_orb * N), N, kk.ctypes.data_as(_dp), n_orb,
                                 _ptr(out, "out", False, n_orb * M), int(bool(subtract_singularity)), _stream_ptr(stream)))
    return out


def bltc_convolve_coulomb(plan, f, n_f, out, subtract_singularity=True, alpha=1.0, stream=None):
    """include/bltc.h bltc_convolve_coulomb (Hartree potential, Gaussian singularity subtraction)."""
    n = int(n_f) * plan.N
    _check(lib().bltc_convolve_coulomb(plan._h, _ptr(f, "f", False, n), int(n_f), _ptr(out, "out", False, n),
                                       int(bool(subtract_singularity)), float(alpha), _stream_ptr(stream)))
    return out


def direct_convolve_coulomb(targets, f_targets, M, sources, weights, f_sources, N, n_f, out,
                            subtract_singularity=True, alpha=1.0, stream=None):
    """include/bltc.h direct_convolve_coulomb."""
    M, N, n_f = int(M), int(N), int(n_f)
    _check(lib().direct_convolve_coulomb(_ptr(targets, "targets", False, 3 * M), _ptr(f_targets, "f_targets", True, n_f * M), M,
                                         _ptr(sources, "sources", False, 3 * N), _ptr(weights, "weights", False, N),
                                         _ptr(f_sources, "f_sources", False, n_f * N), N, n_f, _ptr(out, "out", False, n_f * M),
                                         int(bool(subtract_singularity)), float(alpha), _stream_ptr(stream)))
    return out


def bltc_gi_update(w, psi_old, f_old, psi_new, phi, n_prev, N, eps_old, result, stream=None):
    """include/bltc.h bltc_gi_update (Green Iteration, Alg. 2 lines 4-7).  psi_new is updated in place;
    result: float64[4 + n_prev] buffer (device or host) = eps_new, delta, norm, residual, coefficients."""
    N, n_prev = int(N), int(n_prev)
    _check(lib().bltc_gi_update(_ptr(w, "w", False, N), _ptr(psi_old, "psi_old", False, N), _ptr(f_old, "f_old", False, N),
                                _ptr(psi_new, "psi_new", False, N), _ptr(phi, "phi", True, n_prev * N), n_prev, N,
                                float(eps_old), _ptr(result, "result", False, 4 + n_prev), _stream_ptr(stream)))
    return result


GI_NOALLOC_MAX_PREV = 64      # BLTC_GI_NOALLOC_MAX_PREV of include/bltc.h


def bltc_gi_update_noalloc(w, psi_old, f_old, psi_new, phi, n_prev, N, eps_old, result, stream=None):
    """include/bltc.h bltc_gi_update_noalloc: bltc_gi_update for callers that cannot allocate device memory (an
    application whose own arena already owns all of HBM, a host that forbids driver allocations in its callbacks, a
    fixed memory budget, a loop that cannot afford an allocation's synchronisation).  The reduction scratch is a
    1.06 MiB array inside libbltc.so instead of pool memory, so: every buffer must be a CUDA tensor,
    n_prev <= GI_NOALLOC_MAX_PREV (64), and two calls that may overlap on one GPU race on that array -- keep them on
    one stream.  The first call on a device looks up the array's address; make it before any stream capture.
    This wrapper allocates nothing either: it passes the addresses of the caller's tensors."""
    N, n_prev = int(N), int(n_prev)
    _check(lib().bltc_gi_update_noalloc(
        _ptr(w, "w", False, N), _ptr(psi_old, "psi_old", False, N), _ptr(f_old, "f_old", False, N),
        _ptr(psi_new, "psi_new", False, N), _ptr(phi, "phi", True, n_prev * N), n_prev, N,
        float(eps_old), _ptr(result, "result", False, 4 + n_prev), _stream_ptr(stream)))
    return result


def bltc_destroy(plan):
    plan.destroy()


def bltc_get_stats(plan):
    s = bltc_stats()
    _check(lib().bltc_get_stats(plan._h, C.byref(s)))
    return {n: getattr(s, n) for n, _ in bltc_stats._fields_}


def bltc_export_plan(plan):
    st = bltc_get_stats(plan)
    nc, nb, N = st["n_clusters"], st["n_batches"], st["n_points"]
    o = dict(
        src_perm=np.empty(N, np.int64), tgt_perm=np.empty(N, np.int64),
        cl_begin=np.empty(nc, np.int64), cl_end=np.empty(nc, np.int64),
        cl_lo=np.empty((nc, 3)), cl_hi=np.empty((nc, 3)),
        cl_parent=np.empty(nc, np.int32), cl_nchild=np.empty(nc, np.int32),
        b_begin=np.empty(nb, np.int64), b_end=np.empty(nb, np.int64),
        far_ptr=np.empty(nb + 1, np.int64), far_idx=np.empty(st["n_far"], np.int32),
        near_ptr=np.empty(nb + 1, np.int64), near_idx=np.empty(st["n_near"], np.int32))
    p64 = lambda a: a.ctypes.data_as(_i64p)
    p32 = lambda a: a.ctypes.data_as(_i32p)
    pd = lambda a: a.ctypes.data_as(_dp)
    _check(lib().bltc_export_plan(
        plan._h, p64(o["src_perm"]), p64(o["tgt_perm"]), p64(o["cl_begin"]), p64(o["cl_end"]),
        pd(o["cl_lo"]), pd(o["cl_hi"]), p32(o["cl_parent"]), p32(o["cl_nchild"]),
        p64(o["b_begin"]), p64(o["b_end"]), p64(o["far_ptr"]), p32(o["far_idx"]),
        p64(o["near_ptr"]), p32(o["near_idx"])))
    return o


def bltc_export_proxy(plan):
    st = bltc_get_stats(plan)
    ns, n1 = st["n_proxy_clusters"], st["interp_degree"] + 1
    P = n1 ** 3
    cl = np.empty(ns, np.int32); nodes = np.empty((ns, 3, n1)); what = np.empty((ns, P))
    fhat = np.zeros((ns, P, MAX_ORBITAL_TILE)); ot = C.c_int32(0)      # sized for the widest tile (include/bltc.h)
    _check(lib().bltc_export_proxy(plan._h, cl.ctypes.data_as(_i32p), nodes.ctypes.data_as(_dp),
                                   what.ctypes.data_as(_dp), fhat.ctypes.data_as(_dp), C.byref(ot)))
    o = ot.value
    fh = fhat.reshape(-1)[: ns * P * o].reshape(ns, P, o) if o else np.zeros((ns, P, 0))
    return dict(cluster=cl, nodes=nodes, what=what, fhat=fh)


def bltc_set_profiling(plan, enable=True):
    _check(lib().bltc_set_profiling(plan._h, int(bool(enable))))


def bltc_get_phase_ms(plan):
    ms = (C.c_float * len(PHASES))()
    _check(lib().bltc_get_phase_ms(plan._h, ms))
    return dict(zip(PHASES, [float(v) for v in ms]))


def bltc_direct_set_profiling(enable=True):
    _check(lib().bltc_direct_set_profiling(int(bool(enable))))


def bltc_direct_get_kernel_ms():
    ms = C.c_float(0)
    _check(lib().bltc_direct_get_kernel_ms(C.byref(ms)))
    return float(ms.value)


def bltc_probe_fp64(iters=64, stream=None, form=0):
    """DFMA-only probe in TFLOP/s; form 1 = three distinct vector-register sources per DFMA (include/bltc.h)."""
    t = C.c_double(0)
    _check(lib().bltc_probe_fp64_form(int(form), int(iters), C.byref(t), _stream_ptr(stream)))
    return float(t.value)


def bltc_orbital_tiles(n_orb):
    """Widths of the register tiles a call with n_orb orbitals is cut into (include/bltc.h)."""
    n = lib().bltc_orbital_tiles(int(n_orb), None, 0)
    if n < 0:
        _check(n)
    w = (C.c_int * n)()
    _check(min(0, lib().bltc_orbital_tiles(int(n_orb), w, n)))
    return [int(v) for v in w]


def bltc_version():
    return lib().bltc_version().decode()
