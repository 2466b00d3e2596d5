"""bltc_gi_update_noalloc (include/bltc.h): the Green-Iteration update for callers that cannot allocate device memory.

Some users of the library call it from a place where cudaMalloc is not available to them: their application gave all
of HBM to its own arena at start-up, or their host forbids driver allocations inside its callbacks, or they run under
a device-memory budget that is fixed once they are initialised, or they sit in a loop that cannot afford the
synchronisation an allocation may bring.  bltc_gi_update takes its reduction scratch from a memory pool on every call;
the _noalloc variant keeps that scratch in a fixed 1.06 MiB array inside libbltc.so and makes no allocating call.

What is checked here, on a GPU:
  * its output against bltc_gi_update's on the same device buffers, within the tolerances of
    tests/test_gpu_gi_update.py (1e-12 relative on the scalars, 1e-11 on residual and coefficients, 1e-13 relative
    2-norm on psi), on TWO CALLS IN A ROW that share the array: a large call that fills many slots of it, then at once
    a smaller call with another n_prev (another slot layout) that must not see what the first one left behind, then the
    large one again;
  * that sizes beyond the array (n_prev > 64) and host buffers are refused with a message that says why.
On a CPU (no device needed: the size check comes before any CUDA call): the limit and its message.

The file name sorts last on purpose: the driver runs the GPU suite with -x, so a failure here hides no other test.
It passes alone in a fresh process (its first call does the per-device set-up) and after the other tests.
"""
import math

import numpy as np
import pytest

from paper_2003_01833_b200 import binding as B


def _fields(N, n_prev, seed):
    # seeded inputs shaped like the real ones (see tests/test_gpu_gi_update.py): uneven positive weights, a w-orthonormal
    # set phi, a normalised psi_old and a psi_new with a component along every phi_j
    rng = np.random.default_rng(20030183 + 9000 + seed)
    w = rng.random(N) ** 3 + 1e-6
    raw = rng.standard_normal((n_prev + 2, N))
    basis = []
    for v in raw:
        for b in basis:
            v = v - (w * v * b).sum() * b
        basis.append(v / math.sqrt((w * v * v).sum()))
    phi = np.ascontiguousarray(np.stack(basis[:n_prev])) if n_prev else None
    psi_old = basis[n_prev]
    psi_new = 0.9 * psi_old + 0.3 * basis[n_prev + 1] + (rng.standard_normal(n_prev) @ phi if n_prev else 0.0)
    f_old = -psi_old / (0.1 + rng.random(N))
    return w, psi_old, f_old, np.ascontiguousarray(psi_new), phi


def test_noalloc_limit_is_the_headers_and_is_enforced_without_a_device():
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "bltc.h")).read()
    assert int(re.search(r"#define\s+BLTC_GI_NOALLOC_MAX_PREV\s+(\d+)", hdr).group(1)) == B.GI_NOALLOC_MAX_PREV
    n_prev = B.GI_NOALLOC_MAX_PREV + 1
    a = np.ones(8)
    with pytest.raises(B.BltcError) as ei:
        B.bltc_gi_update_noalloc(a, a, a, a.copy(), np.ones((n_prev, 8)), n_prev, 8, -0.5, np.empty(4 + n_prev))
    assert ei.value.code == B.BLTC_EINVAL
    assert "BLTC_GI_NOALLOC_MAX_PREV = 64" in str(ei.value) and str(n_prev) in str(ei.value)


@pytest.mark.gpu
def test_noalloc_matches_gi_update_on_calls_in_a_row_sharing_the_scratch_array():
    import torch
    assert torch.cuda.is_available()
    B.lib()
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # (N, n_prev): many blocks and a wide slot layout; then few blocks and a narrow one; n_prev = 0; the limit itself
    cases = [(300007, 20), (4133, 3), (300007, 20), (50001, 0), (20011, B.GI_NOALLOC_MAX_PREV)]
    dev = []
    for n, (N, n_prev) in enumerate(cases):
        w, po, f, pn, phi = _fields(N, n_prev, seed=n)
        dev.append((N, n_prev, d(w), d(po), d(f), d(pn), d(phi) if n_prev else None))
    # the existing path first, on copies of psi_new (both entry points update it in place)
    want = []
    for N, n_prev, w, po, f, pn, phi in dev:
        psi = pn.clone()
        res = torch.empty(4 + n_prev, dtype=torch.float64, device="cuda")
        B.bltc_gi_update(w, po, f, psi, phi, n_prev, N, -0.8, res)
        want.append((res, psi))
    torch.cuda.synchronize()
    # outputs are allocated up front, so that between the calls below nothing but the library's kernels runs
    got = [(torch.empty(4 + n_prev, dtype=torch.float64, device="cuda"), pn.clone()) for _, n_prev, *_, pn, _ in dev]
    torch.cuda.synchronize()
    for (N, n_prev, w, po, f, _, phi), (res, psi) in zip(dev, got):      # back to back on one stream, no sync between
        B.bltc_gi_update_noalloc(w, po, f, psi, phi, n_prev, N, -0.8, res)
    torch.cuda.synchronize()
    for (N, n_prev, *_), (res, psi), (res0, psi0) in zip(dev, got, want):
        r, r0 = res.cpu().numpy(), res0.cpu().numpy()
        assert np.all(np.isfinite(r))
        assert r[0] == pytest.approx(r0[0], rel=1e-12)                   # eps_new
        assert r[1] == pytest.approx(r0[1], rel=1e-12)                   # delta
        assert r[2] == pytest.approx(r0[2], rel=1e-12)                   # norm
        assert r[3] == pytest.approx(r0[3], rel=1e-11)                   # residual
        if n_prev:
            np.testing.assert_allclose(r[4:], r0[4:], rtol=1e-11, atol=1e-13)
        p, p0 = psi.cpu().numpy(), psi0.cpu().numpy()
        assert np.linalg.norm(p - p0) / np.linalg.norm(p0) <= 1e-13, (N, n_prev)


@pytest.mark.gpu
def test_noalloc_refuses_what_it_cannot_hold_and_then_still_works():
    import torch
    assert torch.cuda.is_available()
    N = 1000
    w, po, f, pn, _ = _fields(N, 0, seed=77)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dw, dpo, df = d(w), d(po), d(f)
    n_big = B.GI_NOALLOC_MAX_PREV + 1
    with pytest.raises(B.BltcError) as ei:                                # more phi_j than the fixed array has slots for
        B.bltc_gi_update_noalloc(dw, dpo, df, d(pn), torch.zeros((n_big, N), dtype=torch.float64, device="cuda"), n_big, N,
                                 -0.5, torch.empty(4 + n_big, dtype=torch.float64, device="cuda"))
    assert ei.value.code == B.BLTC_EINVAL and "BLTC_GI_NOALLOC_MAX_PREV" in str(ei.value)
    with pytest.raises(B.BltcError) as ei:                                # a host buffer would have to be staged = allocated
        B.bltc_gi_update_noalloc(dw, dpo, df, d(pn), None, 0, N, -0.5, np.empty(4))
    assert ei.value.code == B.BLTC_EINVAL and "device memory" in str(ei.value)
    with pytest.raises(B.BltcError):
        B.bltc_gi_update_noalloc(w, dpo, df, d(pn), None, 0, N, -0.5, torch.empty(4, dtype=torch.float64, device="cuda"))
    # a refused call leaves the entry point usable
    res, res0 = (torch.empty(4, dtype=torch.float64, device="cuda") for _ in range(2))
    psi, psi0 = d(pn), d(pn)
    B.bltc_gi_update_noalloc(dw, dpo, df, psi, None, 0, N, -0.5, res)
    B.bltc_gi_update(dw, dpo, df, psi0, None, 0, N, -0.5, res0)
    torch.cuda.synchronize()
    np.testing.assert_allclose(res.cpu().numpy(), res0.cpu().numpy(), rtol=1e-12)
    assert np.linalg.norm((psi - psi0).cpu().numpy()) / np.linalg.norm(psi0.cpu().numpy()) <= 1e-13
