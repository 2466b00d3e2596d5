#!/usr/bin/env python
"""Accuracy / speed sweep of the GPU treecode on BASELINE.json configs[4] (seeded uniform-random points in the unit
cube, w ~ U(0,1)/N, f ~ U(-1,1); the single-GPU analogue of PAPER.md:464-472 Fig. 10 and PAPER.md:494-500 Fig. 11):

  python -m paper_2003_01833_b200.sweep [--quick] [--kernel yukawa|coulomb] > sweep.md

For every (N, k, theta, degree) it prints one markdown row: time per convolution (CUDA events, median of 3 after a
warm-up), equivalent interactions/s = N^2 / t, the kernel evaluations the plan performs, and the relative 2-norm error
of bltc_convolve against direct_convolve on 1e4 seeded sampled targets (both on the GPU; the direct sum itself is
pinned to the CPU oracle by tests/).  Subtraction is off: the points are not a quadrature.  Needs a CUDA device.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


def run(N, k, theta, degree, kernel, torch, B, I, n_sample=10000):
    c = I.config4(N=N, k=k, theta=theta, degree=degree)
    X = torch.from_numpy(c.coords()).cuda()
    w = torch.from_numpy(c.w).cuda()
    f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
    plan = B.bltc_create(None, X, w, N, theta, degree, c.batch_size, c.leaf_size)
    st = B.bltc_get_stats(plan)
    out = torch.empty((1, N), dtype=torch.float64, device="cuda")

    def conv():
        if kernel == "coulomb":
            B.bltc_convolve_coulomb(plan, f, 1, out, False, 1.0)
        else:
            B.bltc_convolve(plan, c.k, f, 1, out, False)

    conv()
    torch.cuda.synchronize()
    ts = []
    for _ in range(3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); conv(); b.record(); b.synchronize()
        ts.append(a.elapsed_time(b))
    ms = float(np.median(ts))
    idx = torch.from_numpy(I.sample_targets(N, n_sample, seed=3)).cuda()
    T = X[:, idx].contiguous()
    ds = torch.empty((1, idx.numel()), dtype=torch.float64, device="cuda")
    if kernel == "coulomb":
        B.direct_convolve_coulomb(T, None, idx.numel(), X, w, f, N, 1, ds, False, 1.0)
    else:
        B.direct_convolve(T, None, idx.numel(), X, w, f, N, c.k, 1, ds, False)
    torch.cuda.synchronize()
    err = float(torch.linalg.norm(out[0, idx] - ds[0]) / torch.linalg.norm(ds[0]))
    B.bltc_destroy(plan)
    return dict(N=N, k=k, theta=theta, degree=degree, ms=ms, rate=float(N) ** 2 / (ms * 1e-3),
                far=st["far_evals"], near=st["near_evals"], build_ms=st["build_ms"], err=err)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="N = 1e6 at k = 1 only")
    ap.add_argument("--kernel", default="yukawa", choices=["yukawa", "coulomb"])
    args = ap.parse_args()
    import torch
    from . import binding as B
    from . import inputs as I
    if not torch.cuda.is_available():
        sys.exit("sweep: no CUDA device -- the product has no CPU fallback")
    B.lib()
    cases = [(1_000_000, k, th, n) for k in ((1.0,) if args.quick else (0.5, 1.0, 5.0))
             for th in (0.5, 0.7, 0.9) for n in (4, 6, 8, 10)]
    if not args.quick:
        cases += [(2_000_000, 1.0, 0.7, 8), (8_000_000, 1.0, 0.7, 8), (8_000_000, 1.0, 0.7, 7)]
    print(f"| N | k | theta | degree | ms / convolution | equiv. interactions/s | far evals | near evals | "
          f"N^2 / evals | host plan build ms | BLTC vs direct (rel. 2-norm, 1e4 targets) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for N, k, th, n in cases:
        r = run(N, k, th, n, args.kernel, torch, B, I)
        print(f"| {N} | {k} | {th} | {n} | {r['ms']:.1f} | {r['rate']:.3e} | {r['far']:.3e} | {r['near']:.3e} | "
              f"{float(N) ** 2 / (r['far'] + r['near']):.2f} | {r['build_ms']:.0f} | {r['err']:.2e} |", flush=True)


if __name__ == "__main__":
    main()
