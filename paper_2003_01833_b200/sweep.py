#!/usr/bin/env python
"""Accuracy / speed sweep of the GPU treecode on BASELINE.json configs[4] (seeded uniform-random points in the unit
cube, w ~ U(0,1)/N, f ~ U(-1,1); the single-GPU analogue of PAPER.md:464-472 Fig. 10 and PAPER.md:494-500 Fig. 11):

  python -m paper_2003_01833_b200.sweep [--quick] [--kernel yukawa|coulomb] > sweep.md

For every (N, theta, degree, k) -- N in {1e6, 2e6, 8e6}, theta in {0.5, 0.7, 0.9}, degree 4..10, k in {0.5, 1, 5} -- it
prints one markdown row: time per convolution (CUDA events, median of 3 (2 at N = 8e6) after a warm-up), equivalent
interactions/s = N^2 / t, the kernel evaluations the plan performs, and the relative 2-norm error
of bltc_convolve against direct_convolve on 1e4 seeded sampled targets (both on the GPU; the direct sum itself is
pinned to the CPU oracle by tests/).  Subtraction is off: the points are not a quadrature.  Needs a CUDA device.
"""
from __future__ import annotations

import argparse
import sys

import numpy as np


class Cloud:
    """configs[4] input of one N, resident on the device; the direct sums on the sampled targets are cached per k."""

    def __init__(self, N, torch, B, I, n_sample=10000):
        c = I.config4(N=N)
        self.N, self.c = N, c
        self.X = torch.from_numpy(c.coords()).cuda()
        self.w = torch.from_numpy(c.w).cuda()
        self.f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
        self.idx = torch.from_numpy(I.sample_targets(N, n_sample, seed=3)).cuda()
        self.T = self.X[:, self.idx].contiguous()
        self.out = torch.empty((1, N), dtype=torch.float64, device="cuda")
        self._ds = {}
        self.torch, self.B = torch, B

    def direct(self, kernel, k):
        key = (kernel, k)
        if key not in self._ds:
            torch, B = self.torch, self.B
            ds = torch.empty((1, self.idx.numel()), dtype=torch.float64, device="cuda")
            if kernel == "coulomb":
                B.direct_convolve_coulomb(self.T, None, self.idx.numel(), self.X, self.w, self.f, self.N, 1, ds, False, 1.0)
            else:
                B.direct_convolve(self.T, None, self.idx.numel(), self.X, self.w, self.f, self.N, [k], 1, ds, False)
            torch.cuda.synchronize()
            self._ds[key] = ds
        return self._ds[key]


def run(cloud, plan, st, k, kernel, repeats):
    torch, B = cloud.torch, cloud.B
    out = cloud.out

    def conv():
        if kernel == "coulomb":
            B.bltc_convolve_coulomb(plan, cloud.f, 1, out, False, 1.0)
        else:
            B.bltc_convolve(plan, [k], cloud.f, 1, out, False)

    conv()
    torch.cuda.synchronize()
    ts = []
    for _ in range(repeats):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); conv(); b.record(); b.synchronize()
        ts.append(a.elapsed_time(b))
    ms = float(np.median(ts))
    ds = cloud.direct(kernel, k)
    err = float(torch.linalg.norm(out[0, cloud.idx] - ds[0]) / torch.linalg.norm(ds[0]))
    N = cloud.N
    return dict(ms=ms, rate=float(N) ** 2 / (ms * 1e-3), far=st["far_evals"], near=st["near_evals"],
                create_ms=st["create_ms"], err=err)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="N = 1e6 at k = 1, degrees 4, 6, 8, 10 only")
    ap.add_argument("--kernel", default="yukawa", choices=["yukawa", "coulomb"])
    args = ap.parse_args()
    import torch
    from . import binding as B
    from . import inputs as I
    if not torch.cuda.is_available():
        sys.exit("sweep: no CUDA device -- the product has no CPU fallback")
    B.lib()
    Ns = (1_000_000,) if args.quick else (1_000_000, 2_000_000, 8_000_000)
    ks = (1.0,) if args.quick or args.kernel == "coulomb" else (0.5, 1.0, 5.0)      # the Coulomb kernel has no k
    degrees = (4, 6, 8, 10) if args.quick else tuple(range(4, 11))
    print(f"| N | k | theta | degree | ms / convolution | equiv. interactions/s | far evals | near evals | "
          f"N^2 / evals | bltc_create ms | BLTC vs direct (rel. 2-norm, 1e4 targets) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for N in Ns:
        cloud = Cloud(N, torch, B, I)
        for th in (0.5, 0.7, 0.9):
            for n in degrees:
                plan = B.bltc_create(None, cloud.X, cloud.w, N, th, n, cloud.c.batch_size, cloud.c.leaf_size)
                st = B.bltc_get_stats(plan)
                for k in ks:
                    r = run(cloud, plan, st, k, args.kernel, 3 if N < 4_000_000 else 2)
                    kk = "-" if args.kernel == "coulomb" else k
                    print(f"| {N} | {kk} | {th} | {n} | {r['ms']:.1f} | {r['rate']:.3e} | {r['far']:.3e} | {r['near']:.3e} | "
                          f"{float(N) ** 2 / (r['far'] + r['near']):.2f} | {r['create_ms']:.0f} | {r['err']:.2e} |", flush=True)
                B.bltc_destroy(plan)
        del cloud


if __name__ == "__main__":
    main()
