#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 BLTC Yukawa convolution (BASELINE.json metric).

  python bench.py --gpus N --steps K --warmup W            our CUDA path (one rank per GPU)
  python bench.py --impl reference --steps K --warmup W     the CPU oracle, as it stands, on host cores

A "step" is one pass of the whole hot path: one bltc_convolve call for all
orbitals of the workload = BASELINE.json configs[1] (Be-like atom, adaptive Fejer mesh, 2 orbitals,
theta 0.7, degree 8, N_L = N_B = 2000).  The plan (a0, host tree build) is built once before the
timed region and reported separately, as the paper does (stage 1 vs stage 2).

value   = equivalent direct interactions per second = n_orb * N^2 * n_gpus / t_step (inputs in HBM)
e2e     = the same through the C ABI with HOST (pinned) buffers: H2D of f and D2H of out inside the
          timed region
roofline= FP64 ALU bound: executed FP64 flops of the dominant kernel / its CUDA-event time / FP64 peak
Multi-GPU: the path does not need to shard on one node ("replicas only"): every rank runs
the same convolution on its own GPU (weak scaling), no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "fp64 BLTC convolution, equivalent direct interactions/s"
UNIT = "interactions/s"

# FP64 instruction mix of one kernel evaluation, counted in the SASS of the inner loops
# (profiles/r01*_sass_counts.md; tests/test_library_host.py re-counts them from the built library).  flops = 2*DFMA + DMUL + DADD.
# key: (kernel, orbital tile width OT) -> flops per (target, source/proxy point) pair for ALL OT orbitals
FLOPS_PER_PAIR = {
    ("near", 1): 32.0, ("near", 2): 46.0, ("near", 3): 60.0, ("near", 4): 74.0,
    ("far", 1): 27.0, ("far", 2): 42.0, ("far", 3): 57.0, ("far", 4): 72.0,
    # degree 8: far_kernel<..., N1 = 9>, one (k1, k2) row of 9 proxy points per loop trip incl. its dx^2 + dy^2
    ("far9", 1): 239.0 / 9, ("far9", 2): 374.0 / 9, ("far9", 3): 509.0 / 9, ("far9", 4): 644.0 / 9,
    # Coulomb kernel with Gaussian singularity subtraction (bltc_convolve_coulomb)
    ("cnear", 1): 31.0, ("cnear", 2): 35.0, ("cnear", 3): 39.0, ("cnear", 4): 43.0,
    ("cfar", 1): 26.0, ("cfar", 2): 30.0, ("cfar", 3): 34.0, ("cfar", 4): 38.0,
    ("cfar9", 1): 230.0 / 9, ("cfar9", 2): 266.0 / 9, ("cfar9", 3): 302.0 / 9, ("cfar9", 4): 338.0 / 9,
}
# 148 SMs x 64 FP64 FMA lanes x 2 flops x 1.965 GHz (MEASURED_PEAKS.json sm_max_mhz); the DFMA-only
# probe (bltc_probe_fp64) measures 36.8 TFLOP/s on this pool's B200s.
FP64_PEAK_TFLOPS_NOMINAL = 148 * 64 * 2 * 1.965e9 / 1e12


def orbital_groups(n_orb, max_ot=4):
    ng = (n_orb + max_ot - 1) // max_ot
    g = [n_orb // ng] * ng
    for i in range(n_orb % ng):
        g[i] += 1
    return g


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def workload(name="cfg1", kernel="yukawa", orbitals=0):
    """cfg1 (BASELINE.json configs[1]) is the bench workload; the others are for profiling and context runs.
    kernel = "coulomb": the same mesh with ONE field, the density rho = 2 sum_o psi_o^2 -- the Hartree
    potential of bltc_convolve_coulomb (Table 4's workload shape)."""
    from paper_2003_01833_b200 import inputs as I
    c = {"cfg0": I.config0, "cfg1": I.config1, "cfg2": I.config2, "cfg3": I.config3}[name]()
    if kernel == "coulomb":
        c = I.density_workload(c)
    if orbitals > 0:      # profiling aid: the config's fields cycled to `orbitals` orbitals, k spread by 7 % steps
        src = c.f.copy(); k0 = c.k.copy()
        c.f = np.ascontiguousarray(np.stack([src[o % src.shape[0]] * (1.0 + 0.01 * o) for o in range(orbitals)]))
        c.k = np.array([k0[o % k0.shape[0]] * (1.0 + 0.07 * (o // k0.shape[0])) for o in range(orbitals)])
        c.name += f"_x{orbitals}orb"
    return c


def sample_batches(n_batches, count=4):
    """Evenly spread batch ids; cfg1 (568 batches) keeps the ids the earlier rounds used."""
    if n_batches == 568:
        return [0, 137, 301, 567][:count]
    return sorted(set(int(round(i * (n_batches - 1) / max(count - 1, 1))) for i in range(count)))


def cpu_oracle_sample(c, batches, repeat=1, kernel="yukawa"):
    """Time the CPU oracle's BLTC (as it stands) on a bounded sample of target batches and scale to the
    whole convolution by evaluation count.  Returns (equiv. interactions/s, seconds, description)."""
    import oracle
    op = oracle.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    e = op.export()
    size = e["cl_end"] - e["cl_begin"]
    ev = 0
    if isinstance(batches, int):
        batches = sample_batches(op.n_batches, batches)
    for b in batches:
        nt = e["b_end"][b] - e["b_begin"][b]
        ev += nt * (op.P * (e["far_ptr"][b + 1] - e["far_ptr"][b])
                    + size[e["near_idx"][e["near_ptr"][b]:e["near_ptr"][b + 1]]].sum())
    total = op.far_evals + op.near_evals
    best = None
    for _ in range(repeat):
        t0 = time.perf_counter()
        if kernel == "coulomb":
            op.evaluate_coulomb(c.w, c.f, alpha=1.0, batches=list(batches))
        else:
            op.evaluate(c.w, c.f, c.k, batches=list(batches))
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    t_full = best * total / ev                       # seconds for all batches, all orbitals
    value = c.n_orb * float(c.N) ** 2 / t_full
    ntg = int(sum(e["b_end"][b] - e["b_begin"][b] for b in batches))
    desc = (f"CPU BLTC oracle (oracle/bltc_cpu.c, strict IEEE, long-double sums) on {len(batches)} of "
            f"{op.n_batches} target batches ({ntg} targets, {c.n_orb} orbitals, {ev * c.n_orb:.3g} kernel "
            f"evaluations incl. their proxy charges), {best:.2f} s, scaled by evaluation count to the "
            f"whole convolution")
    return value, best, desc, oracle.n_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c = workload(args.workload, args.kernel, args.orbitals)
    batches = [137] if args.workload == "cfg1" else 1
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt, desc, cores = cpu_oracle_sample(c, batches, kernel=args.kernel)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": c.name, "N": c.N, "n_orb": c.n_orb, "theta": c.theta, "degree": c.degree,
                   "leaf_size": c.leaf_size, "batch_size": c.batch_size,
                   "note": "each step = the CPU oracle on a bounded sample of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2003_01833_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()

    c = workload(args.workload, args.kernel, args.orbitals)
    coulomb = args.kernel == "coulomb"
    N, O = c.N, c.n_orb

    def convolve(f_, out_):
        if coulomb:
            B.bltc_convolve_coulomb(plan, f_, O, out_, True, 1.0)
        else:
            B.bltc_convolve(plan, c.k, f_, O, out_, True)
        if exchange is not None and out_.is_cuda:
            exchange.all_gather_out(out_)

    X = torch.from_numpy(c.coords()).cuda()
    w = torch.from_numpy(c.w).cuda()
    f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
    out = torch.zeros((O, N), dtype=torch.float64, device="cuda")      # a sharded plan writes its slice only
    t0 = time.perf_counter()
    sharded = args.shard == "batches" and world > 1
    exchange = None
    if sharded:      # strong scaling: rank r computes its slice of the target batches; the only exchange is the
        # all-gather of `out` that the next Green-Iteration step needs on every rank
        from paper_2003_01833_b200.multi_gpu import ShardExchange
        plan = B.bltc_create_sharded(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size, rank, world)
        exchange = ShardExchange(B.bltc_get_shard_targets(plan), N, "cuda")
    else:
        plan = B.bltc_create(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size)
    create_ms = (time.perf_counter() - t0) * 1e3
    st = B.bltc_get_stats(plan)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    groups = orbital_groups(O)
    launches_per_step = int(st["launches_per_group"]) * len(groups)

    # ---- device-resident timing -------------------------------------------------------------
    B.bltc_set_profiling(plan, True)
    for _ in range(max(args.warmup, 3)):
        convolve(f, out)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phase_sum = {p: 0.0 for p in B.PHASES}
    barrier()
    for i in range(args.steps):
        flush.fill_(0.0)                                        # L2 flush between timed iterations
        ev[i][0].record(stream)
        convolve(f, out)
        ev[i][1].record(stream)
        ph = B.bltc_get_phase_ms(plan)                          # syncs on the step's last event
        for p in B.PHASES:
            phase_sum[p] += ph[p]
    barrier()
    clocks = sampler.stop()
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    if world > 1:
        t = torch.tensor([t_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_ms = float(t.item())
    ms_per_step = t_ms / args.steps
    jobs = 1 if sharded else world          # replicas: every rank convolves its own orbitals on the same mesh
    value = jobs * O * float(N) ** 2 / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with host buffers ------------------------------------
    B.bltc_set_profiling(plan, False)
    f_host = torch.from_numpy(np.ascontiguousarray(c.f)).pin_memory()
    out_host = torch.zeros((O, N), dtype=torch.float64).pin_memory()
    for _ in range(2):
        convolve(f_host, out_host)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_ms = 0.0
    for i in range(args.steps):
        flush.fill_(0.0)
        e0.record(stream)
        convolve(f_host, out_host)                              # H2D(f) + a1..a5 + D2H(out) + stream sync
        e1.record(stream)
        e1.synchronize()
        e2e_ms += e0.elapsed_time(e1)
    barrier()
    if world > 1:
        t = torch.tensor([e2e_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t.item())
    e2e_value = jobs * O * float(N) ** 2 / (e2e_ms / args.steps * 1e-3)
    same = bool(np.array_equal(out_host.numpy(), out.cpu().numpy()))

    # ---- a6: brute-force direct sum on a bounded target sample of this workload --------
    direct = None
    if rank == 0:
        from paper_2003_01833_b200 import inputs as I
        M = min(N, 16384)
        idx = torch.from_numpy(I.sample_targets(N, M, seed=1)).cuda()
        Tg = X[:, idx].contiguous()
        fT = f[:, idx].contiguous()
        dout = torch.empty((O, M), dtype=torch.float64, device="cuda")
        B.bltc_direct_set_profiling(True)
        d_ms, d_total = [], []
        for i in range(2 + 5):
            flush.fill_(0.0)
            e0.record(stream)
            if coulomb:
                B.direct_convolve_coulomb(Tg, fT, M, X, w, f, N, O, dout, True, 1.0)
            else:
                B.direct_convolve(Tg, fT, M, X, w, f, N, c.k, O, dout, True)
            e1.record(stream)
            e1.synchronize()
            if i >= 2:
                d_ms.append(B.bltc_direct_get_kernel_ms()); d_total.append(e0.elapsed_time(e1))
        B.bltc_direct_set_profiling(False)
        dk = float(np.median(d_ms))
        d_flops = sum(float(M) * N * FLOPS_PER_PAIR[(("c" if coulomb else "") + "near", g)] for g in orbital_groups(O))
        direct = {"targets": M, "sources": N, "n_orb": O, "pair_kernel_ms": dk, "call_ms": float(np.median(d_total)),
                  "pairs_per_s": O * float(M) * N / (dk * 1e-3), "tflops": d_flops / (dk * 1e-3) / 1e12,
                  "frac": d_flops / (dk * 1e-3) / 1e12 / FP64_PEAK_TFLOPS_NOMINAL,
                  "note": "direct_convolve on a seeded target sample (same pair kernel as the near field, "
                          "r == 0 test and underflow guard compiled in)"}

    # ---- NEXT-2: Green-Iteration epilogue (Alg. 2 lines 4-7) on this mesh, HBM-bound ------------------
    gi = None
    if rank == 0:
        n_prev = 4
        rng = np.random.default_rng(7)
        phi = torch.from_numpy(rng.standard_normal((n_prev, N))).cuda()
        psi_old = torch.from_numpy(rng.standard_normal(N)).cuda()
        res = torch.empty(4 + n_prev, dtype=torch.float64, device="cuda")
        gi_ms = []
        for i in range(3 + 10):
            psi_new = out[0].clone()
            flush.fill_(0.0)
            e0.record(stream)
            B.bltc_gi_update(w, psi_old, f[0], psi_new, phi, n_prev, N, -0.5, res)
            e1.record(stream)
            e1.synchronize()
            if i >= 3:
                gi_ms.append(e0.elapsed_time(e1))
        gi_bytes = (11 + 2 * n_prev) * 8 * N          # K1 reads 4+n, K2 reads 2+n writes 1, K3 reads 3 writes 1
        gi_t = float(np.median(gi_ms))
        gi = {"ms": gi_t, "n_prev": n_prev, "launches": 4, "algorithmic_bytes": gi_bytes,
              "GBps": gi_bytes / (gi_t * 1e-3) / 1e9, "note": "L2 flushed before each call; 4 small kernels: launch-latency bound at this N"}

    if rank == 0:
        near_ms = phase_sum["near"] / args.steps / len(groups)      # average launch duration
        far_ms = phase_sum["far"] / args.steps / len(groups)
        pre = "c" if coulomb else ""
        if sharded:                          # rank 0's kernels work on rank 0's slice
            st = dict(st, near_evals=st["shard_near_evals"], far_evals=st["shard_far_evals"])
        near_flops = sum(st["near_evals"] * FLOPS_PER_PAIR[(pre + "near", g)] for g in groups) / len(groups)
        far_key = pre + ("far9" if c.degree == 8 else "far")
        far_flops = sum(st["far_evals"] * FLOPS_PER_PAIR[(far_key, g)] for g in groups) / len(groups)
        peak = FP64_PEAK_TFLOPS_NOMINAL
        near_tf = near_flops / (near_ms * 1e-3) / 1e12
        far_tf = far_flops / (far_ms * 1e-3) / 1e12 if far_ms > 0 else 0.0
        probe = B.bltc_probe_fp64(64)
        # DRAM bytes of one near-kernel launch of THIS workload from the committed ncu capture
        # (profiles/r01g_summary.md names the command); null for other workloads / kernels
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "r01g_near_cfg1_dram.csv")
        if args.workload == "cfg1" and not coulomb and os.path.exists(tpath):
            try:
                import csv
                rows = [r for r in csv.reader(open(tpath)) if len(r) > 5 and r[-3].startswith("dram__bytes")]
                traffic = float(sum(float(r[-1].replace(",", "")) for r in rows)) if rows else None
            except Exception:
                traffic = None
        cpu_v, cpu_dt, cpu_desc, cores = cpu_oracle_sample(c, 4, kernel=args.kernel)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": c.name + (" (BASELINE.json configs[1])" if args.workload == "cfg1" and not coulomb else ""),
                       "kernel": "coulomb 1/r, Gaussian subtraction alpha = 1 (Eq. (23)-(24))" if coulomb
                       else "yukawa e^{-kr}/(4 pi r), subtraction Eq. (20)-(21)", "N": N, "n_orb": O, "theta": c.theta,
                       "degree": c.degree, "leaf_size": c.leaf_size, "batch_size": c.batch_size,
                       "subtract_singularity": True, "l2": "flushed between timed iterations (256 MB write)",
                       "parallelism": ("1 GPU" if world == 1 else
                                       f"target batches sharded over {world} ranks + all-gather of out (NCCL)" if sharded
                                       else f"{world} replicas (each rank its own orbitals), no collective")},
            "time_per_convolution_ms": ms_per_step / O,
            "actual_evals_per_s": (st["near_evals"] + st["far_evals"]) * O * world / (ms_per_step * 1e-3),
            "phase_ms": {p: phase_sum[p] / args.steps for p in B.PHASES},
            "plan": {"create_ms": create_ms, "host_build_ms": st["build_ms"], "upload_ms": st["upload_ms"],
                     "clusters": st["n_clusters"], "batches": st["n_batches"],
                     "far_evals": st["far_evals"], "near_evals": st["near_evals"]},
            "roofline": {"bound": "alu", "kernel": "near_kernel", "achieved": near_tf, "peak": peak,
                         "unit": "TFLOP/s", "frac": near_tf / peak, "traffic": traffic,
                         "peak_source": "nominal: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md)",
                         "peak_measured_dfma_probe": probe, "avg_launch_ms": near_ms,
                         "flops_per_launch": near_flops},
            "roofline_far": {"bound": "alu", "kernel": "far_kernel", "achieved": far_tf, "peak": peak,
                             "unit": "TFLOP/s", "frac": far_tf / peak, "avg_launch_ms": far_ms,
                             "flops_per_launch": far_flops},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": O * N * 8,
                    "d2h_bytes_per_step": O * N * 8, "ms_per_step": e2e_ms / args.steps,
                    "bitwise_equal_to_device_path": same},
            "direct": direct,
            "gi_update": gi,
            "gpu_launches": launches_per_step * args.steps,
            "clocks": clocks,
            "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_desc},
        }
        print(json.dumps(line))
    B.bltc_destroy(plan)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--shard", default="replicas", choices=["replicas", "batches"],
                    help="N > 1: replicas = each rank convolves its own orbitals (weak scaling, default); "
                         "batches = one convolution, target batches sharded over the ranks (strong scaling)")
    ap.add_argument("--workload", default="cfg1", choices=["cfg0", "cfg1", "cfg2", "cfg3"],
                    help="cfg1 = BASELINE.json configs[1] (the bench line); others: profiling / context")
    ap.add_argument("--orbitals", type=int, default=0,
                    help="profiling aid: cycle the workload's fields to this many orbitals (0 = as configured)")
    ap.add_argument("--kernel", default="yukawa", choices=["yukawa", "coulomb"],
                    help="coulomb: Hartree potential with Gaussian singularity subtraction (NEXT-1)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
