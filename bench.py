#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 BLTC Yukawa convolution (BASELINE.json metric).

  python bench.py --gpus N --steps K --warmup W            our CUDA path (one rank per GPU)
  python bench.py --impl reference --steps K --warmup W     the CPU oracle, as it stands, on host cores

A "step" is one pass of the whole hot path: one bltc_convolve call for all
orbitals of the workload = BASELINE.json configs[3], the largest single-GPU configuration (C6H6-like
molecule, adaptive Fejer mesh of 3,462,656 points, 21 orbitals, theta 0.7, degree 8, N_L = N_B = 2000;
PAPER.md:518 is the paper's largest system).  The plan (a0) is built once before the timed region and
reported separately, as the paper does (stage 1 vs stage 2).  The round-1 workload
(configs[1]) is timed for a few steps on the same build and reported under "cfg1".

value   = equivalent direct interactions per second = n_orb * N^2 / t_step (inputs in HBM)
e2e     = the same through the C ABI with HOST (pinned) buffers: H2D of f and D2H of out inside the
          timed region (min(K, 5) steps: a step is ~17 s)
roofline= FP64 ALU bound: executed FP64 flops of the pair kernel that dominates the step / its CUDA-event
          time / FP64 peak; the other pair kernel is reported beside it
cpu_baseline / cpu_baseline_fast = the CPU oracle (strict build = the parity oracle; -O3 -march=native
          -ffast-math build of the same sources) on a bounded sample, all host cores busy
Multi-GPU (--gpus N > 1): target batches are sharded over the ranks (strong scaling, one convolution),
the ranks' slices of `out` are all-gathered over NCCL; --shard replicas: every rank
convolves its own orbitals on the same mesh (weak scaling, no collective).
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
def _mix(first, per_extra, div=1.0):
    return {ot: (first + per_extra * (ot - 1)) / div for ot in range(1, 8)}


FLOPS_PER_PAIR = {(kern, ot): v for kern, tab in {
    "near": _mix(32.0, 14.0), "far": _mix(27.0, 15.0),
    # degree 8: far_kernel<..., N1 = 9>, one (k1, k2) row of 9 proxy points per loop trip incl. its dx^2 + dy^2
    "far9": _mix(239.0, 135.0, 9.0),
    # Coulomb kernel with Gaussian singularity subtraction (bltc_convolve_coulomb)
    "cnear": _mix(31.0, 4.0), "cfar": _mix(26.0, 4.0), "cfar9": _mix(230.0, 36.0, 9.0),
}.items() for ot, v in tab.items()}
# tiles of 6-7 orbitals unroll 3 proxy points per trip instead of a whole row (kernels.cu): the inner loop executes the
# generic far kernel's mix; the row prologue (dx^2 + dy^2, 5 flops per target and row of 9) is then NOT counted
for _ot in (6, 7):
    FLOPS_PER_PAIR[("far9", _ot)] = FLOPS_PER_PAIR[("far", _ot)]
    FLOPS_PER_PAIR[("cfar9", _ot)] = FLOPS_PER_PAIR[("cfar", _ot)]
# 148 SMs x 64 FP64 FMA lanes x 2 flops x 1.965 GHz (MEASURED_PEAKS.json sm_max_mhz); the DFMA-only
# probe (bltc_probe_fp64) measures 36.8 TFLOP/s on this pool's B200s.
FP64_PEAK_TFLOPS_NOMINAL = 148 * 64 * 2 * 1.965e9 / 1e12


def measured_hbm_gbs():
    """MEASURED_PEAKS.json's copy bandwidth (driver-written), else the profiling guide's fallback."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return 6650.0


def orbital_groups(n_orb):
    """The register tiles (orbital groups) the library cuts n_orb orbitals into: asked of the library itself."""
    from paper_2003_01833_b200 import binding as B
    return B.bltc_orbital_tiles(n_orb)


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
    """cfg3 (BASELINE.json configs[3], the largest single-GPU config) is the bench workload; cfg1 rides along as a
    5-step context run, the others are for profiling.
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
    """Evenly spread batch ids."""
    return sorted(set(int(round(i * (n_batches - 1) / max(count - 1, 1))) for i in range(count)))


# Both CPU legs (cpu_baseline inside the CUDA arm, --impl reference) time this sample.  40 and not 4: with 4 batches the
# batch-sum phase ran 0.14-0.19 s and carried 97 % of the extrapolated time, so two runs of the same oracle on the same
# box differed by 24 % (BENCH_r02); 40 batches give it ~2 s on configs[3] while the proxy-charge phase barely grows
# (a few batches already need the charges of most clusters).
CPU_SAMPLE_BATCHES = 40


_ORACLE_PLANS = {}


def cpu_oracle_sample(c, repeat=1, kernel="yukawa", fast=False, n_batches=None):
    """Time the CPU oracle's BLTC (as it stands) on a bounded sample of the workload -- CPU_SAMPLE_BATCHES evenly
    spread target batches, the first orbital -- and scale to the whole convolution phase by phase: the proxy-charge
    phase (Alg. 3 line 2) by particle-cluster pairs, the batch-cluster sums (line 3) by kernel evaluations, both times
    n_orb.  (A few batches need the proxy charges of a large share of all clusters, so scaling the whole sample by
    evaluation count alone would charge the CPU for upward passes it does once per convolution.)  The oracle's loops
    are parallel over clusters and over targets: every core is busy.  fast=True: the same sources built
    -O3 -march=native -ffast-math (oracle/liboracle_fast.so; timing only, never used for parity).
    Returns (equiv. interactions/s, seconds of the sample, description, threads)."""
    import oracle
    key = (c.name, c.theta, c.degree, c.leaf_size, c.batch_size, fast)
    if key not in _ORACLE_PLANS:          # the oracle's tree + lists: built once, outside every timed sample
        op = oracle.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size, fast=fast)
        _ORACLE_PLANS[key] = (op, op.export())
    op, e = _ORACLE_PLANS[key]
    size = e["cl_end"] - e["cl_begin"]
    batches = sample_batches(op.n_batches, n_batches or CPU_SAMPLE_BATCHES)
    ev, need = 0, set()
    for b in batches:
        nt = e["b_end"][b] - e["b_begin"][b]
        ev += nt * (op.P * (e["far_ptr"][b + 1] - e["far_ptr"][b])
                    + size[e["near_idx"][e["near_ptr"][b]:e["near_ptr"][b + 1]]].sum())
        need.update(e["far_idx"][e["far_ptr"][b]:e["far_ptr"][b + 1]].tolist())
    up_sample = int(size[sorted(need)].sum()) if need else 0
    up_total = int(size[np.unique(e["far_idx"])].sum()) if len(e["far_idx"]) else 0
    ev_total = op.far_evals + op.near_evals
    best = None
    for _ in range(repeat):
        t0 = time.perf_counter()
        if kernel == "coulomb":
            op.evaluate_coulomb(c.w, c.f[:1], alpha=1.0, batches=batches)
        else:
            op.evaluate(c.w, c.f[:1], c.k[:1], batches=batches)
        dt = time.perf_counter() - t0
        if best is None or dt < best[0]:
            best = (dt, op.phase_seconds[0], op.phase_seconds[1])
    dt, t_up, t_ev = best
    t_full = c.n_orb * ((t_up * up_total / up_sample if up_sample else 0.0) + t_ev * ev_total / ev)
    value = c.n_orb * float(c.N) ** 2 / t_full
    ntg = int(sum(e["b_end"][b] - e["b_begin"][b] for b in batches))
    threads = oracle.n_threads()
    build = ("-O3 -march=native -ffast-math build of the same sources (timing only)" if fast
             else "strict IEEE build, long-double sums: the parity oracle")
    desc = (f"CPU BLTC oracle (oracle/bltc_cpu.c, {build}) on {len(batches)} of {op.n_batches} target batches "
            f"({ntg} targets) x 1 of {c.n_orb} orbitals, {threads} OpenMP threads over clusters / targets: "
            f"{t_up:.2f} s proxy charges ({up_sample:.3g} of {up_total:.3g} particle-cluster pairs) + {t_ev:.2f} s "
            f"batch sums ({ev:.3g} of {ev_total:.3g} kernel evaluations); each phase scaled by its count, x n_orb")
    cpu_oracle_sample.last_phase_s = {"proxy_charges": t_up, "batch_sums": t_ev}
    return value, dt, desc, threads


def config_dict(c, args, world):
    """The `config` object of the JSON line -- the same for the CUDA arm and the reference arm."""
    coulomb = args.kernel == "coulomb"
    sharded = args.shard == "batches" and world > 1
    return {"workload": c.name + (f" (BASELINE.json configs[{args.workload[3:]}])" if not coulomb and not args.orbitals else ""),
            "kernel": "coulomb 1/r, Gaussian subtraction alpha = 1 (Eq. (23)-(24))" if coulomb
            else "yukawa e^{-kr}/(4 pi r), subtraction Eq. (20)-(21)", "N": c.N, "n_orb": c.n_orb, "theta": c.theta,
            "degree": c.degree, "leaf_size": c.leaf_size, "batch_size": c.batch_size,
            "subtract_singularity": True, "l2": "flushed between timed iterations (256 MB write)",
            "parallelism": ("1 GPU" if world == 1 else
                            f"target batches sharded over {world} ranks + all-gather of out "
                            f"({'fused into the epilogue over NVLink peer memory' if args.exchange == 'fused' else 'NCCL'})" if sharded
                            else f"{world} replicas (each rank its own orbitals), no collective")}


def run_reference(args):
    """The reference arm of this tier: the CPU oracle, as it stands, on the host cores -- every step times the
    same bounded sample as the CUDA arm's cpu_baseline leg."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c = workload(args.workload, args.kernel, args.orbitals)
    vals = []
    for i in range(args.warmup + args.steps):
        v, dt, desc, cores = cpu_oracle_sample(c, kernel=args.kernel)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals])) * 1e3
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "strong" if args.shard == "batches" and args.gpus > 1 else "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": config_dict(c, args, args.gpus),
        "note": "each step = the CPU oracle on a bounded sample of the workload (see cpu_baseline.sample)",
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "phase_s": cpu_oracle_sample.last_phase_s},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# FP64 instructions per (target, source / proxy point) pair of a tile of ot orbitals, as (first orbital, each further one),
# counted in the SASS (python -m paper_2003_01833_b200.sass_count), and how many of them are DFMAs with three distinct
# vector-register sources -- those hold the FP64 pipe for 3 cycles instead of 2 on sm_100a (microbenchmark table; this run's own dfma_probe_tflops)
FP64_INSTR_PER_PAIR = {"near": (22.0, 9.0), "far": (17.0, 9.0), "far9": (148.0 / 9, 9.0)}
FP64_3REG_PER_PAIR = {"near": 1.0, "far": 2.0, "far9": 2.0}            # per orbital: the accumulate (+ fhat - f_i what)


def fp64_pipe_busy(key, groups, evals, ms, sm_mhz, n_sm=148):
    """Share of the FP64 pipe's cycles that the kernel's FP64 instructions occupy: (2 cycles per instruction + 1 per
    three-register DFMA) x warp instructions / (4 sub-partitions x SMs x clock x time).  None for the Coulomb kernels."""
    if key not in FP64_INSTR_PER_PAIR or not sm_mhz or ms <= 0:
        return None
    cyc = 0.0
    for g in groups:
        first, extra = FP64_INSTR_PER_PAIR["far" if key == "far9" and g >= 6 else key]   # 6-7 orbitals: 3 points per trip
        cyc += evals / 32.0 * (2.0 * (first + extra * (g - 1)) + FP64_3REG_PER_PAIR[key] * g)
    return cyc / (4.0 * n_sm * sm_mhz * 1e6 * ms * 1e-3)


def roofline_of(phase_ms, st, groups, degree, coulomb, probe, steps, sm_mhz=None):
    """FP64-ALU roofline of the two pair kernels from the library's per-phase CUDA events: executed FP64 flops
    (SASS-counted mix x the plan's exact pair counts, summed over the orbital groups of one step) / kernel time."""
    pre = "c" if coulomb else ""
    far_key = pre + ("far9" if degree == 8 else "far")
    peak = FP64_PEAK_TFLOPS_NOMINAL
    out = {}
    for name, key, evals in (("near", pre + "near", st["near_evals"]), ("far", far_key, st["far_evals"])):
        ms = phase_ms[name] / steps                      # all launches of one step
        flops = sum(evals * FLOPS_PER_PAIR[(key, g)] for g in groups)
        tf = flops / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        out[name] = {"bound": "alu", "kernel": name + "_kernel", "achieved": tf, "peak": peak, "unit": "TFLOP/s",
                     "frac": tf / peak, "frac_of_measured_dfma_probe": tf / probe if probe else None,
                     "peak_source": "nominal: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md 6)",
                     "peak_measured_dfma_probe": probe, "launches_per_step": len(groups),
                     "orbital_tiles": groups, "avg_launch_ms": ms / len(groups),
                     "flops_per_launch": flops / len(groups), "ms_per_step": ms,
                     "fp64_pipe_busy": fp64_pipe_busy(key, groups, evals, ms, sm_mhz)}
    return out


def committed_traffic(workload_name, kernel):
    """DRAM bytes of one launch of `kernel` on this workload from the committed ncu capture (profiles/r02_traffic.csv:
    workload,kernel,dram_bytes_per_launch -- profiles/r02h_cfg3_launches.md names the command); None if not captured.
    A CONSTANT read from that file, not measured in this run: the line says so in roofline.traffic_source."""
    tpath = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    try:
        for line in open(tpath):
            p = [x.strip() for x in line.split(",")]
            if len(p) >= 3 and p[0] == workload_name and p[1] == kernel:
                return float(p[2])
    except Exception:
        pass
    return None


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
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log (NVLS / ring) stays on
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()

    coulomb = args.kernel == "coulomb"
    sharded = args.shard == "batches" and world > 1
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")   # > 126 MB L2
    warmup = max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(v):
        if world > 1:
            t = torch.tensor([v], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return v

    def time_workload(c, steps, warm, shard, e2e_steps, sample_clocks):
        """Plan + `steps` timed convolutions (device-resident) + `e2e_steps` through host buffers."""
        N, O = c.N, c.n_orb
        X = torch.from_numpy(c.coords()).cuda()
        w = torch.from_numpy(c.w).cuda()
        f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
        out = torch.zeros((O, N), dtype=torch.float64, device="cuda")      # a sharded plan writes its slice only
        exchange = None
        fused = None                                     # --exchange fused: results stored straight into the peers' buffers
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if shard and args.exchange == "fused":
            from paper_2003_01833_b200.multi_gpu import ShardedPlan
            fused = ShardedPlan(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size, fused_scatter=True)
            plan = fused.plan
        elif shard:  # strong scaling: rank r computes its slice of the target batches; the only exchange is the
            # all-gather of `out` that the next Green-Iteration step needs on every rank
            from paper_2003_01833_b200.multi_gpu import ShardExchange
            plan = B.bltc_create_sharded(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size, rank, world)
            exchange = ShardExchange(B.bltc_get_shard_targets(plan), N, "cuda")
        else:
            plan = B.bltc_create(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size)
        create_ms = (time.perf_counter() - t0) * 1e3
        create_cold_ms = create_ms
        if not shard:                                    # the first build pays module load and pool growth: time a second
            B.bltc_destroy(plan)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            plan = B.bltc_create(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size)
            create_ms = (time.perf_counter() - t0) * 1e3
        st = B.bltc_get_stats(plan)
        host_builder = None
        if not shard:                                    # the threaded host builder on the same box, for comparison
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            hplan = B.bltc_create_with_builder(None, X, w, N, c.theta, c.degree, c.batch_size, c.leaf_size, 0, 1,
                                               B.BUILDER_HOST)
            hms = (time.perf_counter() - t0) * 1e3
            hst = B.bltc_get_stats(hplan)
            host_builder = {"create_ms": hms, "build_ms": hst["build_ms"], "upload_ms": hst["upload_ms"]}
            B.bltc_destroy(hplan)

        def convolve(f_, out_):
            if fused is not None:                        # epilogue scatters over NVLink peer memory (symmetric memory)
                if coulomb:
                    fused.convolve_coulomb(f_, O, out_, True, 1.0)
                else:
                    fused.convolve(c.k, f_, O, out_, True)
                return
            if coulomb:
                B.bltc_convolve_coulomb(plan, f_, O, out_, True, 1.0)
            else:
                B.bltc_convolve(plan, c.k, f_, O, out_, True)
            if exchange is not None:
                exchange.all_gather_out(out_)

        # ---- device-resident timing ---------------------------------------------------------
        B.bltc_set_profiling(plan, True)
        for _ in range(warm):
            convolve(f, out)
        barrier()
        sampler = ClockSampler(local) if sample_clocks else None
        if sampler:
            sampler.start()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        phase_sum = {p: 0.0 for p in B.PHASES}
        barrier()
        for i in range(steps):
            flush.fill_(0.0)                                        # L2 flush between timed iterations
            ev[i][0].record(stream)
            convolve(f, out)
            ev[i][1].record(stream)
            ph = B.bltc_get_phase_ms(plan)                          # syncs on the step's last event
            for p in B.PHASES:
                phase_sum[p] += ph[p]
        barrier()
        clocks = sampler.stop() if sampler else None
        ms_per_step = max_over_ranks(sum(a.elapsed_time(b) for a, b in ev)) / steps

        # ---- end to end through the C ABI with host (pinned) buffers ----------------------------
        B.bltc_set_profiling(plan, False)
        e2e = None
        if e2e_steps > 0:
            f_host = torch.from_numpy(np.ascontiguousarray(c.f)).pin_memory()
            out_host = torch.zeros((O, N), dtype=torch.float64).pin_memory()
            out_dev = torch.zeros((O, N), dtype=torch.float64, device="cuda") if exchange is not None else None
            f_dev2 = torch.empty((O, N), dtype=torch.float64, device="cuda") if fused is not None else None

            def convolve_host():            # H2D(f) + a1..a5 + D2H(out) + stream sync, all inside the C call
                if fused is not None:       # the scatter call takes device buffers: copies made here, inside the timed region
                    f_dev2.copy_(f_host, non_blocking=True)
                    res_ = fused.convolve_coulomb(f_dev2, O, None, True, 1.0) if coulomb else fused.convolve(c.k, f_dev2, O, None, True)
                    out_host.copy_(res_, non_blocking=True)
                    torch.cuda.current_stream().synchronize()
                    return
                if coulomb:
                    B.bltc_convolve_coulomb(plan, f_host, O, out_host, True, 1.0)
                else:
                    B.bltc_convolve(plan, c.k, f_host, O, out_host, True)
                if exchange is not None:    # sharded: the ranks' slices are exchanged on the device
                    out_dev.copy_(out_host, non_blocking=True)
                    exchange.all_gather_out(out_dev)

            convolve_host()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e2e_ms = 0.0
            for i in range(e2e_steps):
                flush.fill_(0.0)
                e0.record(stream)
                convolve_host()
                e1.record(stream)
                e1.synchronize()
                e2e_ms += e0.elapsed_time(e1)
            barrier()
            e2e_ms = max_over_ranks(e2e_ms) / e2e_steps
            res = out_dev if exchange is not None else torch.from_numpy(out_host.numpy())
            same = bool(torch.equal(res.cpu(), out.cpu()))
            e2e = {"ms_per_step": e2e_ms, "steps": e2e_steps, "bitwise_equal_to_device_path": same}
        return dict(plan=plan, st=st, X=X, w=w, f=f, out=out, ms_per_step=ms_per_step, phase_sum=phase_sum,
                    create_ms=create_ms, create_cold_ms=create_cold_ms, host_builder=host_builder, clocks=clocks, e2e=e2e)

    # ---- the headline workload ----------------------------------------------------------------
    c = workload(args.workload, args.kernel, args.orbitals)
    N, O = c.N, c.n_orb
    e2e_steps = min(args.steps, 5)
    R = time_workload(c, args.steps, warmup, sharded, e2e_steps, True)
    plan, st, X, w, f, out = R["plan"], R["st"], R["X"], R["w"], R["f"], R["out"]
    ms_per_step = R["ms_per_step"]
    jobs = 1 if sharded else world          # replicas: every rank convolves its own orbitals on the same mesh
    value = jobs * O * float(N) ** 2 / (ms_per_step * 1e-3)
    e2e_value = jobs * O * float(N) ** 2 / (R["e2e"]["ms_per_step"] * 1e-3)
    groups = orbital_groups(O)
    launches_per_step = int(st["launches_per_group"]) * len(groups)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

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
        for i in range(1 + 3):
            flush.fill_(0.0)
            e0.record(stream)
            if coulomb:
                B.direct_convolve_coulomb(Tg, fT, M, X, w, f, N, O, dout, True, 1.0)
            else:
                B.direct_convolve(Tg, fT, M, X, w, f, N, c.k, O, dout, True)
            e1.record(stream)
            e1.synchronize()
            if i >= 1:
                d_ms.append(B.bltc_direct_get_kernel_ms()); d_total.append(e0.elapsed_time(e1))
        B.bltc_direct_set_profiling(False)
        dk = float(np.median(d_ms))
        d_flops = sum(float(M) * N * FLOPS_PER_PAIR[(("c" if coulomb else "") + "near", g)] for g in groups)
        direct = {"targets": M, "sources": N, "n_orb": O, "pair_kernel_ms": dk, "call_ms": float(np.median(d_total)),
                  "pairs_per_s": O * float(M) * N / (dk * 1e-3), "tflops": d_flops / (dk * 1e-3) / 1e12,
                  "frac": d_flops / (dk * 1e-3) / 1e12 / FP64_PEAK_TFLOPS_NOMINAL,
                  "note": "direct_convolve on a seeded target sample (the near field's pair kernel over all sources)"}

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
              "GBps": gi_bytes / (gi_t * 1e-3) / 1e9, "hbm_peak_GBps_measured": measured_hbm_gbs(),
              "note": "L2 flushed before each call; 4 dependent streaming kernels"}
        del phi, psi_old
    probe = B.bltc_probe_fp64(64) if rank == 0 else None
    probe3 = B.bltc_probe_fp64(64, form=1) if rank == 0 else None      # three-register DFMAs: 2/3 of the pipe's peak
    stq = dict(st, near_evals=st["shard_near_evals"], far_evals=st["shard_far_evals"]) if sharded else st
    roof = (roofline_of(R["phase_sum"], stq, groups, c.degree, coulomb, probe, args.steps, R["clocks"].get("sm_mhz"))
            if rank == 0 else None)
    phase_ms = {p: v / args.steps for p, v in R["phase_sum"].items()}
    create_ms, create_cold_ms, clocks, e2e_info = R["create_ms"], R["create_cold_ms"], R["clocks"], R["e2e"]
    host_builder = R["host_builder"]
    B.bltc_destroy(plan)
    del X, w, f, out, R

    # ---- context: the round-1 bench workload (configs[1]) on the same build, a few steps -----------------
    cfg1 = None
    if rank == 0 and world == 1 and args.workload == "cfg3" and not coulomb and not args.orbitals:
        c1 = workload("cfg1", args.kernel, 0)
        R1 = time_workload(c1, 5, 3, False, 0, False)
        r1 = roofline_of(R1["phase_sum"], R1["st"], orbital_groups(c1.n_orb), c1.degree, False, probe, 5,
                         clocks.get("sm_mhz"))
        cfg1 = {"workload": c1.name, "N": c1.N, "n_orb": c1.n_orb, "ms_per_step": R1["ms_per_step"],
                "value": c1.n_orb * float(c1.N) ** 2 / (R1["ms_per_step"] * 1e-3), "steps": 5,
                "near_frac": r1["near"]["frac"], "far_frac": r1["far"]["frac"],
                "plan_create_ms": R1["create_ms"]}
        B.bltc_destroy(R1["plan"])
        del R1

    if rank == 0:
        dom = "near" if roof["near"]["ms_per_step"] >= roof["far"]["ms_per_step"] else "far"
        other = "far" if dom == "near" else "near"
        roof[dom]["traffic"] = committed_traffic(args.workload if not args.orbitals else "", dom + "_kernel")
        roof[dom]["traffic_source"] = (None if roof[dom]["traffic"] is None else
                                       "committed ncu capture of an earlier build, not this run: profiles/r02_traffic.csv "
                                       "(command in profiles/r02h_cfg3_launches.md)")
        cpu_v, cpu_dt, cpu_desc, cores = cpu_oracle_sample(c, kernel=args.kernel)
        cpu_phase_s = cpu_oracle_sample.last_phase_s
        fast_v, fast_dt, fast_desc, fast_cores = cpu_oracle_sample(c, kernel=args.kernel, fast=True)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(c, args, world),
            "time_per_convolution_ms": ms_per_step / O,
            "actual_evals_per_s": (st["near_evals"] + st["far_evals"]) * O * jobs / (ms_per_step * 1e-3),
            "phase_ms": phase_ms,
            "plan": {"create_ms": create_ms, "create_cold_ms": create_cold_ms,
                     "built_on_device": bool(st["built_on_device"]), "build_ms": st["build_ms"],
                     "stage_ms": {"tree": st["tree_ms"], "lists": st["lists_ms"], "decomposition": st["decomp_ms"],
                                  "upload_and_proxy_weights": st["upload_ms"]},
                     "host_builder": host_builder,
                     "clusters": st["n_clusters"], "batches": st["n_batches"],
                     "far_evals": st["far_evals"], "near_evals": st["near_evals"]},
            "roofline": roof[dom], "roofline_" + other: roof[other],
            "dfma_probe_tflops": {"two_register_sources": probe, "three_register_sources": probe3,
                                  "note": "DFMA-only kernels (bltc_probe_fp64_form): a DFMA with three distinct vector-"
                                          "register sources holds the FP64 pipe for 3 cycles instead of 2"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": O * N * 8,
                    "d2h_bytes_per_step": O * N * 8, "ms_per_step": e2e_info["ms_per_step"],
                    "steps": e2e_info["steps"],
                    "bitwise_equal_to_device_path": e2e_info["bitwise_equal_to_device_path"]},
            "direct": direct,
            "gi_update": gi,
            "cfg1": cfg1,
            "gpu_launches": launches_per_step * args.steps,
            "clocks": clocks,
            "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": cpu_desc,
                             "phase_s": cpu_phase_s},
            "cpu_baseline_fast": {"value": fast_v, "unit": UNIT, "cores": fast_cores, "kind": "oracle, fast-math build",
                                  "sample": fast_desc},
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--shard", default="batches", choices=["replicas", "batches"],
                    help="N > 1: batches = one convolution, target batches sharded over the ranks + all-gather of out "
                         "(strong scaling, default); replicas = each rank convolves its own orbitals (weak scaling)")
    ap.add_argument("--exchange", default="nccl", choices=["nccl", "fused"],
                    help="N > 1, --shard batches: nccl = gather kernel + ONE all_gather_into_tensor + scatter kernel (default); "
                         "fused = the epilogue kernel stores into every rank's buffer over NVLink peer memory "
                         "(torch symmetric memory), no collective")
    ap.add_argument("--workload", default="cfg3", choices=["cfg0", "cfg1", "cfg2", "cfg3"],
                    help="cfg3 = BASELINE.json configs[3], the largest single-GPU config (the bench line); "
                         "others: profiling / context")
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
