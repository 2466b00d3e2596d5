"""Multi-GPU batch sharding: bltc_create_sharded gives rank r of
`world` a contiguous slice of the target batches with ~1/world of the kernel evaluations; no data-path
collective is needed (batches are independent given the sources and the proxy charges).

CPU tests: the slicing itself, and a world_size-2 `gloo` run of the whole N > 1 host logic (each rank takes its
slice, computes it -- with the CPU oracle standing in for the device -- and the ranks assemble the result).
GPU test: every rank's plan run one after the other on one device into one output buffer.
"""
import os
import socket

import numpy as np
import pytest

from paper_2003_01833_b200 import binding as B
from paper_2003_01833_b200 import inputs as I


def _cloud():
    return I.random_cloud(20000, n_orb=2, seed=21, clustered=True, leaf_size=300, batch_size=300, degree=4)


@pytest.mark.parametrize("world", [1, 2, 3, 5, 8])
def test_shard_slices_partition_the_batches(world):
    c = _cloud()
    X = c.coords()
    full = B.bltc_get_stats(B.bltc_create_host_plan(None, X, None, c.N, c.theta, c.degree, c.batch_size, c.leaf_size))
    nb = full["n_batches"]
    assert (full["shard_rank"], full["shard_world"], full["shard_batch_begin"], full["shard_batch_end"]) == (0, 1, 0, nb)
    assert full["shard_targets"] == c.N
    at, seen, ev = 0, [], []
    for r in range(world):
        p = B.bltc_create_host_plan_sharded(None, X, None, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, r, world)
        st = B.bltc_get_stats(p)
        # the tree, batches and lists are the whole problem's on every rank
        for key in ("n_clusters", "n_leaves", "n_batches", "n_far", "n_near", "far_evals", "near_evals"):
            assert st[key] == full[key], key
        assert (st["shard_rank"], st["shard_world"]) == (r, world)
        assert st["shard_batch_begin"] == at and st["shard_batch_end"] >= at      # contiguous, in rank order
        at = st["shard_batch_end"]
        idx = B.bltc_get_shard_targets(p)
        assert idx.shape[0] == st["shard_targets"]
        e = B.bltc_export_plan(p)
        b0, b1 = st["shard_batch_begin"], st["shard_batch_end"]
        if b1 > b0:                                                              # exactly its batches' targets
            np.testing.assert_array_equal(idx, e["tgt_perm"][e["b_begin"][b0]:e["b_end"][b1 - 1]])
        seen.append(idx)
        ev.append(st["shard_far_evals"] + st["shard_near_evals"])
        assert st["n_proxy_clusters"] <= full["n_proxy_clusters"]
    assert at == nb
    allidx = np.concatenate(seen)
    np.testing.assert_array_equal(np.sort(allidx), np.arange(c.N))               # disjoint cover of the targets
    assert sum(ev) == full["far_evals"] + full["near_evals"]
    # balance: no slice is further from the mean than the most expensive single batch
    e = B.bltc_export_plan(B.bltc_create_host_plan(None, X, None, c.N, c.theta, c.degree, c.batch_size, c.leaf_size))
    size = e["cl_end"] - e["cl_begin"]
    cost = np.array([(e["b_end"][b] - e["b_begin"][b]) * ((c.degree + 1) ** 3 * (e["far_ptr"][b + 1] - e["far_ptr"][b])
                     + size[e["near_idx"][e["near_ptr"][b]:e["near_ptr"][b + 1]]].sum()) for b in range(nb)])
    assert cost.sum() == sum(ev)
    assert max(abs(v - cost.sum() / world) for v in ev) <= cost.max()


def test_shard_rejects_bad_rank():
    c = I.random_cloud(500, seed=1, leaf_size=100, batch_size=100, degree=3)
    for rank, world in ((-1, 2), (2, 2), (0, 0)):
        with pytest.raises(B.BltcError):
            B.bltc_create_host_plan_sharded(None, c.coords(), None, c.N, 0.7, 3, 100, 100, rank, world)


def test_more_ranks_than_batches_leaves_empty_slices():
    c = I.random_cloud(300, seed=2, leaf_size=200, batch_size=200, degree=2)     # a handful of batches
    X = c.coords()
    nb = B.bltc_get_stats(B.bltc_create_host_plan(None, X, None, c.N, 0.7, 2, 200, 200))["n_batches"]
    world = nb + 3
    tot = 0
    for r in range(world):
        st = B.bltc_get_stats(B.bltc_create_host_plan_sharded(None, X, None, c.N, 0.7, 2, 200, 200, r, world))
        tot += st["shard_targets"]
    assert tot == c.N


def test_shards_with_separate_targets_and_second_tree():
    # targets != sources (batches from a second tree) and N_B != N_L: slices are cut over the TARGET batches
    c = I.random_cloud(8000, seed=23, leaf_size=300, batch_size=120, degree=3)
    rng = np.random.default_rng(5)
    T = np.ascontiguousarray(rng.random((3, c.N)))
    world, seen = 4, []
    for r in range(world):
        p = B.bltc_create_host_plan_sharded(T, c.coords(), None, c.N, 0.7, 3, 120, 300, r, world)
        st = B.bltc_get_stats(p)
        assert st["shared_batches"] == 0
        seen.append(B.bltc_get_shard_targets(p))
        assert len(seen[-1]) == st["shard_targets"]
    np.testing.assert_array_equal(np.sort(np.concatenate(seen)), np.arange(c.N))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _gloo_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        c = I.random_cloud(6000, n_orb=2, seed=22, clustered=True, leaf_size=200, batch_size=200, degree=4)
        p = B.bltc_create_host_plan_sharded(None, c.coords(), None, c.N, c.theta, c.degree, c.batch_size,
                                            c.leaf_size, rank, world)
        st = B.bltc_get_stats(p)
        idx = B.bltc_get_shard_targets(p)
        # the device's part, played by the CPU oracle on exactly this rank's batches (same tree: checked in
        # test_library_host.py): out is written only for the slice's targets
        op = oracle.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
        mine = op.evaluate(c.w, c.f, c.k, batches=list(range(st["shard_batch_begin"], st["shard_batch_end"])))
        written = ~np.isnan(mine[0])
        assert np.array_equal(np.sort(np.nonzero(written)[0]), np.sort(idx))
        # assembly, the product's way: ShardExchange all-gathers the slices (values only; indices exchanged once)
        from paper_2003_01833_b200.multi_gpu import ShardExchange
        ex = ShardExchange(idx, c.N, "cpu")
        assert ex.counts[rank] == len(idx) and sum(ex.counts) == c.N
        out = torch.from_numpy(mine.copy())                       # NaN outside this rank's slice
        ex.all_gather_out(out)
        assert not torch.isnan(out).any()
        # and the simple way: untouched elements zero, sum over ranks (exact: x + 0) -- must agree bitwise
        out2 = torch.from_numpy(np.where(np.isnan(mine), 0.0, mine))
        dist.all_reduce(out2, op=dist.ReduceOp.SUM)
        assert torch.equal(out, out2)
        counts = torch.tensor([int(written.sum())], dtype=torch.int64)
        dist.all_reduce(counts, op=dist.ReduceOp.SUM)
        evals = torch.tensor([st["shard_far_evals"] + st["shard_near_evals"]], dtype=torch.int64)
        dist.all_reduce(evals, op=dist.ReduceOp.SUM)
        if rank == 0:
            full = op.evaluate(c.w, c.f, c.k)
            q.put((bool(np.array_equal(out.numpy(), full)), int(counts.item()) == c.N,
                   int(evals.item()) == op.far_evals + op.near_evals))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_gloo_sharded_convolution_assembles_to_the_full_result(oracle_mod, world):
    # world 4 on this cloud's batches leaves uneven slices; test_gloo_exchange_with_an_empty_slice covers an empty one
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == (True, True, True), res


def _gloo_empty_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2003_01833_b200.multi_gpu import ShardExchange
        # 3 batches over 4 ranks: at least one rank owns nothing (bltc_create_sharded gives it an empty slice)
        c = I.random_cloud(150, seed=3, leaf_size=200, batch_size=200, degree=3)   # one batch: three ranks own nothing
        p = B.bltc_create_host_plan_sharded(None, c.coords(), None, c.N, 0.5, 3, 200, 200, rank, world)
        idx = B.bltc_get_shard_targets(p)
        ex = ShardExchange(idx, c.N, "cpu")
        out = torch.full((3, c.N), float("nan"), dtype=torch.float64)
        col = torch.from_numpy(idx)
        out[:, col] = torch.arange(3, dtype=torch.float64)[:, None] * 1000.0 + col.to(torch.float64)[None, :]
        ex.all_gather_out(out)
        want = torch.arange(3, dtype=torch.float64)[:, None] * 1000.0 + torch.arange(c.N, dtype=torch.float64)[None, :]
        n_empty = torch.tensor([int(len(idx) == 0)])
        dist.all_reduce(n_empty)
        ok = torch.tensor([int(torch.equal(out, want))])
        dist.all_reduce(ok)
        if rank == 0:
            q.put((int(ok.item()), int(n_empty.item()), ex.bytes_per_step(3)))
    finally:
        dist.destroy_process_group()


def test_gloo_exchange_with_an_empty_slice():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_empty_worker, args=(r, 4, port, q)) for r in range(4)]
    for p in procs:
        p.start()
    ok, n_empty, nbytes = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ok == 4 and n_empty >= 1 and nbytes > 0


@pytest.mark.gpu
def test_gpu_sharded_plan_host_out_keeps_the_other_ranks_elements():
    # bltc.h: a sharded plan writes its own targets only -- also when `out` is a host buffer staged through the device
    import torch
    c = _cloud()
    X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
    f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
    plan = B.bltc_create_sharded(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, 1, 3)
    idx = B.bltc_get_shard_targets(plan)
    dev = torch.full((c.n_orb, c.N), float("nan"), dtype=torch.float64, device="cuda")
    B.bltc_convolve(plan, c.k, f, c.n_orb, dev, True)
    host = np.full((c.n_orb, c.N), np.nan)
    B.bltc_convolve(plan, c.k, f, c.n_orb, host, True)
    torch.cuda.synchronize()
    mine = np.zeros(c.N, bool); mine[idx] = True
    assert np.isnan(host[:, ~mine]).all() and not np.isnan(host[:, mine]).any()
    np.testing.assert_array_equal(host[:, mine], dev.cpu().numpy()[:, mine])
    B.bltc_destroy(plan)


@pytest.mark.gpu
@pytest.mark.parametrize("kernel", ["yukawa", "coulomb"])
def test_gpu_sharded_plans_cover_all_targets_and_match_the_oracle(oracle_mod, kernel):
    import torch
    assert torch.cuda.is_available()
    c = _cloud()
    X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
    f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
    world = 3
    out = torch.full((c.n_orb, c.N), float("nan"), dtype=torch.float64, device="cuda")
    seen = 0
    for r in range(world):
        plan = B.bltc_create_sharded(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, r, world)
        before = torch.isnan(out[0]).sum().item()
        if kernel == "yukawa":
            B.bltc_convolve(plan, c.k, f, c.n_orb, out, True)
        else:
            B.bltc_convolve_coulomb(plan, f, c.n_orb, out, True, 0.2)
        torch.cuda.synchronize()
        st = B.bltc_get_stats(plan)
        assert before - torch.isnan(out[0]).sum().item() == st["shard_targets"]   # wrote its slice, nothing else
        seen += st["shard_targets"]
        B.bltc_destroy(plan)
    assert seen == c.N and not torch.isnan(out).any()
    op = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    ref = op.evaluate(c.w, c.f, c.k) if kernel == "yukawa" else op.evaluate_coulomb(c.w, c.f, alpha=0.2)
    got = out.cpu().numpy()
    err = max(np.linalg.norm(got[o] - ref[o]) / np.linalg.norm(ref[o]) for o in range(c.n_orb))
    assert err <= 1e-12, err


@pytest.mark.gpu
def test_gpu_sharded_plan_with_nccl_world1_equals_plain_convolve():
    # the CUDA-tensor path of ShardedPlan / ShardExchange (NCCL backend; a 1-rank group is all one GPU allows)
    import torch
    import torch.distributed as dist
    from paper_2003_01833_b200.multi_gpu import ShardedPlan
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(_free_port())
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        c = I.random_cloud(6000, n_orb=3, seed=24, clustered=True, leaf_size=200, batch_size=200, degree=4)
        X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
        f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
        sp = ShardedPlan(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
        out = torch.full((c.n_orb, c.N), float("nan"), dtype=torch.float64, device="cuda")
        sp.convolve(c.k, f, c.n_orb, out)
        plan = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
        ref = torch.empty_like(out)
        B.bltc_convolve(plan, c.k, f, c.n_orb, ref)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
        got = sp.convolve(c.k, f, c.n_orb)            # `out` left out: the plain path allocates the result itself
        torch.cuda.synchronize()
        assert got.data_ptr() != out.data_ptr() and torch.equal(got, ref)
        sp.destroy(); B.bltc_destroy(plan)
    finally:
        dist.destroy_process_group()


def _cuda_world2_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2003_01833_b200.multi_gpu import ShardExchange
        torch.cuda.set_device(0)                                  # both ranks share the one GPU there is
        c = I.random_cloud(6000, n_orb=3, seed=22, clustered=True, leaf_size=200, batch_size=200, degree=4)
        X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
        f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
        plan = B.bltc_create_sharded(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, rank, world)
        st = B.bltc_get_stats(plan)
        idx = B.bltc_get_shard_targets(plan)
        out = torch.full((c.n_orb, c.N), float("nan"), dtype=torch.float64, device="cuda")
        B.bltc_convolve(plan, c.k, f, c.n_orb, out, True)         # this rank's CUDA kernels, its slice of the batches only
        torch.cuda.synchronize()
        mine = out.cpu()
        written = ~torch.isnan(mine[0])
        only_own = bool(np.array_equal(np.sort(torch.nonzero(written)[:, 0].numpy()), np.sort(idx)))
        ex = ShardExchange(idx, c.N, "cpu")                       # the exchange: values over gloo, no GPU rank waits on another
        ex.all_gather_out(mine)
        evals = torch.tensor([st["shard_far_evals"] + st["shard_near_evals"], int(only_own), len(idx)], dtype=torch.int64)
        dist.all_reduce(evals, op=dist.ReduceOp.SUM)
        if rank == 0:
            full = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
            ref = torch.empty_like(out)
            B.bltc_convolve(full, c.k, f, c.n_orb, ref, True)
            torch.cuda.synchronize()
            fs = B.bltc_get_stats(full)
            q.put((mine.numpy(), ref.cpu().numpy(), [int(v) for v in evals], fs["far_evals"] + fs["near_evals"]))
            B.bltc_destroy(full)
        B.bltc_destroy(plan)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_gpu_world2_sharded_cuda_path_two_processes_on_one_gpu(oracle_mod):
    """The N > 1 path with the CUDA kernels in it, as far as one GPU allows: two processes, both on cuda:0, each builds
    its bltc_create_sharded(rank, 2) plan and runs bltc_convolve for its slice; the slices are exchanged as CPU tensors
    by ShardExchange over gloo (no kernel of one rank waits on the other's).  The assembled result must be BITWISE the
    unsharded GPU result (the slice's work items and summation order are the full plan's) and within 1e-12 of the oracle."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_cuda_world2_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got, ref, sums, full_evals = q.get(timeout=600)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    c = I.random_cloud(6000, n_orb=3, seed=22, clustered=True, leaf_size=200, batch_size=200, degree=4)
    assert sums[0] == full_evals and sums[1] == 2 and sums[2] == c.N     # the slices partition work and targets
    assert not np.isnan(got).any()
    np.testing.assert_array_equal(got, ref)
    op = oracle_mod.OraclePlan((c.x, c.y, c.z), c.theta, c.degree, c.leaf_size, c.batch_size)
    want = op.evaluate(c.w, c.f, c.k)
    err = max(np.linalg.norm(got[o] - want[o]) / np.linalg.norm(want[o]) for o in range(c.n_orb))
    assert err <= 1e-12, err


@pytest.mark.gpu
def test_gpu_scatter_epilogue_writes_every_destination():
    # bltc_convolve_scatter: the epilogue stores each result into `out` and into every peer buffer (here: more buffers
    # on the same GPU stand in for the peers' NVLink-mapped ones); a sharded plan still writes only its own targets
    import torch
    c = _cloud()
    X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
    f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
    full = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
    ref = torch.empty((c.n_orb, c.N), dtype=torch.float64, device="cuda")
    B.bltc_convolve(full, c.k, f, c.n_orb, ref, True)
    outs = [torch.full((c.n_orb, c.N), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    for r in range(3):                                   # "rank r" scatters its slice into all three buffers
        plan = B.bltc_create_sharded(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, r, 3)
        peers = [outs[q] for q in range(3) if q != r]
        B.bltc_convolve_scatter(plan, c.k, f, c.n_orb, outs[r], peers, True)
        torch.cuda.synchronize()
        B.bltc_destroy(plan)
    for o in outs:
        assert torch.equal(o, ref)                       # every "rank" holds the whole result, bitwise the unsharded one
    cref = torch.empty_like(ref)
    B.bltc_convolve_coulomb(full, f, c.n_orb, cref, True, 0.2)
    co = [torch.empty_like(ref) for _ in range(2)]
    B.bltc_convolve_coulomb_scatter(full, f, c.n_orb, co[0], [co[1].data_ptr()], True, 0.2)      # raw addresses work too
    torch.cuda.synchronize()
    assert torch.equal(co[0], cref) and torch.equal(co[1], cref)
    with pytest.raises(B.BltcError):
        B.bltc_convolve_scatter(full, c.k, f, c.n_orb, outs[0], [outs[1]] * 16, True)            # at most 15 peers
    B.bltc_destroy(full)


@pytest.mark.gpu
def test_gpu_sharded_plan_fused_scatter_over_symmetric_memory_world1():
    # the symmetric-memory plumbing of ShardedPlan(fused_scatter=True); a 1-rank group is all one GPU allows
    import torch
    import torch.distributed as dist
    from paper_2003_01833_b200.multi_gpu import ShardedPlan
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(_free_port())
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        c = I.random_cloud(6000, n_orb=3, seed=24, clustered=True, leaf_size=200, batch_size=200, degree=4)
        X = torch.from_numpy(c.coords()).cuda(); w = torch.from_numpy(c.w).cuda()
        f = torch.from_numpy(np.ascontiguousarray(c.f)).cuda()
        try:
            sp = ShardedPlan(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size, fused_scatter=True)
            got = sp.convolve(c.k, f, c.n_orb)
            got2 = sp.convolve(c.k, f, c.n_orb, out=torch.empty((c.n_orb, c.N), dtype=torch.float64, device="cuda"))
        except (RuntimeError, NotImplementedError) as e:         # symmetric memory not available on this box
            pytest.skip(f"torch symmetric memory unavailable: {e}")
        plan = B.bltc_create(None, X, w, c.N, c.theta, c.degree, c.batch_size, c.leaf_size)
        ref = torch.empty((c.n_orb, c.N), dtype=torch.float64, device="cuda")
        B.bltc_convolve(plan, c.k, f, c.n_orb, ref)
        torch.cuda.synchronize()
        assert torch.equal(got, ref) and torch.equal(got2, ref)
        sp.destroy(); B.bltc_destroy(plan)
    finally:
        dist.destroy_process_group()
