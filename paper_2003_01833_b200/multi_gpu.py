"""Batch-sharded convolution over several ranks.

One process per GPU.  Every rank builds the same tree and lists and owns a contiguous slice of the target batches
(`bltc_create_sharded`); the convolution itself needs no communication.  What does need one exchange is the NEXT
Green-Iteration step: its source field f = V_eff * psi_new is needed at ALL points on every rank (the sources are
replicated), so after the convolution the ranks all-gather their slices of `out` -- O * N * 8 bytes in total per
step, over NCCL (NVLink 5 / NVSwitch) for CUDA tensors, or gloo for CPU tensors (tests).

`ShardedPlan(fused_scatter=True)` fuses that exchange into the convolution's epilogue kernel: results are stored
straight into every rank's buffer over NVLink peer memory (torch.distributed symmetric memory provides the mappings
and the barriers), so no separate collective runs.

This module is plumbing only (torch.distributed + index bookkeeping); all arithmetic stays in the CUDA kernels.
"""
from __future__ import annotations

import numpy as np

from . import binding as B


class ShardExchange:
    """All-gather of per-rank slices of out[n_orb][N] given each rank's target indices (caller order).

    Built once per plan: the index lists of all ranks are exchanged here, so a step moves values only.
    """

    def __init__(self, shard_idx, N, device, group=None):
        import torch
        import torch.distributed as dist
        self.dist, self.torch, self.group = dist, torch, group
        self.world = dist.get_world_size(group)
        self.rank = dist.get_rank(group)
        self.N = int(N)
        idx = torch.as_tensor(np.ascontiguousarray(shard_idx), dtype=torch.int64, device=device)
        counts = torch.zeros(self.world, dtype=torch.int64, device=device)
        counts[self.rank] = idx.numel()
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
        self.counts = [int(v) for v in counts.cpu()]
        if sum(self.counts) != self.N:
            raise ValueError(f"shards cover {sum(self.counts)} of {self.N} targets")
        self.cmax = max(max(self.counts), 1)
        pad = torch.zeros(self.cmax, dtype=torch.int64, device=device)       # padding reads column 0: harmless
        pad[: idx.numel()] = idx
        gathered = torch.empty(self.world * self.cmax, dtype=torch.int64, device=device)
        dist.all_gather_into_tensor(gathered, pad, group=group)              # flat: rank r's block is [r*cmax, ...)
        gathered = gathered.view(self.world, self.cmax)
        self.idx = [gathered[r, : self.counts[r]] for r in range(self.world)]      # every rank's targets
        allidx = torch.cat(self.idx)
        if int(torch.unique(allidx).numel()) != self.N:
            raise ValueError("shards overlap")
        self.local_idx = idx
        self._send_idx = pad
        self._maps = {}                      # n_orb -> (positions in the gathered buffer, positions in out)

    def _map(self, n_orb, device):
        m = self._maps.get(n_orb)
        if m is None:
            torch = self.torch
            src, dst = [], []
            for r in range(self.world):
                if r == self.rank or not self.counts[r]:
                    continue
                j = torch.arange(self.counts[r], dtype=torch.int64, device=device)
                for o in range(n_orb):
                    src.append((r * n_orb + o) * self.cmax + j)
                    dst.append(o * self.N + self.idx[r])
            e = torch.empty(0, dtype=torch.int64, device=device)
            m = (torch.cat(src) if src else e, torch.cat(dst) if dst else e)
            self._maps[n_orb] = m
        return m

    def bytes_per_step(self, n_orb):
        """Bytes each rank receives per exchange: world x n_orb x cmax doubles (its own slice included)."""
        return self.world * n_orb * self.cmax * 8

    def all_gather_out(self, out):
        """out: contiguous [n_orb][N] tensor whose columns `local_idx` are valid on this rank; on return every
        column is.  One gather kernel, ONE collective (all_gather_into_tensor of the ranks' padded slices), one
        scatter kernel; the index maps are built once per n_orb."""
        torch, dist = self.torch, self.dist
        n_orb = out.shape[0]
        send = out.index_select(1, self._send_idx).view(-1)                     # [n_orb][cmax], flat
        recv = torch.empty(self.world * n_orb * self.cmax, dtype=out.dtype, device=out.device)
        dist.all_gather_into_tensor(recv, send, group=self.group)               # [world][n_orb][cmax], flat
        src, dst = self._map(n_orb, out.device)
        if src.numel():
            out.view(-1).index_copy_(0, dst, recv.index_select(0, src))
        return out


class ShardedPlan:
    """bltc_create_sharded + the exchange: `convolve` leaves the full out[n_orb][N] on every rank.

    fused_scatter=False: convolution, then ShardExchange (gather kernel + ONE NCCL all-gather + scatter kernel).
    fused_scatter=True:  the exchange is fused into the convolution's epilogue (bltc_convolve_scatter): every rank's
        result buffer lives in torch.distributed symmetric memory, the epilogue kernel stores each value into its own
        buffer and, over NVLink peer mappings, into every other rank's; a symmetric-memory barrier before (the peers
        have consumed the previous result) and after (all stores have landed) replaces the collective.  The result is
        the symmetric buffer itself (returned; copied into `out` if one is given).
    """

    def __init__(self, targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size, group=None,
                 fused_scatter=False):
        import torch.distributed as dist
        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.N = int(N)
        self.device = sources.device
        self.plan = B.bltc_create_sharded(targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size,
                                          self.rank, self.world)
        self.stats = B.bltc_get_stats(self.plan)
        self.fused = bool(fused_scatter)
        self._symm = {}                      # n_orb -> (tensor, handle, peer pointers)
        self.exchange = None if self.fused else ShardExchange(B.bltc_get_shard_targets(self.plan), N, sources.device, group)

    def _symm_out(self, n_orb):
        """This rank's [n_orb][N] result buffer in symmetric memory and the other ranks' addresses of theirs
        (collective on first use per n_orb)."""
        if n_orb not in self._symm:
            import torch
            import torch.distributed as dist
            import torch.distributed._symmetric_memory as symm_mem
            t = symm_mem.empty((n_orb, self.N), dtype=torch.float64, device=self.device)
            hdl = symm_mem.rendezvous(t, self.group if self.group is not None else dist.group.WORLD)
            peers = [int(p) for r, p in enumerate(hdl.buffer_ptrs) if r != self.rank]
            self._symm[n_orb] = (t, hdl, peers)
        return self._symm[n_orb]

    def _run(self, call_plain, call_scatter, n_orb, out, gather):
        if not self.fused:
            if out is None:                  # `out` is optional in both modes: the plain path needs a buffer of its own
                import torch
                out = torch.empty((n_orb, self.N), dtype=torch.float64, device=self.device)
            call_plain(out)
            return self.exchange.all_gather_out(out) if gather else out
        t, hdl, peers = self._symm_out(n_orb)
        hdl.barrier()                        # every rank has consumed the previous result
        call_scatter(t, peers if gather else [])
        hdl.barrier()                        # every rank's stores have landed
        if out is not None and out.data_ptr() != t.data_ptr():
            out.copy_(t)
            return out
        return t

    def convolve(self, k, f, n_orb, out=None, subtract_singularity=True, gather=True):
        return self._run(lambda o: B.bltc_convolve(self.plan, k, f, n_orb, o, subtract_singularity),
                         lambda t, peers: B.bltc_convolve_scatter(self.plan, k, f, n_orb, t, peers, subtract_singularity),
                         n_orb, out, gather)

    def convolve_coulomb(self, f, n_f, out=None, subtract_singularity=True, alpha=1.0, gather=True):
        return self._run(lambda o: B.bltc_convolve_coulomb(self.plan, f, n_f, o, subtract_singularity, alpha),
                         lambda t, peers: B.bltc_convolve_coulomb_scatter(self.plan, f, n_f, t, peers,
                                                                          subtract_singularity, alpha),
                         n_f, out, gather)

    def destroy(self):
        B.bltc_destroy(self.plan)
        self._symm.clear()
