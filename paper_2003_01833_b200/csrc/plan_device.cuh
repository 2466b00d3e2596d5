// plan_device.cuh -- device-side construction of the tree and the MAC interaction lists (step a0; see plan_device.cu).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "plan_host.hpp"

namespace bltc {

// Stream-ordered scratch from the library's own per-device memory pool (api.cu): after the first bltc_create the
// two dozen temporaries of a plan build are served from memory the pool kept, not by cudaMalloc / cudaFree.
cudaError_t pool_alloc_async(void** p, size_t bytes, cudaStream_t st);

// Builds the cluster tree of the n points d_coords (device, SoA double[3][n]) with leaves of <= max_leaf points:
// t.cl (DFS pre-order, boxes, ranges, parents, children) and t.leaves on the host, the tree-order -> caller-index
// permutation in d_perm (device int32[n]); t.perm stays empty.  Identical to build_tree() of plan_host.cpp.
// n must be < 2^28.  Synchronises `st`.
cudaError_t build_tree_device(Tree& t, const double* d_coords, int64_t n, int64_t max_leaf, int32_t* d_perm,
                              cudaStream_t st);

// Given p.src.cl and the batches (plan_set_batches): far_ptr / near_ptr and the evaluation counts of ALL batches by a
// counting traversal, the shard cut (plan_set_shard), then far_idx / near_idx of this rank's batches only
// (p.lists_b0, p.lists_b1).  Identical, entry for entry, to plan_lists_host().  Synchronises `st`.
cudaError_t build_lists_device(HostPlan& p, int shard_rank, int shard_world, cudaStream_t st);

}  // namespace bltc
