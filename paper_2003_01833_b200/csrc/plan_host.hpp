// plan_host.hpp -- host-side plan of the barycentric Lagrange treecode (built once per mesh).
//
// Step a0 of the hot path: source-cluster tree, target batches, per-batch
// MAC interaction lists (Algorithm 3), the per-cluster
// Chebyshev grids (Eq. (37)), and the B200 work decomposition (tiles, list
// segments, cost-sorted work items) that the CUDA kernels consume.  Pure C++, no CUDA.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace bltc {

// Warps of a pair-kernel CTA (near / far / direct).  A CTA is laid out as G target groups x S source-split ways,
// G * S = kPairWarps, G a power of two <= kTileGroupsMax -- the host cuts batches into tiles accordingly.
#ifndef BLTC_PAIR_WARPS
#define BLTC_PAIR_WARPS 8
#endif
constexpr int kPairWarps = BLTC_PAIR_WARPS;
// Targets per thread of a full pair-kernel tile (register tile R x OT): a target group is 32 * R consecutive targets.
#ifndef BLTC_TARGETS_PER_THREAD
#define BLTC_TARGETS_PER_THREAD 2
#endif
constexpr int kTargetsPerThread = BLTC_TARGETS_PER_THREAD;
static_assert(kTargetsPerThread == 1 || kTargetsPerThread == 2 || kTargetsPerThread == 4, "R is 1, 2 or 4");
constexpr int kTileGroupsMax = (kPairWarps % 8 == 0) ? 8 : 4;
static_assert(kPairWarps % kTileGroupsMax == 0, "source-split ways must be an integer");

struct Cluster {
    int64_t begin = 0, end = 0;      // particle range in tree order
    double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};   // minimal bounding box
    int parent = -1, level = 0, nchild = 0;
    int child[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

struct Tree {
    std::vector<Cluster> cl;         // DFS pre-order, cl[0] = root
    std::vector<int64_t> perm;       // tree order -> caller index
    std::vector<int> leaves;         // leaf ids in DFS order
};

// One CTA's work: a tile of targets (2^gshift groups of 32 R consecutive targets, R per thread -- or ONE narrower group
// of 32 (R >> rshift), so that a ragged batch wastes at most 31 lanes)
// against one segment of its batch's far or near list.
struct WorkItem {
    int32_t tgt_begin;               // first target (target tree order)
    int32_t tgt_count;               // targets in the tile
    int32_t gshift;                  // log2(number of target groups in the tile), 0..3
    int32_t list_begin, list_end;    // slice of near_ranges / far_slots
    int32_t rshift;                  // the tile runs R >> rshift targets per thread: 0 = full groups of 32 R targets;
                                     // > 0: one narrower group holding the tail of a ragged batch
    int64_t partial_off;             // where this (batch, segment) slice starts in the partial buffer
};

// source range in tree order; flags & kRangeMayCoincide: a source of the range may coincide with a
// target of the batch (their bounding boxes intersect), so the kernel must test r == 0 (reading R3)
struct Range { int32_t begin, end, flags; };
constexpr int32_t kRangeMayCoincide = 1;

// Upward pass work: one CTA computes the proxy charges of the particle chunk [begin, end) of a slot's
// cluster.  dst < 0: the slot has a single chunk, the CTA writes the slot's charges directly;
// dst >= 0: it writes chunk-partial charges number dst, summed afterwards in chunk order (UpReduce).
struct UpItem { int32_t slot, begin, end, dst; };
struct UpReduce { int32_t slot, first, count; };
// Child -> parent upward pass (upward_children): one CTA interpolates the proxy charges of a parent's children onto the
// parent's grid (reading R23).  Items are grouped by tree level, deepest first: a level needs the one below.
struct C2PItem { int32_t parent, nchild; int32_t child[8]; };   // proxy slot ids

struct HostPlan {
    // parameters
    int64_t N = 0, M = 0;
    bool same_points = true;         // targets are the sources
    bool shared_order = true;        // batches are the source leaves (N_B == N_L, same points)
    double theta = 0;
    int degree = 0, P = 0, leaf_size = 0, batch_size = 0;

    Tree src, tgt;                   // tgt used only when !shared_order
    const std::vector<int64_t>& tgt_perm() const { return shared_order ? src.perm : tgt.perm; }

    // batches (target tree order ranges + boxes)
    std::vector<int64_t> b_begin, b_end;
    std::vector<double> b_lo, b_hi;  // [nb][3]

    // interaction lists, CSR over batches, cluster ids in traversal order (for export/stats)
    std::vector<int64_t> far_ptr, near_ptr;
    std::vector<int32_t> far_idx, near_idx;
    int64_t far_evals = 0, near_evals = 0;
    int lists_b0 = 0, lists_b1 = 0;  // far_idx / near_idx are filled for the batches [lists_b0, lists_b1) (the device builder
                                     // of a sharded plan traverses only its own batches; far_ptr / near_ptr are always complete)

    // clusters that carry proxy charges ("slots")
    std::vector<int32_t> slot_of_cluster;      // -1 if never approximated
    std::vector<int32_t> cluster_of_slot;
    std::vector<double> slot_nodes;            // [nslot][3][degree+1], Eq. (37)
    int64_t upward_pairs = 0;                  // particle-cluster pairs of the upward pass (slots computed from particles)
    bool upward_children = false;              // proxy charges of internal clusters from their children's (reading R23)
    std::vector<C2PItem> c2p_items;            // by level, deepest first
    std::vector<int32_t> c2p_level_ptr;        // [nlevels + 1] into c2p_items
    std::vector<UpItem> up_items;              // chunked upward-pass work, largest first
    std::vector<UpReduce> up_reduce;           // slots whose chunks must be summed
    int64_t up_partial_chunks = 0;             // chunk-partial buffers needed (each P * OT doubles)

    // device work decomposition
    std::vector<Range> near_ranges;            // merged + cut source ranges, per (batch, segment)
    std::vector<int32_t> far_slots;            // proxy slot ids, per (batch, segment)
    std::vector<int32_t> b_nseg_far, b_nseg_near;
    std::vector<int64_t> b_partial_base;       // per batch
    int64_t partial_len = 0;                   // doubles per orbital
    std::vector<WorkItem> far_items, near_items;   // target groups of 64 (2 targets per thread)

    // multi-GPU batch sharding: this plan carries the device work of the
    // batches [shard_b0, shard_b1) only -- a contiguous slice of the batch list holding ~1/world of the
    // far + near kernel evaluations.  Tree, batches and lists above are always the whole problem's.
    int shard_rank = 0, shard_world = 1;
    int shard_b0 = 0, shard_b1 = 0;
    int64_t shard_far_evals = 0, shard_near_evals = 0;

    double max_dist = 0;                       // upper bound of |target - source| over all pairs (root boxes)
    double build_ms = 0;
    double stage_ms[4] = {0, 0, 0, 0};         // tree(s) + batches, MAC traversal, (unused), proxy slots + work decomposition
    bool built_on_device = false;              // tree and lists came from plan_device.cu
};

// Throws std::invalid_argument / std::bad_alloc.  targets == nullptr: targets are the sources.
// coords: SoA double[3][n].
// shard_rank / shard_world: see HostPlan::shard_b0 (world = 1: the whole problem).
void build_host_plan(HostPlan& p, const double* targets, const double* sources, int64_t N,
                     double theta, int degree, int batch_size, int leaf_size, int sm_count,
                     int shard_rank = 0, int shard_world = 1, bool upward_children = false);

// The stages build_host_plan is made of; the device builder (plan_device.cu) replaces the tree and the list
// traversal by kernels and shares the rest.
void plan_begin(HostPlan& p, int64_t N, bool same_points, double theta, int degree, int batch_size, int leaf_size,
                bool upward_children = false);
void build_tree(Tree& t, const double* x, const double* y, const double* z, int64_t n, int64_t max_leaf);   // host
void plan_set_batches(HostPlan& p);                       // batches = leaves of the batch tree; max_dist
void plan_lists_host(HostPlan& p, std::vector<int64_t>& b_far_evals, std::vector<int64_t>& b_near_evals);
void plan_set_shard(HostPlan& p, const std::vector<int64_t>& b_far_evals, const std::vector<int64_t>& b_near_evals,
                    int shard_rank, int shard_world);
void plan_finish(HostPlan& p, int sm_count);              // slots, Chebyshev grids, upward items, work decomposition

// Cut nb batches with the given costs into `world` contiguous slices of nearly equal cost:
// slice r = [cut[r], cut[r+1]), cut[0] = 0, cut[world] = nb; every cut is the first batch whose
// cost prefix reaches r/world of the total (deterministic, identical on every rank).
std::vector<int> shard_cuts(const std::vector<int64_t>& batch_cost, int world);

}  // namespace bltc
