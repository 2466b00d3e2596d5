/*
 * bltc.h -- C ABI of libbltc: the discrete modified-Helmholtz (Yukawa) convolution of
 * treecode-accelerated Green Iteration (arXiv 2003.01833) on one NVIDIA B200 (sm_100a).
 *
 * What is computed, for every orbital o and target point x_i (Eq. (18) discretised
 * as PAPER.md:371 Eq. (32), with the singularity subtraction of PAPER.md:204-208 Eq. (20)-(21)):
 *
 *   subtract_singularity = 1:
 *     out[o][i] = -2 * ( sum_{j : r_ij != 0} G_k(r_ij) w_j (f[o][j] - f[o][i])  +  f[o][i] / k_o^2 )
 *   subtract_singularity = 0:
 *     out[o][i] = -2 *   sum_{j : r_ij != 0} G_k(r_ij) w_j  f[o][j]
 *
 *   G_k(r) = exp(-k r) / (4 pi r),   k_o = sqrt(-2 eps_o) > 0,   r_ij = |x_i - y_j|.
 *
 * "The singular r' = r term in the quadrature sums is skipped": a term is skipped
 * iff r_ij == 0 exactly.  direct_convolve evaluates the sum as written (O(M N)); bltc_convolve
 * evaluates it with the barycentric Lagrange treecode of PAPER.md:361-462 (Section 6, Algorithm 3):
 * source-cluster tree, target batches and MAC interaction lists built once per mesh by bltc_create,
 * proxy charges on tensor Chebyshev grids (Eq. (35) right, (37)-(39)), batch-cluster far field
 * (Eq. (35) left) and batch-leaf direct near field (Eq. (34)).
 *
 * Conventions
 *   - All floating point is IEEE double.  Coordinates are SoA: double[3][N] = x-row, y-row, z-row.
 *   - Every data pointer may be a DEVICE pointer or a HOST pointer; the library asks
 *     cudaPointerGetAttributes.  Host buffers are staged through device memory inside the call
 *     (copies are enqueued on `stream`).  k is always a HOST array.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls that
 *     take a stream only ENQUEUE work and return without synchronising, except when `out` is a
 *     host pointer: then the call returns after the stream has been synchronised.
 *   - The library copies what it needs: inputs of bltc_create may be freed after it returns;
 *     f/out of a convolve call must stay valid until the stream has executed the call.
 *   - Return value: 0 on success, a negative bltc_status otherwise; bltc_last_error() gives a
 *     thread-local message.  No exceptions, no exit(); handles are independent and the library keeps no state
 *     between calls other than a stream-ordered memory pool of its own per device (staging buffers of
 *     direct_convolve / bltc_gi_update and the temporaries of bltc_create are reused, the device's default pool is
 *     not touched), the fixed scratch array of bltc_gi_update_noalloc, and the per-thread profiling switch of
 *     direct_convolve.  It reads one environment variable, BLTC_ORBITAL_TILE (see "Diagnostics" below).
 *     A handle must not be used by two threads at once.  Calls on one handle share its scratch (proxy charges,
 *     partial sums, staging); the library orders them itself: a convolve enqueued on another stream than the
 *     previous one first waits (cudaStreamWaitEvent) for that one to finish.
 *   - There is no CPU fallback: every compute entry point fails with BLTC_ECUDA / BLTC_ENODEVICE
 *     if no CUDA device is usable.
 *   - Limits: 1 <= N <= 2e9 (int32 indices), 1 <= interp_degree <= 20, 0 <= theta < 1,
 *     1 <= n_orb, k_o > 0 and k_o * (domain diameter) < 2^30.
 */
#ifndef BLTC_H_
#define BLTC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bltc_plan_s* bltc_handle;   /* opaque, owned by the library */
typedef void* bltc_stream;                 /* cudaStream_t */

typedef enum bltc_status {
    BLTC_OK = 0,
    BLTC_EINVAL = -1,      /* bad argument (message says which) */
    BLTC_ENOMEM = -2,      /* host or device allocation failed */
    BLTC_ECUDA = -3,       /* a CUDA call failed (message carries cudaGetErrorString) */
    BLTC_ENODEVICE = -4    /* handle has no device state (bltc_create_host_plan) */
} bltc_status;

/* Counters of a plan (step a0).  "evals" = kernel evaluations per orbital per convolution. */
typedef struct bltc_stats {
    int64_t n_points;          /* N */
    int64_t n_clusters;        /* source clusters in the tree */
    int64_t n_leaves;          /* leaf clusters */
    int64_t n_batches;         /* target batches */
    int64_t n_far;             /* batch-cluster far interactions, total (Eq. (35)) */
    int64_t n_near;            /* batch-cluster direct interactions, total (Eq. (34)) */
    int64_t far_evals;         /* sum over far interactions of targets * (n+1)^3 */
    int64_t near_evals;        /* sum over near interactions of targets * N_S */
    int64_t n_proxy_clusters;  /* clusters that carry proxy charges */
    int64_t upward_pairs;      /* particle-cluster pairs of the upward pass (clusters whose charges come from particles) */
    int64_t n_far_items;       /* CTAs launched by the far-field kernel (R = 2 tiling) */
    int64_t n_near_items;      /* CTAs launched by the near-field kernel (R = 2 tiling) */
    int64_t partial_len;       /* doubles of partial-sum scratch per orbital */
    int64_t n_upward_items;    /* CTAs launched by the upward pass (cluster chunks) */
    int64_t n_upward_reduce;   /* clusters whose chunk-partial proxy charges are summed by a second kernel */
    int64_t launches_per_group;/* kernels one bltc_convolve launches per orbital tile (of <= 7 orbitals, bltc_orbital_tiles) */
    int32_t shared_batches;    /* 1: batches are the source leaves */
    int32_t interp_degree;
    double  theta;
    double  build_ms;          /* wall-clock of tree + lists + work decomposition (device builder: kernels included) */
    double  upload_ms;         /* host wall-clock of device upload + f-independent proxy weights */
    /* batch sharding (bltc_create_sharded); an unsharded plan reports rank 0 of 1 and all batches */
    int32_t shard_rank, shard_world;
    int64_t shard_batch_begin; /* this plan computes the batches [begin, end) ... */
    int64_t shard_batch_end;
    int64_t shard_targets;     /* ... = this many targets (a contiguous range in target tree order) */
    int64_t shard_far_evals;   /* kernel evaluations per orbital of this plan's batches */
    int64_t shard_near_evals;
    /* step a0 timing (host wall-clock, ms; the kernels of the device builder are synchronised inside) */
    double  tree_ms;           /* cluster tree(s) + batches */
    double  lists_ms;          /* MAC traversal of Algorithm 3 (decisions) */
    double  decomp_ms;         /* proxy slots, Chebyshev grids, work decomposition */
    double  create_ms;         /* all of bltc_create, uploads and the proxy weights of w included */
    int32_t built_on_device;   /* 1: tree and lists were built by kernels (BLTC_BUILDER_DEVICE) */
    int32_t upward_from_children; /* 1: BLTC_UPWARD_FROM_CHILDREN */
} bltc_stats;

/* Phases of one bltc_convolve, for bltc_get_phase_ms (device times, CUDA events on `stream`). */
enum { BLTC_PHASE_GATHER = 0, BLTC_PHASE_UPWARD = 1, BLTC_PHASE_FAR = 2, BLTC_PHASE_NEAR = 3,
       BLTC_PHASE_EPILOGUE = 4, BLTC_NUM_PHASES = 5 };

/*
 * bltc_create: Algorithm 3 line 1 plus everything that does not depend on f or k.
 *   targets  double[3][N] SoA, or NULL / == sources when the targets are the sources (the TAGI case:
 *            "the target particles and source particles correspond to the same set").
 *   sources  double[3][N] SoA.        weights  double[N] quadrature weights w_j.
 *   theta, interp_degree: MAC parameter and degree n of Eq. (36).
 *   batch_size N_B, leaf_size N_L: PAPER.md:378,428.  If N_B == N_L and targets are the sources the
 *   batches are the leaf clusters.
 * Builds the tree, batches and lists ON THE DEVICE (SURVEY.md 8(f) NEXT-4a; the precompute stage is
 * what limits the paper's multi-GPU scaling): per tree level exact min/max boxes, the split decisions of DESIGN.md
 * readings R4-R5, one stable radix sort of (segment, child code) keys; one thread per batch walks the tree for the
 * MAC lists.  The plan is identical -- cluster for cluster, list entry for list entry -- to the host builder's and
 * to the CPU oracle's.  Then uploads the work decomposition and computes the proxy weights of w (what_k).
 * Inputs on the device are used in place (no copy to the host).  Synchronous.  *h is set only on success.
 */
int bltc_create(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                int64_t N, double theta, int interp_degree, int batch_size, int leaf_size);

/*
 * Multi-GPU batch sharding (the paper's multi-GPU split, PAPER.md:494-500:
 * "the compute stage has close to ideal scaling").  Target batches are independent given the sources and the
 * proxy charges, so rank r of `world` builds the SAME tree, batches and lists (the whole problem's: every rank
 * holds all sources) and keeps the device work of a contiguous slice of the batch list that carries ~1/world of
 * the far + near kernel evaluations; proxy charges are computed (redundantly, ~0.5 % of the work) only for the
 * clusters its own far lists use.  No data-path collective is needed: bltc_convolve / bltc_convolve_coulomb on
 * such a plan write out[o][i] ONLY for the targets i of the plan's batches and leave every other element of
 * `out` untouched; bltc_get_shard_targets lists those i (caller's point indices, `shard_targets` of them, in
 * target tree order).  Slices of different ranks are disjoint and cover all targets.  world = 1 is bltc_create.
 */
int bltc_create_sharded(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                        int64_t N, double theta, int interp_degree, int batch_size, int leaf_size,
                        int rank, int world);
/* The same with the builder named: BLTC_BUILDER_DEVICE (what bltc_create / bltc_create_sharded use) or
 * BLTC_BUILDER_HOST (tree, lists and decomposition by the threaded host code of plan_host.cpp -- the setup
 * alternative; also taken automatically for N >= 2^28).  Both give the same plan. */
enum { BLTC_BUILDER_DEVICE = 0, BLTC_BUILDER_HOST = 1,
       /* OR-able options for the upward pass (readings R9 / R23).
        * FROM_CHILDREN: the proxy charges of LEAF clusters come from their particles (Eq. (35) right) and those of
        *   every internal cluster from its children's proxy charges, re-interpolated onto its own grid, level by level,
        *   deepest first.  In exact arithmetic the charges are the SAME as from the particles (the Lagrange basis of the
        *   parent is a polynomial of degree n, which the child's grid reproduces exactly); measured difference of the
        *   convolution <= 2e-15; the work is O(N (n+1)^3) instead of O(N (n+1)^3 depth) (configs[3]: 3.7x faster).
        *   This is what bltc_create / bltc_create_sharded / bltc_create_host_plan use.
        * FROM_PARTICLES: every cluster from its own particles, the literal reading of Alg. 3 line 2 (R9).
        * Neither bit: the library default (FROM_CHILDREN). */
       BLTC_UPWARD_FROM_CHILDREN = 2, BLTC_UPWARD_FROM_PARTICLES = 4 };
int bltc_create_with_builder(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                             int64_t N, double theta, int interp_degree, int batch_size, int leaf_size,
                             int rank, int world, int builder);
int bltc_create_host_plan_sharded(bltc_handle* h, const double* targets, const double* sources,
                                  const double* weights, int64_t N, double theta, int interp_degree,
                                  int batch_size, int leaf_size, int rank, int world);
int bltc_get_shard_targets(bltc_handle h, int64_t* idx /* HOST int64[shard_targets] */);

/* Same plan, host part only (no CUDA call is made): for structural inspection through
 * bltc_get_stats / bltc_export_plan.  weights may be NULL.  bltc_convolve on such a handle
 * returns BLTC_ENODEVICE.  coordinates must be HOST pointers. */
int bltc_create_host_plan(bltc_handle* h, const double* targets, const double* sources,
                          const double* weights, int64_t N, double theta, int interp_degree,
                          int batch_size, int leaf_size);

/*
 * bltc_convolve: Algorithm 3 lines 2-3 + Eq. (18),(20),(21), all orbitals.
 *   k    HOST double[n_orb], k_o > 0 (one per orbital: each wavefunction has its own eps).
 *   f    double[n_orb][N], caller's original point order: f = V_eff * psi at the quadrature points.
 *   out  double[n_orb][N], caller's original point order.
 *   subtract_singularity = 1 requires that the plan's targets are its sources.
 * Steps (all on `stream`): gather to tree order; upward pass (proxy charges fhat_k of f*w: leaves from particles,
 * parents from their children unless the plan was created with BLTC_UPWARD_FROM_PARTICLES);
 * far-field kernel; near-field kernel; epilogue (-2 (far + near + f_i/k^2), scatter).
 */
int bltc_convolve(bltc_handle h, const double* k, const double* f, int n_orb, double* out,
                  int subtract_singularity, bltc_stream stream);

/*
 * bltc_convolve_scatter / bltc_convolve_coulomb_scatter: the same convolution, with the exchange of a batch-sharded
 * run fused into the kernel that produces the result ("outputs stay sharded or one all-gather of
 * out").  The epilogue stores every out[o][i] of this plan's targets into `out` AND into each of the n_peers <= 15
 * buffers peer_outs[r] (HOST array of DEVICE pointers, each double[n_orb][N] in the caller's point order): the other
 * ranks' `out` buffers, peer-mapped over NVLink (cudaIpc / CUDA symmetric memory; torch.distributed's symmetric
 * memory gives the pointers, paper_2003_01833_b200/multi_gpu.py).  When every rank has run its call and the ranks have
 * synchronised (a barrier on the symmetric memory), each rank's `out` holds the whole result: no separate gather,
 * collective or scatter kernel.  All buffers must be device memory; n_peers = 0 is bltc_convolve.
 */
int bltc_convolve_scatter(bltc_handle h, const double* k, const double* f, int n_orb, double* out,
                          double* const* peer_outs, int n_peers, int subtract_singularity, bltc_stream stream);
int bltc_convolve_coulomb_scatter(bltc_handle h, const double* f, int n_f, double* out, double* const* peer_outs,
                                  int n_peers, int subtract_singularity, double alpha, bltc_stream stream);

/*
 * direct_convolve: the definition, O(M N), no plan (Eq. (32); the "ds" column of
 * PAPER.md:482-490 Table 4).  M targets against N sources.
 *   targets double[3][M], f_targets double[n_orb][M] (may be NULL iff subtract_singularity == 0),
 *   sources double[3][N], weights double[N], f_sources double[n_orb][N], k HOST double[n_orb],
 *   out double[n_orb][M].
 * The call synchronises `stream` once before the pair kernel is enqueued: the bounding boxes of target and
 * source chunks are read back to choose the kernel variant (exp underflow guard only if k_max x the largest
 * distance can reach 700).  Every pair goes through the r == 0 test: the kernel runs the one loop that skips
 * coincident points everywhere (it costs no FP64 instruction; a second loop without it was slower).  Its
 * profiling switch (bltc_direct_set_profiling) is per calling thread.
 */
int direct_convolve(const double* targets, const double* f_targets, int64_t M,
                    const double* sources, const double* weights, const double* f_sources, int64_t N,
                    const double* k, int n_orb, double* out, int subtract_singularity,
                    bltc_stream stream);

/*
 * the Hartree potential (Eq. (19)) through the same plan: Coulomb kernel
 * 1/r with the Gaussian singularity subtraction of PAPER.md:220-224 Eq. (23)-(24) ("alpha = 1 a.u.",
 * PAPER.md:229).  This is the convolution the paper times in Table 4 and Fig. 11.
 *
 *   subtract_singularity = 1:
 *     out[o][i] = sum_{j : r_ij != 0} (f[o][j] - f[o][i] e^{-r_ij^2/alpha^2}) w_j / r_ij  +  2 pi alpha^2 f[o][i]
 *   subtract_singularity = 0:
 *     out[o][i] = sum_{j : r_ij != 0} f[o][j] w_j / r_ij                      (alpha ignored)
 *
 * No 1/(4 pi) and no -2: the kernel of Eq. (19) as printed.  The treecode approximates the first integrand of
 * Eq. (23) as two interpolated convolutions (reading R21): far field
 *     sum_k [ fhat_k - f_i what_k e^{-|x_i - s_k|^2/alpha^2} ] / |x_i - s_k|.
 * f, out: double[n_f][N] in the caller's point order (n_f densities share every kernel evaluation);
 * pointers, stream and error conventions as bltc_convolve / direct_convolve.  alpha > 0 (and
 * alpha > 2e-6 x the domain diameter) when subtract_singularity = 1.
 */
int bltc_convolve_coulomb(bltc_handle h, const double* f, int n_f, double* out, int subtract_singularity,
                          double alpha, bltc_stream stream);

int direct_convolve_coulomb(const double* targets, const double* f_targets, int64_t M,
                            const double* sources, const double* weights, const double* f_sources, int64_t N,
                            int n_f, double* out, int subtract_singularity, double alpha, bltc_stream stream);

/*
 * the steps of Green Iteration that follow the convolution (Algorithm 2 lines 4-7,
 * PAPER.md:127-133), fused on the device so that psi never leaves it between two convolutions:
 *   line 4  eps_new = eps_old - <f_old, psi_old - psi_new> / <psi_new, psi_new>     (Eq. (27),
 *           f_old = V_eff psi_old; psi_new as computed by the convolution, before lines 5-6)
 *   line 5  psi_new <- psi_new - sum_{j < n_prev} <psi_new, phi_j> phi_j            (deflation)
 *   line 6  psi_new <- psi_new / sqrt(<psi_new, psi_new>)
 *   line 7  residual = sqrt(<psi_new - psi_old, psi_new - psi_old>)
 * with <a, b> = sum_i w_i a_i b_i (reading R22: quadrature inner product; one classical Gram-Schmidt
 * projection with coefficients taken from the un-projected psi_new, subtracted in the order j = 0, 1, ...).
 *   w, psi_old, f_old  double[N];  psi_new double[N], IN: G(eps_old) psi_old, OUT: the new normalised iterate;
 *   phi double[n_prev][N] orthonormal converged wavefunctions (NULL iff n_prev == 0), 0 <= n_prev <= 4096;
 *   result double[4 + n_prev]: [0] eps_new, [1] delta = eps_old - eps_new, [2] norm before line 6,
 *           [3] residual, [4 + j] = <psi_new, phi_j>.
 * Every pointer may be device or host; with all pointers on the device the call only enqueues 4 kernels on
 * `stream`; a host psi_new or result makes it synchronise.  Sums are two-level in a fixed order (reproducible).
 */
int bltc_gi_update(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                   const double* phi, int n_prev, int64_t N, double eps_old, double* result,
                   bltc_stream stream);

/*
 * bltc_gi_update_noalloc -- bltc_gi_update for callers that must not allocate device memory.
 *
 * Who needs it: callers for whom cudaMalloc / cudaMallocAsync is off limits or bound to fail at the point where
 * they call us.  Examples: a solver embedded in a host application that handed all of HBM to its own arena at
 * start-up, so the driver has nothing left to give; a plug-in whose host forbids driver allocations inside its
 * callbacks; a process that runs under a fixed device-memory budget it may not exceed once initialised; a
 * latency-bound inner loop (one such update follows each of the 188-1246 convolutions of an SCF step,
 * PAPER.md:311,338) that cannot accept the implicit synchronisation or the milliseconds an allocation may cost.
 * bltc_gi_update itself takes the block partial sums of its reductions from the library's stream-ordered pool on
 * every call; this variant keeps them in a fixed array inside the library image instead.
 *
 * Same arithmetic, same kernels, same grid and summation order as bltc_gi_update (Algorithm 2 lines 4-7,
 * PAPER.md:127-133, Eq. (27)): on the same device buffers the two give the same result.  Arguments and
 * the layout of `result` are those of bltc_gi_update, with these differences:
 *   - EVERY buffer (w, psi_old, f_old, psi_new, phi, result) must be device (or managed) memory, owned by the
 *     caller; a host pointer is refused with BLTC_EINVAL, because staging it would need an allocation;
 *   - n_prev <= BLTC_GI_NOALLOC_MAX_PREV (64); a larger n_prev is refused with BLTC_EINVAL and a message naming
 *     the limit (use bltc_gi_update then).  N is not limited beyond bltc_gi_update's [1, 2e9];
 *   - the call makes no cudaMalloc, cudaFree, cudaMallocAsync or other allocating call, ever; it only enqueues
 *     4 kernels on `stream` and returns without synchronising.
 * Cost: the array is 139,264 doubles = 1.06 MiB of device memory on every GPU that loads libbltc.so, held from
 * library load until the process exits, whether or not this entry point is ever called.
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress, with that device current)
 * and the SM count, once, and remembers them.  Make that first call outside any stream capture -- e.g. one warm-up
 * call per device at start-up.
 * Sharing: all calls on one GPU use the SAME array.  It needs no clearing between calls (every slot a call reads
 * was written earlier in that same call), but two calls whose kernels can overlap on the GPU -- different streams,
 * different host threads, without an ordering between them -- race on it and both results are garbage.  Serialise
 * them on one stream or with events.  bltc_gi_update (pool scratch per call) has no such restriction.
 */
#define BLTC_GI_NOALLOC_MAX_PREV 64
int bltc_gi_update_noalloc(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                           const double* phi, int n_prev, int64_t N, double eps_old, double* result,
                           bltc_stream stream);

int bltc_destroy(bltc_handle h);

int bltc_get_stats(bltc_handle h, bltc_stats* s);

/*
 * bltc_export_plan: copy the plan's structure into caller-provided HOST buffers (any may be NULL),
 * for comparison with an independently built tree.  Sizes come from bltc_get_stats.
 *   src_perm[N], tgt_perm[N]        tree order -> caller index (sources, targets)
 *   cl_begin/cl_end[n_clusters]     particle range of each cluster in source tree order (DFS pre-order ids)
 *   cl_lo/cl_hi[n_clusters][3]      minimal bounding boxes
 *   cl_parent/cl_nchild[n_clusters]
 *   b_begin/b_end[n_batches]        target range of each batch in target tree order
 *   far_ptr/near_ptr[n_batches+1], far_idx[n_far], near_idx[n_near]   CSR lists of cluster ids,
 *                                   in the traversal order of Algorithm 3
 */
int bltc_export_plan(bltc_handle h, int64_t* src_perm, int64_t* tgt_perm,
                     int64_t* cl_begin, int64_t* cl_end, double* cl_lo, double* cl_hi,
                     int32_t* cl_parent, int32_t* cl_nchild, int64_t* b_begin, int64_t* b_end,
                     int64_t* far_ptr, int32_t* far_idx, int64_t* near_ptr, int32_t* near_idx);

/*
 * bltc_export_proxy: after a bltc_convolve has completed on the device, copy the Chebyshev grids and
 * proxy charges of the LAST orbital group to HOST buffers (any may be NULL):
 *   proxy_cluster[n_proxy_clusters]          cluster id of each proxy slot
 *   nodes[n_proxy_clusters][3][n+1]          Eq. (37) mapped to the cluster box
 *   what[n_proxy_clusters][(n+1)^3]          proxy weights of w
 *   fhat[n_proxy_clusters][(n+1)^3][ot]      proxy charges of f*w for the `*ot` orbitals of that group; the buffer
 *                                            must hold BLTC_MAX_ORBITAL_TILE orbitals (ot is known only afterwards)
 * Synchronises the device.
 */
int bltc_export_proxy(bltc_handle h, int32_t* proxy_cluster, double* nodes, double* what,
                      double* fhat, int32_t* ot);

/*
 * ---------------------------------------------------------------------------------------------------------------
 * Diagnostics.  Everything from here to bltc_orbital_tiles serves measurement (bench.py, the tuning runs behind
 * DESIGN.md 10) and is not needed to compute a convolution: per-phase and per-kernel timers, the DFMA-rate probes
 * behind the roofline denominator, and the orbital-tile query.
 * One environment variable belongs here too, the only one the library reads: BLTC_ORBITAL_TILE = 1 .. 7 caps the
 * width of the orbital register tile (tuning runs and the tile-width tests); it is read by every bltc_convolve /
 * direct_convolve / bltc_orbital_tiles call, so it may be changed between calls.  Unset, the library chooses the
 * widths itself (bltc_orbital_tiles).  Results at different widths agree to rounding, not bitwise.
 * ---------------------------------------------------------------------------------------------------------------
 */
/* Per-phase device timing.  enable = 1: every later bltc_convolve records CUDA events on its stream
 * around each phase.  bltc_get_phase_ms synchronises on the last recorded event and returns the
 * milliseconds of each phase of the most recent convolve, summed over its orbital groups. */
int bltc_set_profiling(bltc_handle h, int enable);
int bltc_get_phase_ms(bltc_handle h, float ms[BLTC_NUM_PHASES]);

/* Device time (ms, CUDA events) of the pair kernel inside the most recent direct_convolve that was
 * called with profiling on (bltc_direct_set_profiling(1)); synchronises on its last event. */
int bltc_direct_set_profiling(int enable);
int bltc_direct_get_kernel_ms(float* ms);

/*
 * bltc_probe_fp64: measurement utility for the roofline denominator.  Runs a kernel of dependent-
 * chain-free DFMA instructions on every SM for about `iters` x 4096 DFMAs per thread and reports the
 * achieved FP64 rate in TFLOP/s (2 flops per DFMA) in *tflops, timed with CUDA events on `stream`.
 */
int bltc_probe_fp64(int iters, double* tflops, bltc_stream stream);
/* The same with the operand form chosen: form 0 = bltc_probe_fp64 (two distinct register sources per DFMA, the third
 * reused: the pipe's peak); form 1 = three distinct vector-register sources per DFMA, the form of the pair kernels'
 * accumulate -- on sm_100a it holds the FP64 pipe for 3 cycles instead of 2, i.e. reads 2/3 of form 0. */
int bltc_probe_fp64_form(int form, int iters, double* tflops, bltc_stream stream);

/*
 * bltc_orbital_tiles: how a call with n_orb orbitals is cut into register tiles.  The pair kernels evaluate the
 * geometry, rsqrt and r of a (target, source) pair once for all orbitals of a tile (at most 7); the library cuts
 * n_orb into equal-as-possible tiles whose widths minimise a measured per-orbital cost, and runs
 * steps a1-a5 once per tile.  widths: HOST int[capacity]; returns the number of tiles (> capacity: nothing is
 * written past capacity), or BLTC_EINVAL.  Measurement code needs it to count the executed flops of a launch.
 */
#define BLTC_MAX_ORBITAL_TILE 7
int bltc_orbital_tiles(int n_orb, int* widths, int capacity);

const char* bltc_last_error(void);
const char* bltc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BLTC_H_ */
