// kernels.cuh -- launchers of the sm_100a kernels of the BLTC hot path.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#include "plan_host.hpp"

namespace bltc {

constexpr int kMaxOT = 7;          // orbitals processed together in one pass (register tile; 7 measured best)
constexpr int kThreads = 256;      // 8 warps per CTA (upward pass, epilogue, utilities)
constexpr int kPairThreads = 32 * kPairWarps;   // pair kernels (plan_host.hpp)
constexpr int kSrcTile = kPairWarps > 8 ? 1024 : 512;   // sources staged per shared-memory tile (near field / direct)
constexpr int kProxyTile = 1024;   // proxy points staged per shared-memory tile (far field), OT <= 4; 768 above (kernels.cu)

// kTargetsPerThread (plan_host.hpp): targets per thread of a full tile, R = 2 for every orbital-tile width -- one staged
// source / proxy record feeds two pair evaluations (measured on B200: near -8 %, far -2 % at OT = 4 against R = 1)

// per-orbital constants of the tile (kernel parameter -> constant bank):
//   nk = -k_o;  c = -k_o T/ln2 (scaled exponent argument of fp64_math.cuh's exp);  c1, c3: polynomial
//   coefficients of that exp (kept in uniform registers)
// guard (launch_far / launch_near): false only if k r < 700 for every pair of the launch (no exp underflow)
struct KPar { double nk[kMaxOT]; double c[kMaxOT]; double c1, c3; };
KPar make_kpar(const double* k, int ot);   // k: ot values (host)

// kernel of the convolution: Yukawa e^{-k r}/(4 pi r) with the subtraction of Eq. (20)-(21),
// or Coulomb 1/r with the Gaussian subtraction of Eq. (23)-(24)
enum { kYukawa = 0, kCoulomb = 1 };
KPar make_kpar_coulomb(double alpha);      // c[*] = -T/(ln2 alpha^2): scaled exponent of e^{-r^2/alpha^2}

// epilogue constants: out = scale * (far + near) + [subtract] coef[o] * f_i
struct EpiPar { double scale; double coef[kMaxOT]; };
EpiPar make_epipar(const double* k, int ot);     // scale = -2/(4 pi), coef = -2/k_o^2
EpiPar make_epipar_coulomb(double alpha);        // scale = 1, coef = 2 pi alpha^2

// a1: f[o0+o][perm[i]] -> dst[i][ot] (tree order, orbital-interleaved)
cudaError_t launch_gather(const double* f, int64_t stride, int o0, int ot, const int32_t* perm,
                          int64_t n, double* dst, cudaStream_t st);

// pack SoA coordinates (+ weights) into double4 records; perm == nullptr: identity
cudaError_t launch_pack_records(const double* coords, const double* w, const int32_t* perm, int64_t n,
                                double4* rec, cudaStream_t st);

// bounding boxes {lo[3], hi[3]} of the chunks [c*chunk, min(n, (c+1)*chunk)) of SoA coords[3][n] -> out[nchunk][6]
cudaError_t launch_chunk_bbox(const double* coords, int64_t n, int64_t chunk, double* out, cudaStream_t st);

// a2: proxy charges.  ot == 0: what[slot][P] from w;  ot >= 1: fhat[slot][P][ot] from f*w.
// items: chunked work (plan_host.hpp); chunk_out: scratch of up_partial_chunks * P * max(ot,1) doubles
cudaError_t launch_upward(int ot, const UpItem* items, int nitems, const UpReduce* red, int nred,
                          const double* slot_nodes, int degree, const double4* src_rec,
                          const double* fsrc, double* out, double* chunk_out, cudaStream_t st);

// a2, child -> parent variant (HostPlan::upward_children): one launch per tree level, deepest first, after launch_upward
// has filled the slots that are computed from particles.  ot == 0: the proxy weights of w ([slot][P]).
cudaError_t launch_upward_children(int ot, const C2PItem* items, int nitems, const double* slot_nodes, int degree,
                                   double* charges, cudaStream_t st);

// a3: far field
cudaError_t launch_far(int kind, int ot, bool subtract, bool guard, const WorkItem* items, int nitems, const int32_t* far_slots,
                       const double* slot_nodes, const double* what, const double* fhat, int degree,
                       const double4* tgt_rec, const double* ftgt, const KPar& kp, double* partial,
                       int64_t partial_len, cudaStream_t st);

// a4 / a6: near field and brute-force direct sum (same kernel, different work items).  all_zero_safe: every tile runs
// the loop that skips r == 0 (direct_convolve), instead of only the ranges flagged kRangeMayCoincide
cudaError_t launch_near(int kind, int ot, bool subtract, bool guard, bool all_zero_safe, const WorkItem* items, int nitems,
                        const Range* ranges, const double4* src_rec, const double* fsrc, const double4* tgt_rec,
                        const double* ftgt, const KPar& kp, double* partial, int64_t partial_len,
                        cudaStream_t st);

// destinations of the epilogue: the caller's out and, for a sharded plan whose all-gather is fused into the epilogue
// (bltc_convolve_scatter), the peer ranks' out buffers (NVLink peer / symmetric memory); all double[n_orb][stride]
constexpr int kMaxOuts = 16;
struct OutSet { double* p[kMaxOuts]; int n; };

// a5: out[o0+o][perm[i]] = ep.scale (far + near) + [subtract] ep.coef[o] f_i
//     (Yukawa: -2 ( (far + near)/(4 pi) + f_i / k_o^2 );  Coulomb: far + near + 2 pi alpha^2 f_i)
cudaError_t launch_epilogue(int ot, bool subtract, int nbatch, const int32_t* b_begin, const int32_t* b_count,
                            const int64_t* b_partial_base, const int32_t* b_nseg, const double* partial,
                            int64_t partial_len, const double* ftgt, const EpiPar& ep, const int32_t* perm,
                            const OutSet& outs, int64_t stride, int o0, cudaStream_t st);

// roofline probe: DFMA-only kernel; returns elapsed ms and the number of DFMAs executed.  form 0: two register sources
// + a reused one (the pipe's peak); form 1: three distinct vector-register sources per DFMA (3 pipe cycles instead of 2)
cudaError_t launch_fp64_probe(int form, int iters, float* ms, double* dfma_count, cudaStream_t st);

}  // namespace bltc
