// kernels.cu -- hand-written FP64 CUDA kernels (sm_100a) of the BLTC Yukawa convolution.
//
//   near_kernel  (a4, a6)  Eq. (34) PAPER.md:389 / Eq. (32) PAPER.md:371 with the subtraction of Eq. (20)
//   far_kernel   (a3)      Eq. (35) left PAPER.md:394 on the tensor Chebyshev grid of Eq. (37)
//   upward_kernel(a2)      Eq. (35) right with the barycentric form Eq. (38)-(39) PAPER.md:416-421
//   gather / pack / epilogue (a1, a5)  Eq. (18),(20),(21) PAPER.md:193-208
//
// Mapping (all three pair kernels): one CTA = kPairWarps (8) warps = one work item = (tile of targets) x (list
// segment).  A thread owns R targets in registers (R*32 per warp = one "group"); a tile has
// 2^gshift <= 8 groups; the 8 warps are laid out as groups x S source-split ways (S = 8 >> gshift),
// so small batches still fill every warp.  Sources / proxy points are staged in shared memory and
// read by broadcast (all lanes of a warp read the same source).  The S partial sums are reduced
// through shared memory in a fixed order and written to a per-(batch, segment) slice of the
// partial buffer; the epilogue adds the slices in a fixed order => bitwise reproducible results.
//
// The bound is the FP64 pipe: per (target, source) pair and orbital tile of OT = 1 ... 7 orbitals the near
// kernel executes 22 + 9 (OT - 1) FP64 instructions and the far kernel (n = 8) 16.4 + 9 (OT - 1) -- the geometry, rsqrt and r
// of a pair are shared by the tile; everything else (LDS, MUFU seed, integer exponent work, loop control) issues in the
// shadow of the half-rate FP64 pipe at ~0.75 cycles per instruction, and from OT = 4 on the exp-table gathers bring the
// shared-memory pipe to the same load (96 % at OT = 7).  A DFMA with three distinct vector-register sources holds the pipe
// for 3 cycles instead of 2: constants are kept in uniform registers / immediates wherever ptxas allows.
#include "kernels.cuh"

#include "fp64_math.cuh"

namespace bltc {
namespace {

constexpr int kNearUnroll = 2, kFarUnroll = 2;
// resident CTAs per SM the pair kernels are compiled for: 2 x 8 warps at <= 128 registers.  Measured alternatives
// (DESIGN.md 10): 1 x 8 warps at 255 registers (ptxas then interleaves every pair of a proxy row) and 1 x 12 warps at
// 168 registers are within +-2 % -- the shared-memory and FP64 pipes co-limit the tile, not the dependent-issue stalls.
constexpr int kPairCtasPerSm = (kPairWarps == 8 && kTargetsPerThread <= 2) ? 2 : 1;     // sources / proxy points per loop trip (x R targets)

constexpr double kInv2Pi = 0.15915494309189533577;   // 2 / (4 pi)

// {0.375, BLTC_EXP_C2, kExpMagic}: constants the pair kernels keep in registers (see fp64_math.cuh, MathRegs)
__device__ double kMathOpaque[3] = {0.375, BLTC_EXP_C2, kExpMagic};

// ------------------------------------------------------------------------------------ a1 / pack
__global__ void gather_kernel(const double* __restrict__ f, int64_t stride, int o0, int ot,
                              const int32_t* __restrict__ perm, int64_t n, double* __restrict__ dst) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t src = perm ? (int64_t)perm[i] : i;
    for (int o = 0; o < ot; ++o) dst[i * ot + o] = f[(int64_t)(o0 + o) * stride + src];
}

__global__ void pack_kernel(const double* __restrict__ coords, const double* __restrict__ w,
                            const int32_t* __restrict__ perm, int64_t n, double4* __restrict__ rec) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t s = perm ? (int64_t)perm[i] : i;
    rec[i] = make_double4(coords[s], coords[n + s], coords[2 * n + s], w ? w[s] : 0.0);
}

// Bounding boxes of consecutive chunks of a SoA point set: out[chunk] = {lo[3], hi[3]}.  direct_convolve uses them
// to decide where a source can coincide with a target (reading R3) and whether exp can underflow.
__global__ void __launch_bounds__(kThreads)
chunk_bbox_kernel(const double* __restrict__ coords, int64_t n, int64_t chunk, double* __restrict__ out) {
    __shared__ double s_lo[3][kThreads / 32], s_hi[3][kThreads / 32];
    const int64_t b = (int64_t)blockIdx.x * chunk, e = min(n, b + chunk);
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t i = b + threadIdx.x; i < e; i += kThreads)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double v = coords[(int64_t)d * n + i];
            lo[d] = fmin(lo[d], v); hi[d] = fmax(hi[d], v);
        }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        for (int s = 16; s > 0; s >>= 1) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], s));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], s));
        }
        if ((threadIdx.x & 31) == 0) { s_lo[d][threadIdx.x >> 5] = lo[d]; s_hi[d][threadIdx.x >> 5] = hi[d]; }
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        const int d = threadIdx.x;
        double a = s_lo[d][0], c = s_hi[d][0];
        for (int w = 1; w < kThreads / 32; ++w) { a = fmin(a, s_lo[d][w]); c = fmax(c, s_hi[d][w]); }
        out[(size_t)blockIdx.x * 6 + d] = a; out[(size_t)blockIdx.x * 6 + 3 + d] = c;
    }
}

// ------------------------------------------------------------------------------------ a2
// One CTA per work item = (proxy cluster, chunk of its particles).  Phase A: barycentric Lagrange
// values L_k(x_j), L_k(y_j), L_k(z_j) for a tile of particles (Eq. (38)-(39); exact node hits give the
// unit vector, reading R7).  Phase B: every thread owns a (k1, k2) row and G3 consecutive k3 and accumulates
//   qhat_k += L_k1 L_k2 L_k3 q_j      (Eq. (35) right)
// A cluster cut into several chunks is finished by upward_reduce_kernel (chunk order => deterministic).
constexpr int kUpTile = 64;

template <int OT, int G3>
__global__ void __launch_bounds__(kThreads)
upward_kernel(const UpItem* __restrict__ items, const double* __restrict__ slot_nodes, int n1,
              const double4* __restrict__ src_rec, const double* __restrict__ fsrc,
              double* __restrict__ out, double* __restrict__ chunk_out) {
    constexpr int NC = OT == 0 ? 1 : OT;
    extern __shared__ double sm[];
    const int LS = n1 + 3;                       // padded row of L values (pad = 0)
    double* s_nodes = sm;                        // [3][n1]
    double* s_L = s_nodes + 3 * n1;              // [kUpTile][3][LS]
    double* s_q = s_L + kUpTile * 3 * LS;        // [kUpTile][NC]
    const int tid = threadIdx.x;
    const UpItem it = items[blockIdx.x];
    const int slot = it.slot, b = it.begin, e = it.end;
    const int n = n1 - 1;
    const int P = n1 * n1 * n1;
    double* dst = it.dst < 0 ? out + (size_t)slot * P * NC : chunk_out + (size_t)it.dst * P * NC;
    for (int i = tid; i < 3 * n1; i += kThreads) s_nodes[i] = slot_nodes[(size_t)slot * 3 * n1 + i];
    for (int i = tid; i < kUpTile * 3 * LS; i += kThreads) s_L[i] = 0.0;
    const int gpr = (n1 + G3 - 1) / G3;          // groups of G3 k3 per (k1, k2) row
    const int units = n1 * n1 * gpr;
    for (int u0 = 0; u0 < units; u0 += kThreads) {
        const int u = u0 + tid;
        const bool active = u < units;
        const int row = active ? u / gpr : 0;
        const int k3a = active ? (u % gpr) * G3 : 0;
        const int k1 = row / n1, k2 = row % n1;
        double acc[G3][NC];
#pragma unroll
        for (int p = 0; p < G3; ++p)
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[p][c] = 0.0;
        for (int j0 = b; j0 < e; j0 += kUpTile) {
            __syncthreads();
            for (int t = tid; t < kUpTile * 3; t += kThreads) {
                const int jj = t / 3, d = t % 3;
                double* L = s_L + (jj * 3 + d) * LS;
                if (j0 + jj < e) {
                    const double4 r = src_rec[j0 + jj];
                    const double v = d == 0 ? r.x : (d == 1 ? r.y : r.z);
                    const double* s = s_nodes + d * n1;
                    int hit = -1;
                    for (int k = 0; k < n1; ++k) if (v == s[k]) hit = k;
                    if (hit >= 0) {
                        for (int k = 0; k < n1; ++k) L[k] = (k == hit) ? 1.0 : 0.0;
                    } else {
                        double sum = 0.0;
                        for (int k = 0; k < n1; ++k) {
                            const double bk = ((k & 1) ? -1.0 : 1.0) * ((k == 0 || k == n) ? 0.5 : 1.0);
                            const double t2 = bk / (v - s[k]);
                            L[k] = t2; sum += t2;
                        }
                        const double inv = 1.0 / sum;
                        for (int k = 0; k < n1; ++k) L[k] *= inv;
                    }
                } else {
                    for (int k = 0; k < n1; ++k) L[k] = 0.0;
                }
            }
            for (int t = tid; t < kUpTile; t += kThreads) {
                if (j0 + t < e) {
                    const double w = src_rec[j0 + t].w;
#pragma unroll
                    for (int c = 0; c < NC; ++c)
                        s_q[t * NC + c] = OT == 0 ? w : fsrc[(size_t)(j0 + t) * NC + c] * w;
                } else {
#pragma unroll
                    for (int c = 0; c < NC; ++c) s_q[t * NC + c] = 0.0;
                }
            }
            __syncthreads();
            if (active) {
                const int cnt = min(kUpTile, e - j0);
                for (int jj = 0; jj < cnt; ++jj) {
                    const double* L = s_L + jj * 3 * LS;
                    const double a12 = L[k1] * L[LS + k2];
                    double q[NC];
#pragma unroll
                    for (int c = 0; c < NC; ++c) q[c] = s_q[jj * NC + c];
#pragma unroll
                    for (int p = 0; p < G3; ++p) {
                        const double a = a12 * L[2 * LS + k3a + p];
#pragma unroll
                        for (int c = 0; c < NC; ++c) acc[p][c] = fma(a, q[c], acc[p][c]);
                    }
                }
            }
        }
        if (active) {
#pragma unroll
            for (int p = 0; p < G3; ++p) {
                const int k3 = k3a + p;
                if (k3 < n1) {
                    const size_t kk = (size_t)(k1 * n1 + k2) * n1 + k3;
#pragma unroll
                    for (int c = 0; c < NC; ++c) dst[kk * NC + c] = acc[p][c];
                }
            }
        }
    }
}

// Child -> parent upward pass (reading R23): one CTA per parent slot.  For every child, in order: the per-axis
// matrices A_d[k'][K] = L^P_K(s^c_{d,k'}) (Eq. (38)-(39) of the PARENT's grid at the child's nodes, node hits per R7),
// then per component the tensor contraction  out[K1][K2][K3] += sum_{k'} A_1[k1'][K1] A_2[k2'][K2] A_3[k3'][K3] q^c[k']
// in three passes through shared memory.  In exact arithmetic the result equals Eq. (35) applied to the parent's own
// particles (L^P_K is a polynomial of degree n); the cost is O(P n) per child and component instead of O(N_C P).
// charges: [slot][P][NC] (fhat) or [slot][P] (what, NC = 1); children are complete when the launch starts (deeper level).
template <int NC>
__global__ void __launch_bounds__(kThreads)
upward_children_kernel(const C2PItem* __restrict__ items, const double* __restrict__ slot_nodes, int n1,
                       double* __restrict__ charges) {
    extern __shared__ double sm[];
    const int P = n1 * n1 * n1, n = n1 - 1, tid = threadIdx.x;
    double* s_A = sm;                            // [3][n1][n1]
    double* s_b0 = s_A + 3 * n1 * n1;            // [P]
    double* s_b1 = s_b0 + P;                     // [P]
    const C2PItem it = items[blockIdx.x];
    const double* sP = slot_nodes + (size_t)it.parent * 3 * n1;
    double* dst = charges + (size_t)it.parent * P * NC;
    for (int q = 0; q < it.nchild; ++q) {
        const double* sC = slot_nodes + (size_t)it.child[q] * 3 * n1;
        const double* src = charges + (size_t)it.child[q] * P * NC;
        __syncthreads();
        for (int t = tid; t < 3 * n1; t += kThreads) {
            const int d = t / n1;
            const double v = sC[t];
            const double* s = sP + d * n1;
            double* L = s_A + t * n1;
            int hit = -1;
            for (int k = 0; k < n1; ++k) if (v == s[k]) hit = k;
            if (hit >= 0) {
                for (int k = 0; k < n1; ++k) L[k] = (k == hit) ? 1.0 : 0.0;
            } else {
                double sum = 0.0;
                for (int k = 0; k < n1; ++k) {
                    const double bk = ((k & 1) ? -1.0 : 1.0) * ((k == 0 || k == n) ? 0.5 : 1.0);
                    const double t2 = bk / (v - s[k]);
                    L[k] = t2; sum += t2;
                }
                const double inv = 1.0 / sum;
                for (int k = 0; k < n1; ++k) L[k] *= inv;
            }
        }
        for (int c = 0; c < NC; ++c) {
            __syncthreads();
            for (int i = tid; i < P; i += kThreads) s_b0[i] = src[(size_t)i * NC + c];
            __syncthreads();
            for (int i = tid; i < P; i += kThreads) {               // b1[K1][k2'][k3'] = sum_k1' A_1[k1'][K1] b0[k1'][k2'][k3']
                const int K1 = i / (n1 * n1), rest = i - K1 * n1 * n1;
                double a = 0.0;
                for (int k = 0; k < n1; ++k) a = fma(s_A[k * n1 + K1], s_b0[k * n1 * n1 + rest], a);
                s_b1[i] = a;
            }
            __syncthreads();
            for (int i = tid; i < P; i += kThreads) {               // b0[K1][K2][k3'] = sum_k2' A_2[k2'][K2] b1[K1][k2'][k3']
                const int K1 = i / (n1 * n1), K2 = (i / n1) % n1, k3 = i % n1;
                double a = 0.0;
                for (int k = 0; k < n1; ++k) a = fma(s_A[(n1 + k) * n1 + K2], s_b1[(K1 * n1 + k) * n1 + k3], a);
                s_b0[i] = a;
            }
            __syncthreads();
            for (int i = tid; i < P; i += kThreads) {               // out[K1][K2][K3] (+)= sum_k3' A_3[k3'][K3] b0[K1][K2][k3']
                const int K3 = i % n1, row = i - K3;
                double a = 0.0;
                for (int k = 0; k < n1; ++k) a = fma(s_A[(2 * n1 + k) * n1 + K3], s_b0[row + k], a);
                const size_t o = (size_t)i * NC + c;
                dst[o] = q == 0 ? a : dst[o] + a;
            }
        }
    }
}

// out[slot][i] = sum over the slot's chunks (in chunk order) of chunk_out[first + c][i],  i < P * NC
__global__ void __launch_bounds__(kThreads)
upward_reduce_kernel(const UpReduce* __restrict__ red, int len, const double* __restrict__ chunk_out,
                     double* __restrict__ out) {
    const UpReduce r = red[blockIdx.y];
    for (int i = blockIdx.x * kThreads + threadIdx.x; i < len; i += gridDim.x * kThreads) {
        double s = 0.0;
        for (int c = 0; c < r.count; ++c) s += chunk_out[(size_t)(r.first + c) * len + i];
        out[(size_t)r.slot * len + i] = s;
    }
}

// ------------------------------------------------------------------------------------ shared pieces
template <int R, int OT>
struct TargetRegs {
    double x[R], y[R], z[R];
    double f[R][OT];
    double acc[R][OT];
    bool valid[R];
    int tl[R];
};

template <int R, int OT, bool SUB>
__device__ __forceinline__ void load_targets(TargetRegs<R, OT>& T, const WorkItem& it, int grp, int lane,
                                             const double4* __restrict__ tgt_rec,
                                             const double* __restrict__ ftgt) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        T.tl[r] = (grp * R + r) * 32 + lane;
        T.valid[r] = T.tl[r] < it.tgt_count;
        const int ti = it.tgt_begin + (T.valid[r] ? T.tl[r] : 0);    // padded lanes shadow target 0
        const double4 t = tgt_rec[ti];
        T.x[r] = t.x; T.y[r] = t.y; T.z[r] = t.z;
#pragma unroll
        for (int o = 0; o < OT; ++o) {
            T.f[r][o] = SUB ? ftgt[(size_t)ti * OT + o] : 0.0;
            T.acc[r][o] = 0.0;
        }
    }
}

// Reduce the S source-split partial sums of each target (fixed order) and store the tile's slice.
template <int R, int OT>
__device__ __forceinline__ void reduce_and_store(TargetRegs<R, OT>& T, const WorkItem& it, int warp,
                                                 int lane, int split, int S, double* s_red,
                                                 double* __restrict__ partial, int64_t partial_len) {
    if (S > 1) {
        __syncthreads();                                   // staging tile no longer needed
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int o = 0; o < OT; ++o) s_red[((r * OT + o) * kPairWarps + warp) * 32 + lane] = T.acc[r][o];
        __syncthreads();
        if (split == 0) {
            const int G = kPairWarps / S;
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int o = 0; o < OT; ++o) {
                    double s = T.acc[r][o];
                    for (int q = 1; q < S; ++q) s += s_red[((r * OT + o) * kPairWarps + warp + q * G) * 32 + lane];
                    T.acc[r][o] = s;
                }
        }
    }
    if (split == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (T.valid[r])
#pragma unroll
                for (int o = 0; o < OT; ++o)
                    partial[(int64_t)o * partial_len + it.partial_off + T.tl[r]] = T.acc[r][o];
    }
}

// ------------------------------------------------------------------------------------ a4 / a6
// Shared-memory tile of sources: one record {x, y, z, w, f[OT]} per source, padded to a multiple of
// 16 bytes, so one source is 3-4 LDS.128 at immediate offsets from one running pointer.  The S
// source-split ways of a tile take contiguous chunks of it (broadcast reads: no bank conflicts).
constexpr int src_rec_doubles(int ot) { return 4 + 2 * ((ot + 1) / 2); }
template <int OT> struct SrcRec { static constexpr int kDoubles = src_rec_doubles(OT); };

// ZS (zero-safe): the tile may hold a source that coincides with a target -> the singular term is
// skipped by an integer select on the rsqrt seed (reading R3).  The host flags the
// ranges for which that can happen (bounding boxes intersect); all other tiles run the ZS = false loop.
//
// KIND = kYukawa:  acc += e^{-k_o r} (w_j / r) (f_j - f_i)                                  Eq. (20), (34)
// KIND = kCoulomb: acc += (w_j / r) (f_j - f_i e^{-r^2/alpha^2})   (one Gaussian per pair, shared by the
//                  orbitals of the tile; kp.c[0] = -T/(ln2 alpha^2))                        Eq. (23), (34)
template <int R, int OT, bool SUB, bool GUARD, bool ZS, int KIND>
__device__ __forceinline__ void near_tile(TargetRegs<R, OT>& T, const double* __restrict__ tile, int j0, int j1,
                                          const KPar& kp, uint32_t tab, const MathRegs& mr) {
    constexpr int RD = SrcRec<OT>::kDoubles;
    const ExpConst ec{kp.c1, kp.c3};
#pragma unroll kNearUnroll
    for (int j = j0; j < j1; ++j) {
        const double* s = tile + j * RD;
        const double2 sxy = *reinterpret_cast<const double2*>(s);
        const double2 szw = *reinterpret_cast<const double2*>(s + 2);
        double sf[OT];
#pragma unroll
        for (int o = 0; o < OT; o += 2) {
            if (o + 1 < OT) {
                const double2 v = *reinterpret_cast<const double2*>(s + 4 + o);
                sf[o] = v.x; sf[o + 1] = v.y;
            } else {
                sf[o] = s[4 + o];
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double dx = T.x[r] - sxy.x, dy = T.y[r] - sxy.y, dz = T.z[r] - szw.x;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            double rinv, rr;
            rsqrt_sqrt<ZS>(r2, rinv, rr, mr);              // ZS and r2 == 0: rinv = 0, the term vanishes
            const double gw = rinv * szw.y;
            if (KIND == kCoulomb) {
                const double gs = SUB ? exp_neg_kr<GUARD>(r2, kp.c[0], tab, mr, ec) : 0.0;   // e^{-r^2/alpha^2}
#pragma unroll
                for (int o = 0; o < OT; ++o) {
                    const double df = SUB ? fma(-T.f[r][o], gs, sf[o]) : sf[o];   // f_j - f_i e^{-r^2/alpha^2}, Eq. (23)
                    T.acc[r][o] = fma(gw, df, T.acc[r][o]);
                }
            } else {
#pragma unroll
                for (int o = 0; o < OT; ++o) {
                    const double ex = exp_neg_kr<GUARD>(rr, kp.c[o], tab, mr, ec);
                    const double g = ex * gw;
                    const double df = SUB ? (sf[o] - T.f[r][o]) : sf[o];     // (f_j - f_i), Eq. (20)
                    T.acc[r][o] = fma(g, df, T.acc[r][o]);
                }
            }
        }
    }
}

// The work of one near-field CTA with R targets per thread (R = 2: groups of 64 targets; R = 1: the half-group tile
// tiles that hold the tail of a ragged batch, WorkItem::rshift).
template <int R, int OT, bool SUB, bool GUARD, int KIND, bool ALLZS>
__device__ __forceinline__ void near_body(const WorkItem& it, const Range* __restrict__ ranges,
                                          const double4* __restrict__ src_rec, const double* __restrict__ fsrc,
                                          const double4* __restrict__ tgt_rec, const double* __restrict__ ftgt,
                                          const KPar& kp, double* __restrict__ partial, int64_t partial_len,
                                          double* s_tile, uint32_t tab, const MathRegs& mr) {
    constexpr int RD = SrcRec<OT>::kDoubles;
    static_assert(RD * kSrcTile >= R * OT * kPairWarps * 32, "reduction scratch fits in the tile");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = 1 << it.gshift, S = kPairWarps >> it.gshift;
    const int grp = warp & (G - 1), split = warp >> it.gshift;
    TargetRegs<R, OT> T;
    load_targets<R, OT, SUB>(T, it, grp, lane, tgt_rec, ftgt);

    int q = it.list_begin;
    int at = q < it.list_end ? ranges[q].begin : 0;
    while (q < it.list_end) {
        __syncthreads();                                   // previous tile consumed (and table ready)
        int fill = 0, flags = 0;
        while (fill < kSrcTile && q < it.list_end) {
            const Range rg = ranges[q];
            const int n = min(kSrcTile - fill, rg.end - at);
            flags |= rg.flags;
            for (int i = tid; i < n; i += kPairThreads) {
                const double4 v = src_rec[at + i];
                double* d = s_tile + (fill + i) * RD;
                *reinterpret_cast<double2*>(d) = make_double2(v.x, v.y);
                *reinterpret_cast<double2*>(d + 2) = make_double2(v.z, v.w);
#pragma unroll
                for (int o = 0; o < OT; ++o) d[4 + o] = fsrc[(size_t)(at + i) * OT + o];
            }
            fill += n; at += n;
            if (at == rg.end) { ++q; if (q < it.list_end) at = ranges[q].begin; }
        }
        __syncthreads();
        const int j0 = (fill * split) / S, j1 = (fill * (split + 1)) / S;
        // ALLZS (direct_convolve: a target sample meets every source segment): ONE pair loop in the kernel.  With two
        // loops ptxas keeps the exp constants of the first one in vector registers instead of uniform registers, and a
        // DFMA with three distinct vector-register sources holds the FP64 pipe for 3 cycles instead of 2;
        // the treecode's near field rarely needs the zero-safe loop, so it is the one that comes first.
        if (ALLZS || (flags & kRangeMayCoincide)) near_tile<R, OT, SUB, GUARD, true, KIND>(T, s_tile, j0, j1, kp, tab, mr);
        else near_tile<R, OT, SUB, GUARD, false, KIND>(T, s_tile, j0, j1, kp, tab, mr);
    }
    reduce_and_store<R, OT>(T, it, warp, lane, split, S, s_tile, partial, partial_len);
}

template <int R, int OT, bool SUB, bool GUARD, int KIND, bool ALLZS>
__global__ void __launch_bounds__(kPairThreads, kPairCtasPerSm)
near_kernel(const WorkItem* __restrict__ items, const Range* __restrict__ ranges,
            const double4* __restrict__ src_rec, const double* __restrict__ fsrc,
            const double4* __restrict__ tgt_rec, const double* __restrict__ ftgt, const KPar kp,
            double* __restrict__ partial, int64_t partial_len) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t tab = exp_table_init((uint32_t)__cvta_generic_to_shared(smem_raw), threadIdx.x, kPairThreads);
    double* s_tile = reinterpret_cast<double*>(smem_raw + kExpTableSmemBytes);
    const MathRegs mr = math_regs_init(kMathOpaque);
    const WorkItem it = items[blockIdx.x];
    if (it.rshift == 0) {
        near_body<R, OT, SUB, GUARD, KIND, ALLZS>(it, ranges, src_rec, fsrc, tgt_rec, ftgt, kp, partial, partial_len, s_tile, tab, mr);
    } else if (R >= 4 && it.rshift == 2) {
        near_body<(R >= 4 ? R / 4 : 1), OT, SUB, GUARD, KIND, ALLZS>(it, ranges, src_rec, fsrc, tgt_rec, ftgt, kp, partial, partial_len, s_tile, tab, mr);
    } else {
        near_body<(R >= 2 ? R / 2 : 1), OT, SUB, GUARD, KIND, ALLZS>(it, ranges, src_rec, fsrc, tgt_rec, ftgt, kp, partial, partial_len, s_tile, tab, mr);
    }
}

// ------------------------------------------------------------------------------------ a3
// Shared-memory tile of proxy points: one record {what_k, fhat_k[OT]} per point (padded to 16 bytes),
// k3 fastest, so a (k1, k2) row of the tensor grid is n1 consecutive records.  N1 > 0: the grid size
// degree + 1 is a compile-time constant and the k3 loop is fully unrolled (no remainder iteration, the
// next row's dx^2 + dy^2 overlaps the tail of the current one); N1 = 0: any degree.
constexpr int proxy_rec_doubles(int ot) { return 2 * ((ot + 2) / 2); }
// tile of proxy points: 64 KB (exp table) + tile must fit kPairCtasPerSm times in an SM's 227 KB of shared memory
constexpr int proxy_tile(int ot) { return (ot <= 4 || kPairCtasPerSm == 1) ? kProxyTile : 768; }
template <int OT> struct ProxyRec {
    static constexpr int kDoubles = proxy_rec_doubles(OT);
    static constexpr int kTile = proxy_tile(OT);
};

// KIND = kCoulomb: acc += (fhat_k - f_i what_k e^{-r^2/alpha^2}) / r  (reading R21: the Gaussian of Eq. (23)
// is interpolated with the proxy weights of w).
template <int R, int OT, bool SUB, bool GUARD, int KIND, int N1>
__device__ __forceinline__ void far_body(const WorkItem& it, const int32_t* __restrict__ far_slots,
                                         const double* __restrict__ slot_nodes, const double* __restrict__ what,
                                         const double* __restrict__ fhat, int n1_arg,
                                         const double4* __restrict__ tgt_rec, const double* __restrict__ ftgt,
                                         const KPar& kp, double* __restrict__ partial, int64_t partial_len,
                                         double* s_pts, uint32_t tab, const MathRegs& mr) {
    constexpr int PD = ProxyRec<OT>::kDoubles;
    constexpr int PT = ProxyRec<OT>::kTile;
    static_assert(PT * PD >= R * OT * kPairWarps * 32, "reduction scratch fits in the tile");
    // compile-time grid size: the k3 loop is fully unrolled up to 5 orbitals; wider tiles unroll 3 proxy points per
    // trip (fully unrolled they spill registers: far kernel at 7 orbitals 567 -> 520 ms on the cfg1 mesh x 21 orbitals)
    constexpr int kU = N1 ? (OT >= 6 ? 3 : N1) : kFarUnroll;
    const int n1 = N1 ? N1 : n1_arg;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* s_nodes = s_pts + PT * PD;                   // [3][21]
    const ExpConst ec{kp.c1, kp.c3};
    const int G = 1 << it.gshift, S = kPairWarps >> it.gshift;
    const int grp = warp & (G - 1), split = warp >> it.gshift;
    TargetRegs<R, OT> T;
    load_targets<R, OT, SUB>(T, it, grp, lane, tgt_rec, ftgt);

    const int plane = n1 * n1;
    const int P = plane * n1;
    const int planes_per_chunk = max(1, PT / plane);
    for (int q = it.list_begin; q < it.list_end; ++q) {
        const int slot = far_slots[q];
        for (int k1a = 0; k1a < n1; k1a += planes_per_chunk) {
            const int k1b = min(n1, k1a + planes_per_chunk);
            const int npts = (k1b - k1a) * plane;
            __syncthreads();
            if (k1a == 0)
                for (int i = tid; i < 3 * n1; i += kPairThreads) s_nodes[i] = slot_nodes[(size_t)slot * 3 * n1 + i];
            const size_t base = (size_t)slot * P + (size_t)k1a * plane;
            for (int i = tid; i < npts; i += kPairThreads) {
                double* d = s_pts + i * PD;
                d[0] = SUB ? what[base + i] : 0.0;
#pragma unroll
                for (int o = 0; o < OT; ++o) d[1 + o] = fhat[(base + i) * OT + o];
            }
            __syncthreads();
            const int rows = (k1b - k1a) * n1;
            for (int row = split; row < rows; row += S) {
                const int kq = row / n1;
                const int k1 = k1a + kq, k2 = row - kq * n1;
                double dxy2[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double dx = T.x[r] - s_nodes[k1], dy = T.y[r] - s_nodes[n1 + k2];
                    dxy2[r] = fma(dy, dy, dx * dx);
                }
                const double* pr = s_pts + row * n1 * PD;
                const double* pz = s_nodes + 2 * n1;
#pragma unroll kU
                for (int k3 = 0; k3 < n1; ++k3) {
                    const double sz = pz[k3];
                    const double* rec = pr + k3 * PD;
                    double wv, fv[OT];
                    if (OT == 1) {
                        const double2 v = *reinterpret_cast<const double2*>(rec);
                        wv = v.x; fv[0] = v.y;
                    } else {
                        const double2 v = *reinterpret_cast<const double2*>(rec);
                        wv = v.x; fv[0] = v.y;
#pragma unroll
                        for (int o = 1; o < OT; o += 2) {
                            if (o + 1 < OT) {
                                const double2 u = *reinterpret_cast<const double2*>(rec + 1 + o);
                                fv[o] = u.x; fv[o + 1] = u.y;
                            } else {
                                fv[o] = rec[1 + o];
                            }
                        }
                    }
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double dz = T.z[r] - sz;
                        const double r2 = fma(dz, dz, dxy2[r]);
                        double rinv, rr;
                        rsqrt_sqrt<false>(r2, rinv, rr, mr);   // MAC keeps targets off the grid (theta < 1)
                        if (KIND == kCoulomb) {
                            const double wg = SUB ? wv * exp_neg_kr<GUARD>(r2, kp.c[0], tab, mr, ec) : 0.0;
#pragma unroll
                            for (int o = 0; o < OT; ++o) {
                                const double qk = SUB ? fma(-T.f[r][o], wg, fv[o]) : fv[o];
                                T.acc[r][o] = fma(rinv, qk, T.acc[r][o]);
                            }
                        } else {
#pragma unroll
                            for (int o = 0; o < OT; ++o) {
                                const double ex = exp_neg_kr<GUARD>(rr, kp.c[o], tab, mr, ec);
                                const double g = ex * rinv;
                                // fhat_k - f_i what_k: interpolated charges of (f_j - f_i) w_j (reading R11)
                                const double qk = SUB ? fma(-T.f[r][o], wv, fv[o]) : fv[o];
                                T.acc[r][o] = fma(g, qk, T.acc[r][o]);
                            }
                        }
                    }
                }
            }
        }
    }
    reduce_and_store<R, OT>(T, it, warp, lane, split, S, s_pts, partial, partial_len);
}

template <int R, int OT, bool SUB, bool GUARD, int KIND, int N1>
__global__ void __launch_bounds__(kPairThreads, kPairCtasPerSm)
far_kernel(const WorkItem* __restrict__ items, const int32_t* __restrict__ far_slots,
           const double* __restrict__ slot_nodes, const double* __restrict__ what,
           const double* __restrict__ fhat, int n1_arg, const double4* __restrict__ tgt_rec,
           const double* __restrict__ ftgt, const KPar kp, double* __restrict__ partial,
           int64_t partial_len) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t tab = exp_table_init((uint32_t)__cvta_generic_to_shared(smem_raw), threadIdx.x, kPairThreads);
    double* s_pts = reinterpret_cast<double*>(smem_raw + kExpTableSmemBytes);
    const MathRegs mr = math_regs_init(kMathOpaque);
    const WorkItem it = items[blockIdx.x];
    if (it.rshift == 0) {
        far_body<R, OT, SUB, GUARD, KIND, N1>(it, far_slots, slot_nodes, what, fhat, n1_arg, tgt_rec, ftgt, kp, partial, partial_len, s_pts, tab, mr);
    } else if (R >= 4 && it.rshift == 2) {
        far_body<(R >= 4 ? R / 4 : 1), OT, SUB, GUARD, KIND, N1>(it, far_slots, slot_nodes, what, fhat, n1_arg, tgt_rec, ftgt, kp, partial, partial_len, s_pts, tab, mr);
    } else {
        far_body<(R >= 2 ? R / 2 : 1), OT, SUB, GUARD, KIND, N1>(it, far_slots, slot_nodes, what, fhat, n1_arg, tgt_rec, ftgt, kp, partial, partial_len, s_pts, tab, mr);
    }
}

// ------------------------------------------------------------------------------------ a5
template <int OT, bool SUB>
__global__ void __launch_bounds__(kThreads)
epilogue_kernel(const int32_t* __restrict__ b_begin, const int32_t* __restrict__ b_count,
                const int64_t* __restrict__ b_partial_base, const int32_t* __restrict__ b_nseg,
                const double* __restrict__ partial, int64_t partial_len, const double* __restrict__ ftgt,
                const EpiPar ep, const int32_t* __restrict__ perm, const OutSet outs, int64_t stride,
                int o0) {
    const int b = blockIdx.x;
    const int begin = b_begin[b], count = b_count[b], nseg = b_nseg[b];
    const int64_t base = b_partial_base[b];
    for (int l = threadIdx.x; l < count; l += kThreads) {
        const int i = begin + l;
        const int64_t dst = perm ? (int64_t)perm[i] : (int64_t)i;
#pragma unroll
        for (int o = 0; o < OT; ++o) {
            double s = 0.0;
            for (int g = 0; g < nseg; ++g) s += partial[(int64_t)o * partial_len + base + (int64_t)g * count + l];
            double v = ep.scale * s;                               // Yukawa: -2 * S / (4 pi);  Coulomb: S
            if (SUB) v = fma(ep.coef[o], ftgt[(size_t)i * OT + o], v);   // -2 f_i/k^2 (Eq. (21)) / 2 pi alpha^2 f_i (Eq. (24))
            // one result, every destination: the rank's own out and, when the all-gather is fused in, its peers'
            for (int r = 0; r < outs.n; ++r) outs.p[r][(int64_t)(o0 + o) * stride + dst] = v;
        }
    }
}

// ------------------------------------------------------------------------------------ probe
// FORM 0: a = fma(a, m, c) with m, c the same for every chain (held in the operand-reuse cache): the FP64 pipe's peak.
// FORM 1: a = fma(b_i, d_j, a) -- three distinct vector-register sources per instruction, nothing to reuse: such a
//         DFMA holds the pipe for 3 cycles instead of 2 on sm_100a (the accumulate of the pair kernels is of this form).
template <int FORM>
__global__ void __launch_bounds__(kThreads)
fp64_probe_kernel(int iters, double seed, double* sink) {
    double a[8], b[8], d[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i] = seed + (double)(threadIdx.x + i);
        b[i] = 1.0 + 1e-9 * (double)(threadIdx.x + i);
        d[i] = 1e-12 * (double)(3 * threadIdx.x + i);
    }
    const double m = 1.0 + 1e-9 * seed, c = 1e-12;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 64; ++u)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = FORM == 0 ? fma(a[i], m, c) : fma(b[i], d[i], a[i]);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == 123.456) sink[0] = s;
}

size_t near_smem_bytes(int ot) { return (size_t)kExpTableSmemBytes + sizeof(double) * (size_t)kSrcTile * src_rec_doubles(ot); }
size_t far_smem_bytes(int ot) {
    return (size_t)kExpTableSmemBytes + sizeof(double) * ((size_t)proxy_tile(ot) * proxy_rec_doubles(ot) + 3 * 21);
}
static_assert(kPairCtasPerSm * (kExpTableSmemBytes + 8 * kSrcTile * src_rec_doubles(kMaxOT) + 1024) <= 228 * 1024 &&
              kPairCtasPerSm * (kExpTableSmemBytes + 8 * (proxy_tile(kMaxOT) * proxy_rec_doubles(kMaxOT) + 63) + 1024) <= 228 * 1024,
              "the resident pair-kernel CTAs (+ 1 KB reserved each) fit in an SM's shared memory at the widest orbital tile");

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
    if (bytes > 48 * 1024) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    return cudaSuccess;
}

}  // namespace

// ===================================================================================== launchers
KPar make_kpar(const double* k, int ot) {
    KPar kp;
    for (int o = 0; o < kMaxOT; ++o) {
        const double kk = o < ot ? k[o] : 1.0;
        kp.nk[o] = -kk;
        kp.c[o] = exp_scale_of_k(kk);
    }
    kp.c1 = BLTC_EXP_C1;
#if BLTC_EXP_DEG == 3
    kp.c3 = BLTC_EXP_C3;
#else
    kp.c3 = 0.0;
#endif
    return kp;
}

KPar make_kpar_coulomb(double alpha) {
    KPar kp;
    for (int o = 0; o < kMaxOT; ++o) {
        kp.nk[o] = 0.0;
        // e^{-r^2/alpha^2} = exp(-(1/alpha^2) r2): the same scaled-argument form as e^{-k r}
        kp.c[o] = (double)(-(long double)BLTC_EXP_T / ((long double)alpha * (long double)alpha *
                                                        0.693147180559945309417232121458176568L));
    }
    kp.c1 = BLTC_EXP_C1;
#if BLTC_EXP_DEG == 3
    kp.c3 = BLTC_EXP_C3;
#else
    kp.c3 = 0.0;
#endif
    return kp;
}

EpiPar make_epipar(const double* k, int ot) {
    EpiPar ep;
    ep.scale = -kInv2Pi;                                   // -2 / (4 pi)
    for (int o = 0; o < kMaxOT; ++o) ep.coef[o] = o < ot ? -2.0 / (k[o] * k[o]) : 0.0;   // Eq. (21)
    return ep;
}

EpiPar make_epipar_coulomb(double alpha) {
    EpiPar ep;
    ep.scale = 1.0;
    for (int o = 0; o < kMaxOT; ++o) ep.coef[o] = 2.0 * 3.14159265358979323846 * alpha * alpha;   // Eq. (24)
    return ep;
}

cudaError_t launch_gather(const double* f, int64_t stride, int o0, int ot, const int32_t* perm,
                          int64_t n, double* dst, cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(f, stride, o0, ot, perm, n, dst);
    return cudaGetLastError();
}

cudaError_t launch_pack_records(const double* coords, const double* w, const int32_t* perm, int64_t n,
                                double4* rec, cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    pack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(coords, w, perm, n, rec);
    return cudaGetLastError();
}

cudaError_t launch_chunk_bbox(const double* coords, int64_t n, int64_t chunk, double* out, cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    chunk_bbox_kernel<<<(unsigned)((n + chunk - 1) / chunk), kThreads, 0, st>>>(coords, n, chunk, out);
    return cudaGetLastError();
}

cudaError_t launch_upward(int ot, const UpItem* items, int nitems, const UpReduce* red, int nred,
                          const double* slot_nodes, int degree, const double4* src_rec,
                          const double* fsrc, double* out, double* chunk_out, cudaStream_t st) {
    if (nitems == 0) return cudaSuccess;
    const int n1 = degree + 1;
    const int nc = ot == 0 ? 1 : ot;
    const size_t smem = sizeof(double) * (3 * n1 + (size_t)kUpTile * 3 * (n1 + 3) + (size_t)kUpTile * nc);
    const bool g3 = (n1 % 3 == 0) || ((n1 + 2) / 3 * 3 - n1 < (n1 + 3) / 4 * 4 - n1);   // less padding with 3 than with 4
    cudaError_t e = cudaSuccess;
#define BLTC_UP(OTV)                                                                                   \
    case OTV:                                                                                          \
        if (g3) {                                                                                      \
            e = set_smem(upward_kernel<OTV, 3>, smem);                                                 \
            if (e != cudaSuccess) return e;                                                            \
            upward_kernel<OTV, 3><<<nitems, kThreads, smem, st>>>(items, slot_nodes, n1, src_rec,      \
                                                                   fsrc, out, chunk_out);              \
        } else {                                                                                       \
            e = set_smem(upward_kernel<OTV, 4>, smem);                                                 \
            if (e != cudaSuccess) return e;                                                            \
            upward_kernel<OTV, 4><<<nitems, kThreads, smem, st>>>(items, slot_nodes, n1, src_rec,      \
                                                                   fsrc, out, chunk_out);              \
        }                                                                                              \
        break;
    switch (ot) {
        BLTC_UP(0) BLTC_UP(1) BLTC_UP(2) BLTC_UP(3) BLTC_UP(4) BLTC_UP(5) BLTC_UP(6) BLTC_UP(7)
        default: return cudaErrorInvalidValue;
    }
#undef BLTC_UP
    e = cudaGetLastError();
    if (e != cudaSuccess || nred == 0) return e;
    const int len = n1 * n1 * n1 * nc;
    upward_reduce_kernel<<<dim3((len + kThreads - 1) / kThreads, nred), kThreads, 0, st>>>(red, len, chunk_out, out);
    return cudaGetLastError();
}

cudaError_t launch_upward_children(int ot, const C2PItem* items, int nitems, const double* slot_nodes, int degree,
                                   double* charges, cudaStream_t st) {
    if (nitems == 0) return cudaSuccess;
    const int n1 = degree + 1;
    const size_t smem = sizeof(double) * (3 * (size_t)n1 * n1 + 2 * (size_t)n1 * n1 * n1);
    cudaError_t e = cudaSuccess;
#define BLTC_C2P(NCV)                                                                                   \
    e = set_smem(upward_children_kernel<NCV>, smem);                                                    \
    if (e != cudaSuccess) return e;                                                                     \
    upward_children_kernel<NCV><<<nitems, kThreads, smem, st>>>(items, slot_nodes, n1, charges);        \
    break;
    switch (ot) {
        case 0: case 1: BLTC_C2P(1)
        case 2: BLTC_C2P(2)
        case 3: BLTC_C2P(3)
        case 4: BLTC_C2P(4)
        case 5: BLTC_C2P(5)
        case 6: BLTC_C2P(6)
        case 7: BLTC_C2P(7)
        default: return cudaErrorInvalidValue;
    }
#undef BLTC_C2P
    return cudaGetLastError();
}

// kernel<R, OT, SUB, GUARD> dispatch on (ot, subtract, guard); R = kTargetsPerThread
template <template <int, int, bool, bool> class K, typename... Args>
cudaError_t dispatch_pair(int ot, bool subtract, bool guard, size_t smem, int grid, cudaStream_t st, Args... args) {
#define BLTC_GO(RV, OTV, SV, GV)                                                                        \
    {                                                                                                   \
        auto kern = K<RV, OTV, SV, GV>::get();                                                          \
        cudaError_t e = set_smem(kern, smem);                                                           \
        if (e != cudaSuccess) return e;                                                                 \
        kern<<<grid, kPairThreads, smem, st>>>(args...);                                                    \
        return cudaGetLastError();                                                                      \
    }
#define BLTC_SG(RV, OTV)                                                                                \
    if (subtract) { if (guard) BLTC_GO(RV, OTV, true, true) else BLTC_GO(RV, OTV, true, false) }        \
    else { if (guard) BLTC_GO(RV, OTV, false, true) else BLTC_GO(RV, OTV, false, false) }
    switch (ot) {
        case 1: BLTC_SG(kTargetsPerThread, 1)
        case 2: BLTC_SG(kTargetsPerThread, 2)
        case 3: BLTC_SG(kTargetsPerThread, 3)
        case 4: BLTC_SG(kTargetsPerThread, 4)
        case 5: BLTC_SG(kTargetsPerThread, 5)
        case 6: BLTC_SG(kTargetsPerThread, 6)
        case 7: BLTC_SG(kTargetsPerThread, 7)
        default: return cudaErrorInvalidValue;
    }
#undef BLTC_SG
#undef BLTC_GO
}

template <int R, int OT, bool SUB, bool GUARD> struct FarK { static auto get() { return far_kernel<R, OT, SUB, GUARD, kYukawa, 0>; } };
template <int R, int OT, bool SUB, bool GUARD> struct FarK9 { static auto get() { return far_kernel<R, OT, SUB, GUARD, kYukawa, 9>; } };
template <int R, int OT, bool SUB, bool GUARD> struct NearK { static auto get() { return near_kernel<R, OT, SUB, GUARD, kYukawa, false>; } };
template <int R, int OT, bool SUB, bool GUARD> struct NearKZ { static auto get() { return near_kernel<R, OT, SUB, GUARD, kYukawa, true>; } };
// Coulomb: the Gaussian's exponent -r^2/alpha^2 is not bounded by a per-launch test, so the underflow guard is always on
template <int R, int OT, bool SUB, bool GUARD> struct FarKC { static auto get() { return far_kernel<R, OT, SUB, true, kCoulomb, 0>; } };
template <int R, int OT, bool SUB, bool GUARD> struct FarK9C { static auto get() { return far_kernel<R, OT, SUB, true, kCoulomb, 9>; } };
template <int R, int OT, bool SUB, bool GUARD> struct NearKC { static auto get() { return near_kernel<R, OT, SUB, true, kCoulomb, false>; } };
template <int R, int OT, bool SUB, bool GUARD> struct NearKCZ { static auto get() { return near_kernel<R, OT, SUB, true, kCoulomb, true>; } };

cudaError_t launch_far(int kind, int ot, bool subtract, bool guard, const WorkItem* items, int nitems, const int32_t* far_slots,
                       const double* slot_nodes, const double* what, const double* fhat, int degree,
                       const double4* tgt_rec, const double* ftgt, const KPar& kp, double* partial,
                       int64_t partial_len, cudaStream_t st) {
    if (nitems == 0) return cudaSuccess;
    if (kind == kCoulomb) {
        if (degree == 8)
            return dispatch_pair<FarK9C>(ot, subtract, true, far_smem_bytes(ot), nitems, st, items, far_slots, slot_nodes,
                                         what, fhat, degree + 1, tgt_rec, ftgt, kp, partial, partial_len);
        return dispatch_pair<FarKC>(ot, subtract, true, far_smem_bytes(ot), nitems, st, items, far_slots, slot_nodes,
                                    what, fhat, degree + 1, tgt_rec, ftgt, kp, partial, partial_len);
    }
    if (degree == 8)          // the paper's n = 8: grid size known at compile time
        return dispatch_pair<FarK9>(ot, subtract, guard, far_smem_bytes(ot), nitems, st, items, far_slots, slot_nodes,
                                    what, fhat, degree + 1, tgt_rec, ftgt, kp, partial, partial_len);
    return dispatch_pair<FarK>(ot, subtract, guard, far_smem_bytes(ot), nitems, st, items, far_slots, slot_nodes,
                               what, fhat, degree + 1, tgt_rec, ftgt, kp, partial, partial_len);
}

cudaError_t launch_near(int kind, int ot, bool subtract, bool guard, bool all_zero_safe, const WorkItem* items, int nitems,
                        const Range* ranges, const double4* src_rec, const double* fsrc, const double4* tgt_rec,
                        const double* ftgt, const KPar& kp, double* partial, int64_t partial_len,
                        cudaStream_t st) {
    if (nitems == 0) return cudaSuccess;
#define BLTC_NEAR(K, G) dispatch_pair<K>(ot, subtract, G, near_smem_bytes(ot), nitems, st, items, ranges, src_rec, fsrc, \
                                         tgt_rec, ftgt, kp, partial, partial_len)
    if (kind == kCoulomb) return all_zero_safe ? BLTC_NEAR(NearKCZ, true) : BLTC_NEAR(NearKC, true);
    return all_zero_safe ? BLTC_NEAR(NearKZ, guard) : BLTC_NEAR(NearK, guard);
#undef BLTC_NEAR
}

cudaError_t launch_epilogue(int ot, bool subtract, int nbatch, const int32_t* b_begin, const int32_t* b_count,
                            const int64_t* b_partial_base, const int32_t* b_nseg, const double* partial,
                            int64_t partial_len, const double* ftgt, const EpiPar& kp, const int32_t* perm,
                            const OutSet& out, int64_t stride, int o0, cudaStream_t st) {
    if (nbatch == 0) return cudaSuccess;
#define BLTC_EPI(OTV)                                                                                  \
    case OTV:                                                                                          \
        if (subtract) epilogue_kernel<OTV, true><<<nbatch, kThreads, 0, st>>>(b_begin, b_count,        \
            b_partial_base, b_nseg, partial, partial_len, ftgt, kp, perm, out, stride, o0);            \
        else epilogue_kernel<OTV, false><<<nbatch, kThreads, 0, st>>>(b_begin, b_count,                \
            b_partial_base, b_nseg, partial, partial_len, ftgt, kp, perm, out, stride, o0);            \
        break;
    switch (ot) {
        BLTC_EPI(1) BLTC_EPI(2) BLTC_EPI(3) BLTC_EPI(4) BLTC_EPI(5) BLTC_EPI(6) BLTC_EPI(7)
        default: return cudaErrorInvalidValue;
    }
#undef BLTC_EPI
    return cudaGetLastError();
}

cudaError_t launch_fp64_probe(int form, int iters, float* ms, double* dfma_count, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    double* sink = nullptr;
    e = cudaMalloc(&sink, sizeof(double));
    if (e != cudaSuccess) return e;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int grid = sms * 8;
    auto run = [&](int n) {
        if (form == 0) fp64_probe_kernel<0><<<grid, kThreads, 0, st>>>(n, 1.0, sink);
        else fp64_probe_kernel<1><<<grid, kThreads, 0, st>>>(n, 1.0, sink);
    };
    run(4);                                                              // warm-up
    cudaEventRecord(a, st);
    run(iters);
    cudaEventRecord(b, st);
    e = cudaEventSynchronize(b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, a, b);
    *dfma_count = (double)grid * kThreads * (double)iters * 64.0 * 8.0;
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(sink);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace bltc
