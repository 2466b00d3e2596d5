// plan_device.cu -- step a0 on the GPU (SURVEY.md 8(f) NEXT-4a): the source-cluster tree and the per-batch MAC
// interaction lists of Algorithm 3 built by kernels, so that bltc_create no longer
// scales with the host ("the precompute stage ... scales worst ... due to some serial computation").
//
// The result is the SAME plan as plan_host.cpp's (and the CPU oracle's), cluster for cluster and entry for entry:
//   * tree: level-synchronous.  Per level, (a) exact min/max boxes of the new clusters by a warp-segmented
//     reduction, (b) the leaf / split decisions of readings R4-R5 taken on the HOST from those boxes with the very
//     expressions of plan_host.cpp (a few thousand clusters: microseconds), (c) a key (segment << 3 | child code)
//     per point and one STABLE radix sort of (key, point) pairs -- the stable partition of every cluster of the
//     level at once, children in code order, finished leaves untouched -- (d) a run-length encode of the sorted
//     keys = the next level's segments.  Clusters are renumbered to DFS pre-order at the end.
//   * lists: one thread per batch walks the pre-order tree with skip pointers (no stack), first counting, then
//     writing its far / near lists in traversal order.  Centres and radii come from the host (plan_host.cpp's
//     expressions); the device evaluates only R = |c_B - c_C| and (r_B + r_C) < theta R with round-to-nearest
//     intrinsics in the written order, so every decision is bitwise the host's (readings R6, R8, R10).
// cub::DeviceRadixSort / DeviceRunLengthEncode (CUDA toolkit headers) serve as the sort and encode primitives of
// this setup step; nothing here is on the per-convolution path.
#include "plan_device.cuh"

#include <cub/cub.cuh>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <stdexcept>
#include <vector>

namespace bltc {
namespace {

constexpr double kSqrt2 = 1.4142135623730951;

#define BLTC_DEV_TRY(call)                                  \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return e__;                 \
    } while (0)

// Temporary of one plan build, from the library's stream-ordered pool (a cudaMalloc / cudaFree pair per temporary
// made bltc_create depend on the host and the driver's state: GPUTEST_r02 read 48 ms for the lists stage on one box
// and 5 ms on another).  The builders run on ONE stream, given once per thread before the first alloc.
thread_local cudaStream_t t_scratch_stream = nullptr;
template <typename T>
struct Scratch {
    T* p = nullptr;
    ~Scratch() { release(); }
    void release() { if (p) cudaFreeAsync(p, t_scratch_stream); p = nullptr; }
    cudaError_t alloc(size_t n) {
        release();
        return pool_alloc_async(reinterpret_cast<void**>(&p), (n ? n : 1) * sizeof(T), t_scratch_stream);
    }
};

// order-preserving map double -> uint64 (exact for min/max by integer atomics)
__device__ __forceinline__ unsigned long long enc(double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
inline double dec(unsigned long long e) {
    const unsigned long long b = (e >> 63) ? (e & 0x7fffffffffffffffull) : ~e;
    double v;
    memcpy(&v, &b, sizeof v);
    return v;
}

__global__ void iota_kernel(int32_t* perm, int32_t* ord, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { perm[i] = (int32_t)i; ord[i] = 0; }
}

// (a) boxes of the segments with box_slot[seg] >= 0: lo/hi[slot][3] as encoded uint64, initialised to ~0 / 0.
// Positions are sorted by segment, so a warp holds a few contiguous runs: inclusive segmented scan by shuffles,
// the last lane of each run issues the atomics.
__global__ void __launch_bounds__(256)
bbox_kernel(const double* __restrict__ coords, int64_t n, const int32_t* __restrict__ perm,
            const int32_t* __restrict__ ord, const int32_t* __restrict__ box_slot,
            unsigned long long* __restrict__ lo, unsigned long long* __restrict__ hi) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int seg = -1, slot = -1;
    unsigned long long mn[3] = {~0ull, ~0ull, ~0ull}, mx[3] = {0ull, 0ull, 0ull};
    if (i < n) {
        seg = ord[i];
        slot = box_slot[seg];
        if (slot >= 0) {
            const int64_t p = perm[i];
#pragma unroll
            for (int d = 0; d < 3; ++d) mn[d] = mx[d] = enc(coords[(int64_t)d * n + p]);
        }
    }
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        const int oseg = __shfl_up_sync(0xffffffffu, seg, s);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const unsigned long long a = __shfl_up_sync(0xffffffffu, mn[d], s);
            const unsigned long long b = __shfl_up_sync(0xffffffffu, mx[d], s);
            if (lane >= s && oseg == seg) { mn[d] = a < mn[d] ? a : mn[d]; mx[d] = b > mx[d] ? b : mx[d]; }
        }
    }
    const int nseg = __shfl_down_sync(0xffffffffu, seg, 1);
    const bool last = lane == 31 || nseg != seg;
    if (slot >= 0 && last) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            atomicMin(lo + (size_t)slot * 3 + d, mn[d]);
            atomicMax(hi + (size_t)slot * 3 + d, mx[d]);
        }
    }
}

// (c) key = segment << 3 | child code (bit0 x, bit1 y, bit2 z; "upper child iff coord > mid", reading R5);
// segments that are not being split (cut mask 0) get code 0 and so keep their order.
struct SegSplit { double mid[3]; int32_t cut; int32_t pad; };
__global__ void __launch_bounds__(256)
key_kernel(const double* __restrict__ coords, int64_t n, const int32_t* __restrict__ perm,
           const int32_t* __restrict__ ord, const SegSplit* __restrict__ split, uint32_t* __restrict__ key) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int seg = ord[i];
    const SegSplit s = split[seg];
    uint32_t code = 0;
    if (s.cut) {
        const int64_t p = perm[i];
        if ((s.cut & 1) && coords[p] > s.mid[0]) code |= 1;
        if ((s.cut & 2) && coords[n + p] > s.mid[1]) code |= 2;
        if ((s.cut & 4) && coords[2 * n + p] > s.mid[2]) code |= 4;
    }
    key[i] = ((uint32_t)seg << 3) | code;
}

// (d') segment index of every position from the segment begins (ascending), by binary search
__global__ void __launch_bounds__(256)
ord_kernel(const int32_t* __restrict__ seg_begin, int nseg, int64_t n, int32_t* __restrict__ ord) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int lo = 0, hi = nseg;                 // last segment with begin <= i
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int64_t)seg_begin[mid] <= i) lo = mid; else hi = mid;
    }
    ord[i] = lo;
}

}  // namespace

cudaError_t build_tree_device(Tree& t, const double* d_coords, int64_t n, int64_t max_leaf, int32_t* d_perm,
                              cudaStream_t st) {
    if (n >= (int64_t)1 << 28) return cudaErrorInvalidValue;      // keys are segment << 3 in 32 bits
    t_scratch_stream = st;
    t.cl.clear(); t.perm.clear(); t.leaves.clear();
    const unsigned grid = (unsigned)((n + 255) / 256);
    Scratch<uint32_t> key0, key1, run_key;
    Scratch<int32_t> val1, ord, run_cnt, num_runs, box_slot, seg_begin;
    Scratch<unsigned long long> lo, hi;
    Scratch<SegSplit> split;
    Scratch<unsigned char> temp;
    BLTC_DEV_TRY(key0.alloc(n)); BLTC_DEV_TRY(key1.alloc(n)); BLTC_DEV_TRY(val1.alloc(n));
    BLTC_DEV_TRY(ord.alloc(n)); BLTC_DEV_TRY(run_key.alloc(n)); BLTC_DEV_TRY(run_cnt.alloc(n));
    BLTC_DEV_TRY(num_runs.alloc(1));
    size_t seg_cap = 0;                                             // capacity of the per-segment device tables
    auto ensure_seg = [&](size_t need) -> cudaError_t {
        if (need <= seg_cap) return cudaSuccess;
        seg_cap = std::max(need, 2 * seg_cap + 1024);
        BLTC_DEV_TRY(box_slot.alloc(seg_cap)); BLTC_DEV_TRY(seg_begin.alloc(seg_cap));
        BLTC_DEV_TRY(lo.alloc(3 * seg_cap)); BLTC_DEV_TRY(hi.alloc(3 * seg_cap)); BLTC_DEV_TRY(split.alloc(seg_cap));
        return cudaSuccess;
    };
    size_t temp_bytes = 0;
    {
        cub::DoubleBuffer<uint32_t> dk(key0.p, key1.p);
        cub::DoubleBuffer<int32_t> dv(d_perm, val1.p);
        size_t a = 0, b = 0;
        BLTC_DEV_TRY(cub::DeviceRadixSort::SortPairs(nullptr, a, dk, dv, (int)n, 0, 32, st));
        BLTC_DEV_TRY(cub::DeviceRunLengthEncode::Encode(nullptr, b, key0.p, run_key.p, run_cnt.p, num_runs.p, (int)n, st));
        temp_bytes = std::max(a, b);
        BLTC_DEV_TRY(temp.alloc(temp_bytes));
    }
    // the permutation lives in a double buffer; `cur` is the half that holds it
    int32_t* vals[2] = {d_perm, val1.p};
    int cur = 0;
    iota_kernel<<<grid, 256, 0, st>>>(vals[0], ord.p, n);
    BLTC_DEV_TRY(cudaGetLastError());

    // host-side level state: segments in position order
    struct Seg { int32_t begin, end; int cluster; bool active; };
    std::vector<Seg> segs(1, Seg{0, (int32_t)n, 0, false});
    std::vector<int> fresh(1, 0);                                   // segments whose cluster was created in this level
    t.cl.emplace_back();
    t.cl[0].begin = 0; t.cl[0].end = n; t.cl[0].parent = -1; t.cl[0].level = 0;
    std::vector<int32_t> h_slot, h_begin, h_cnt;
    std::vector<uint32_t> h_key;
    std::vector<unsigned long long> h_lo, h_hi;
    std::vector<SegSplit> h_split;
    for (;;) {
        const size_t ns = segs.size();
        BLTC_DEV_TRY(ensure_seg(ns));
        // (a) boxes of the fresh clusters
        h_slot.assign(ns, -1);
        for (size_t f = 0; f < fresh.size(); ++f) h_slot[fresh[f]] = (int32_t)f;
        BLTC_DEV_TRY(cudaMemcpyAsync(box_slot.p, h_slot.data(), ns * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        BLTC_DEV_TRY(cudaMemsetAsync(lo.p, 0xff, fresh.size() * 3 * sizeof(unsigned long long), st));
        BLTC_DEV_TRY(cudaMemsetAsync(hi.p, 0x00, fresh.size() * 3 * sizeof(unsigned long long), st));
        bbox_kernel<<<grid, 256, 0, st>>>(d_coords, n, vals[cur], ord.p, box_slot.p, lo.p, hi.p);
        BLTC_DEV_TRY(cudaGetLastError());
        h_lo.resize(fresh.size() * 3); h_hi.resize(fresh.size() * 3);
        BLTC_DEV_TRY(cudaMemcpyAsync(h_lo.data(), lo.p, h_lo.size() * 8, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaMemcpyAsync(h_hi.data(), hi.p, h_hi.size() * 8, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaStreamSynchronize(st));
        // (b) decisions, exactly plan_host.cpp's make_cluster (R4, R5)
        h_split.assign(ns, SegSplit{{0, 0, 0}, 0, 0});
        size_t nactive = 0;
        for (size_t f = 0; f < fresh.size(); ++f) {
            Seg& S = segs[fresh[f]];
            Cluster& C = t.cl[S.cluster];
            for (int d = 0; d < 3; ++d) { C.lo[d] = dec(h_lo[f * 3 + d]); C.hi[d] = dec(h_hi[f * 3 + d]); }
            S.active = false;
            if (C.end - C.begin <= max_leaf) continue;                    // R4: leaf iff count <= N_L
            double ext[3], longest = 0.0;
            for (int d = 0; d < 3; ++d) {
                ext[d] = C.hi[d] - C.lo[d];
                longest = ext[d] > longest ? ext[d] : longest;
            }
            SegSplit sp{{0, 0, 0}, 0, 0};
            for (int d = 0; d < 3; ++d) {                                 // R5: aspect-ratio rule sqrt(2)
                if (ext[d] > 0.0 && ext[d] * kSqrt2 >= longest) sp.cut |= 1 << d;
                sp.mid[d] = 0.5 * (C.lo[d] + C.hi[d]);
            }
            if (sp.cut == 0) continue;                                    // all particles coincide
            S.active = true; ++nactive;
            h_split[fresh[f]] = sp;
        }
        if (nactive == 0) break;
        // (c) keys, (d) stable sort of (key, point), run-length encode
        BLTC_DEV_TRY(cudaMemcpyAsync(split.p, h_split.data(), ns * sizeof(SegSplit), cudaMemcpyHostToDevice, st));
        key_kernel<<<grid, 256, 0, st>>>(d_coords, n, vals[cur], ord.p, split.p, key0.p);
        BLTC_DEV_TRY(cudaGetLastError());
        int bits = 3;
        while (((size_t)1 << (bits - 3)) < ns) ++bits;
        cub::DoubleBuffer<uint32_t> dk(key0.p, key1.p);
        cub::DoubleBuffer<int32_t> dv(vals[cur], vals[cur ^ 1]);
        size_t tb = temp_bytes;
        BLTC_DEV_TRY(cub::DeviceRadixSort::SortPairs(temp.p, tb, dk, dv, (int)n, 0, bits, st));
        cur = dv.Current() == vals[0] ? 0 : 1;
        tb = temp_bytes;
        BLTC_DEV_TRY(cub::DeviceRunLengthEncode::Encode(temp.p, tb, dk.Current(), run_key.p, run_cnt.p, num_runs.p, (int)n, st));
        // one read-back per level: the run count together with the runs themselves.  A segment yields at most 8 runs
        // (its child codes) and there are no more runs than points, so the copy is sized by that bound instead of
        // waiting for the count first (that cost a second host round trip per tree level).
        int32_t nr = 0;
        const size_t run_cap = (size_t)std::min<int64_t>(n, 8 * (int64_t)ns);
        h_key.resize(run_cap); h_cnt.resize(run_cap);
        BLTC_DEV_TRY(cudaMemcpyAsync(&nr, num_runs.p, sizeof nr, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaMemcpyAsync(h_key.data(), run_key.p, run_cap * 4, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaMemcpyAsync(h_cnt.data(), run_cnt.p, run_cap * 4, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaStreamSynchronize(st));
        if (nr < 0 || (size_t)nr > run_cap) return cudaErrorUnknown;
        h_key.resize(nr); h_cnt.resize(nr);
        // next level's segments = the runs; the runs of an active segment are its children in code order
        std::vector<Seg> next;
        next.reserve(nr);
        fresh.clear();
        int32_t at = 0;
        for (int32_t r = 0; r < nr;) {
            const int seg = (int)(h_key[r] >> 3);
            int32_t r1 = r;
            while (r1 < nr && (int)(h_key[r1] >> 3) == seg) ++r1;
            const Seg& S = segs[seg];
            const int live = r1 - r;
            if (!S.active || live < 2) {               // finished leaf, or the midpoint rounded onto a face: stays a leaf
                next.push_back(Seg{S.begin, S.end, S.cluster, false});
                at = S.end;
            } else {
                for (int32_t q = r; q < r1; ++q) {     // empty children dropped
                    const int id = (int)t.cl.size();
                    t.cl.emplace_back();
                    Cluster& C = t.cl.back();
                    C.begin = at; C.end = at + h_cnt[q]; C.parent = S.cluster; C.level = t.cl[S.cluster].level + 1;
                    Cluster& P = t.cl[S.cluster];
                    P.child[P.nchild++] = id;
                    fresh.push_back((int)next.size());
                    next.push_back(Seg{(int32_t)C.begin, (int32_t)C.end, id, false});
                    at += h_cnt[q];
                }
            }
            r = r1;
        }
        segs.swap(next);
        if (fresh.empty()) break;
        BLTC_DEV_TRY(ensure_seg(segs.size()));
        h_begin.resize(segs.size());
        for (size_t s = 0; s < segs.size(); ++s) h_begin[s] = segs[s].begin;
        BLTC_DEV_TRY(cudaMemcpyAsync(seg_begin.p, h_begin.data(), h_begin.size() * 4, cudaMemcpyHostToDevice, st));
        ord_kernel<<<grid, 256, 0, st>>>(seg_begin.p, (int)segs.size(), n, ord.p);
        BLTC_DEV_TRY(cudaGetLastError());
    }
    if (cur != 0) BLTC_DEV_TRY(cudaMemcpyAsync(d_perm, vals[cur], (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    BLTC_DEV_TRY(cudaStreamSynchronize(st));

    // breadth-first creation order -> DFS pre-order (children in code order), as plan_host.cpp / the oracle number them
    const int ncl = (int)t.cl.size();
    std::vector<int> newid(ncl, -1), order;
    order.reserve(ncl);
    {
        std::vector<int> stack(1, 0);
        while (!stack.empty()) {
            const int c = stack.back(); stack.pop_back();
            newid[c] = (int)order.size();
            order.push_back(c);
            for (int q = t.cl[c].nchild - 1; q >= 0; --q) stack.push_back(t.cl[c].child[q]);
        }
    }
    std::vector<Cluster> sorted(ncl);
    for (int i = 0; i < ncl; ++i) {
        Cluster C = t.cl[order[i]];
        C.parent = C.parent < 0 ? -1 : newid[C.parent];
        for (int q = 0; q < C.nchild; ++q) C.child[q] = newid[C.child[q]];
        sorted[i] = C;
    }
    t.cl.swap(sorted);
    for (int i = 0; i < ncl; ++i) if (t.cl[i].nchild == 0) t.leaves.push_back(i);    // pre-order = position order
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------ lists
namespace {

struct MacCluster { double c[3]; double r; int32_t count, skip, nchild, flat; };   // flat: a box extent is 0 (R8)
struct MacBatch { double c[3]; double r; };

// Algorithm 3 ComputePotential, decision part (text PAPER.md:434), one thread per batch.
// FILL = false: counts;  FILL = true: writes the lists at far_ptr / near_ptr (relative to the first batch).
template <bool FILL>
__global__ void __launch_bounds__(128)
mac_kernel(const MacCluster* __restrict__ cl, int ncl, const MacBatch* __restrict__ bt, int b0, int nb, double theta,
           int P, int32_t* __restrict__ nfar, int32_t* __restrict__ nnear, long long* __restrict__ near_src,
           const long long* __restrict__ far_ptr, const long long* __restrict__ near_ptr,
           int32_t* __restrict__ far_idx, int32_t* __restrict__ near_idx) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nb) return;
    const int b = b0 + t;
    const MacBatch B = bt[b];
    int32_t nf = 0, nn = 0;
    long long ns = 0;
    long long fo = FILL ? far_ptr[b] - far_ptr[b0] : 0, no = FILL ? near_ptr[b] - near_ptr[b0] : 0;
    int c = 0;
    while (c < ncl) {
        const MacCluster C = cl[c];
        const double dx = __dsub_rn(B.c[0], C.c[0]), dy = __dsub_rn(B.c[1], C.c[1]), dz = __dsub_rn(B.c[2], C.c[2]);
        const double R = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
        const bool separated = __dadd_rn(B.r, C.r) < __dmul_rn(theta, R);          // Eq. (36) left, R6
        const bool big = P < C.count && !C.flat;                                  // Eq. (36) right, R8
        if (separated && big) {
            if (FILL) far_idx[fo + nf] = c;
            ++nf; c = C.skip;
        } else if (!separated && C.nchild != 0) {
            c = c + 1;                                                            // descend: first child
        } else {                                                                  // leaf, or R10: whole cluster direct
            if (FILL) near_idx[no + nn] = c;
            ++nn; ns += C.count; c = C.skip;
        }
    }
    if (!FILL) { nfar[b] = nf; nnear[b] = nn; near_src[b] = ns; }
}

inline double half_diag(const double* lo, const double* hi) {
    const double ex = hi[0] - lo[0], ey = hi[1] - lo[1], ez = hi[2] - lo[2];
    return 0.5 * std::sqrt((ex * ex + ey * ey) + ez * ez);
}

}  // namespace

cudaError_t build_lists_device(HostPlan& p, int shard_rank, int shard_world, cudaStream_t st) {
    const int ncl = (int)p.src.cl.size(), nb = (int)p.b_begin.size();
    t_scratch_stream = st;
    std::vector<MacCluster> hc(ncl);
    {   // skip pointers: the cluster after c's subtree in pre-order
        std::vector<int> last(ncl);
        for (int c = ncl - 1; c >= 0; --c) {
            const Cluster& C = p.src.cl[c];
            last[c] = C.nchild ? last[C.child[C.nchild - 1]] : c;
        }
        for (int c = 0; c < ncl; ++c) {
            const Cluster& C = p.src.cl[c];
            MacCluster& M = hc[c];
            for (int d = 0; d < 3; ++d) M.c[d] = 0.5 * (C.lo[d] + C.hi[d]);
            M.r = half_diag(C.lo, C.hi);
            M.count = (int32_t)(C.end - C.begin); M.skip = last[c] + 1; M.nchild = C.nchild;
            M.flat = (C.hi[0] == C.lo[0] || C.hi[1] == C.lo[1] || C.hi[2] == C.lo[2]) ? 1 : 0;
        }
    }
    std::vector<MacBatch> hb(nb);
    for (int b = 0; b < nb; ++b) {
        for (int d = 0; d < 3; ++d) hb[b].c[d] = 0.5 * (p.b_lo[3 * b + d] + p.b_hi[3 * b + d]);
        hb[b].r = half_diag(&p.b_lo[3 * b], &p.b_hi[3 * b]);
    }
    Scratch<MacCluster> d_cl; Scratch<MacBatch> d_bt;
    Scratch<int32_t> d_nfar, d_nnear, d_far, d_near;
    Scratch<long long> d_src, d_fptr, d_nptr;
    BLTC_DEV_TRY(d_cl.alloc(ncl)); BLTC_DEV_TRY(d_bt.alloc(nb));
    BLTC_DEV_TRY(d_nfar.alloc(nb)); BLTC_DEV_TRY(d_nnear.alloc(nb)); BLTC_DEV_TRY(d_src.alloc(nb));
    BLTC_DEV_TRY(cudaMemcpyAsync(d_cl.p, hc.data(), (size_t)ncl * sizeof(MacCluster), cudaMemcpyHostToDevice, st));
    BLTC_DEV_TRY(cudaMemcpyAsync(d_bt.p, hb.data(), (size_t)nb * sizeof(MacBatch), cudaMemcpyHostToDevice, st));
    // cost pass over ALL batches (cheap): list lengths and evaluation counts, which also fix the shard cuts
    mac_kernel<false><<<(nb + 127) / 128, 128, 0, st>>>(d_cl.p, ncl, d_bt.p, 0, nb, p.theta, p.P, d_nfar.p, d_nnear.p,
                                                         d_src.p, nullptr, nullptr, nullptr, nullptr);
    BLTC_DEV_TRY(cudaGetLastError());
    std::vector<int32_t> nfar(nb), nnear(nb);
    std::vector<long long> nsrc(nb);
    BLTC_DEV_TRY(cudaMemcpyAsync(nfar.data(), d_nfar.p, (size_t)nb * 4, cudaMemcpyDeviceToHost, st));
    BLTC_DEV_TRY(cudaMemcpyAsync(nnear.data(), d_nnear.p, (size_t)nb * 4, cudaMemcpyDeviceToHost, st));
    BLTC_DEV_TRY(cudaMemcpyAsync(nsrc.data(), d_src.p, (size_t)nb * 8, cudaMemcpyDeviceToHost, st));
    BLTC_DEV_TRY(cudaStreamSynchronize(st));
    p.far_ptr.assign(nb + 1, 0); p.near_ptr.assign(nb + 1, 0);
    std::vector<int64_t> b_far_evals(nb), b_near_evals(nb);
    for (int b = 0; b < nb; ++b) {
        p.far_ptr[b + 1] = p.far_ptr[b] + nfar[b]; p.near_ptr[b + 1] = p.near_ptr[b] + nnear[b];
        const int64_t nt = p.b_end[b] - p.b_begin[b];
        b_far_evals[b] = nt * p.P * nfar[b];
        b_near_evals[b] = nt * (int64_t)nsrc[b];
    }
    plan_set_shard(p, b_far_evals, b_near_evals, shard_rank, shard_world);
    // fill pass: this rank's batches only
    const int B0 = p.shard_b0, B1 = p.shard_b1;
    p.far_idx.assign((size_t)p.far_ptr[nb], 0); p.near_idx.assign((size_t)p.near_ptr[nb], 0);
    p.lists_b0 = B0; p.lists_b1 = B1;
    if (B1 > B0) {
        const size_t nf = (size_t)(p.far_ptr[B1] - p.far_ptr[B0]), nn = (size_t)(p.near_ptr[B1] - p.near_ptr[B0]);
        BLTC_DEV_TRY(d_far.alloc(nf)); BLTC_DEV_TRY(d_near.alloc(nn));
        BLTC_DEV_TRY(d_fptr.alloc(nb + 1)); BLTC_DEV_TRY(d_nptr.alloc(nb + 1));
        static_assert(sizeof(long long) == sizeof(int64_t), "CSR pointers are 64-bit");
        BLTC_DEV_TRY(cudaMemcpyAsync(d_fptr.p, p.far_ptr.data(), (size_t)(nb + 1) * 8, cudaMemcpyHostToDevice, st));
        BLTC_DEV_TRY(cudaMemcpyAsync(d_nptr.p, p.near_ptr.data(), (size_t)(nb + 1) * 8, cudaMemcpyHostToDevice, st));
        mac_kernel<true><<<(B1 - B0 + 127) / 128, 128, 0, st>>>(d_cl.p, ncl, d_bt.p, B0, B1 - B0, p.theta, p.P, nullptr,
                                                                 nullptr, nullptr, d_fptr.p, d_nptr.p, d_far.p, d_near.p);
        BLTC_DEV_TRY(cudaGetLastError());
        if (nf) BLTC_DEV_TRY(cudaMemcpyAsync(p.far_idx.data() + p.far_ptr[B0], d_far.p, nf * 4, cudaMemcpyDeviceToHost, st));
        if (nn) BLTC_DEV_TRY(cudaMemcpyAsync(p.near_idx.data() + p.near_ptr[B0], d_near.p, nn * 4, cudaMemcpyDeviceToHost, st));
        BLTC_DEV_TRY(cudaStreamSynchronize(st));
    }
    return cudaSuccess;
}

}  // namespace bltc
