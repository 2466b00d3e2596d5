// api.cu -- the C ABI of libbltc (include/bltc.h): argument checking, host<->device staging,
// device state of a plan, and the launch sequence of one convolution.  No arithmetic of the
// method lives here; it is all in kernels.cu (device) and plan_host.cpp (tree and lists).
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/bltc.h"
#include "gi_kernels.cuh"
#include "kernels.cuh"
#include "plan_device.cuh"
#include "plan_host.hpp"

using namespace bltc;

namespace {

thread_local std::string g_err;

// NVTX range (tracing) around every stage of bltc_create and every phase of a convolution: a timeline
// tool shows them by name; without one attached the calls are no-ops.
struct Nvtx {
    explicit Nvtx(const char* name) { nvtxRangePushA(name); }
    ~Nvtx() { nvtxRangePop(); }
};

int fail(int code, const std::string& msg) { g_err = msg; return code; }

#define BLTC_CUDA(call)                                                                        \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess) {                                                              \
            cudaGetLastError();                                                                \
            return fail(e__ == cudaErrorMemoryAllocation ? BLTC_ENOMEM : BLTC_ECUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                  \
        }                                                                                      \
    } while (0)

// true if the device can dereference p (device or managed memory)
bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <typename T>
struct DevBuf {
    T* p = nullptr;
    size_t n = 0;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t ensure(size_t count) {
        if (count <= n && p) return cudaSuccess;
        if (p) { cudaFree(p); p = nullptr; n = 0; }
        if (count == 0) count = 1;
        cudaError_t e = cudaMalloc(&p, count * sizeof(T));
        if (e == cudaSuccess) n = count;
        return e;
    }
    cudaError_t upload(const std::vector<T>& v) {
        cudaError_t e = ensure(v.size());
        if (e != cudaSuccess || v.empty()) return e;
        return cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
    }
};

// Stream-ordered temporary (direct_convolve and host staging): freed on the stream.
struct TempBuf {
    void* p = nullptr;
    cudaStream_t st = nullptr;
    ~TempBuf() { if (p) cudaFreeAsync(p, st); }
    cudaError_t alloc(size_t bytes, cudaStream_t s) {
        st = s;
        cudaMemPool_t pool = library_pool();
        if (!pool) return cudaMallocAsync(&p, bytes ? bytes : 1, s);
        return cudaMallocFromPoolAsync(&p, bytes ? bytes : 1, pool, s);
    }
    // The library's OWN stream-ordered pool, one per device, created on first use and kept for the life of the
    // process.  Its release threshold is unlimited, so the staging buffers of one call are reused by the next
    // instead of going back to the driver at every synchronisation (a real cudaMalloc/cudaFree, ~ms per call);
    // the device's default pool -- the caller's -- is left as it is.
    static cudaMemPool_t library_pool() {
        static std::mutex mu;
        static cudaMemPool_t pools[64] = {};
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return nullptr; }
        std::lock_guard<std::mutex> lock(mu);
        if (!pools[dev]) {
            cudaMemPoolProps props = {};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            cudaMemPool_t pool = nullptr;
            if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            cudaGetLastError();
            pools[dev] = pool;
        }
        return pools[dev];
    }
    template <typename T> T* as() const { return static_cast<T*>(p); }
};

// Returns a device-readable view of `src` (count doubles): src itself, or a staged copy.
cudaError_t stage_in(const double* src, size_t count, TempBuf& tmp, cudaStream_t st, const double** dev) {
    if (!src) { *dev = nullptr; return cudaSuccess; }
    if (is_device_ptr(src)) { *dev = src; return cudaSuccess; }
    cudaError_t e = tmp.alloc(count * sizeof(double), st);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(tmp.p, src, count * sizeof(double), cudaMemcpyHostToDevice, st);
    *dev = tmp.as<double>();
    return e;
}

// Orbitals are processed in groups ("tiles") of <= kMaxOT = the register tile of the pair kernels, sizes as equal as
// possible.  The number of tiles minimises a per-orbital cost measured on B200 (near + far kernel time per orbital and
// pair at tile width w, relative units): wider tiles share the geometry / rsqrt of a pair among more
// orbitals (7 is what fits in 128 registers with two targets per thread).  BLTC_ORBITAL_TILE = 1 .. kMaxOT forces a maximum width
// (tuning runs).
static_assert(kMaxOT == BLTC_MAX_ORBITAL_TILE, "include/bltc.h states the widest orbital tile");
std::vector<int> orbital_groups(int n_orb) {
    // ms per orbital of one near + one far launch on the configs[1] mesh at tile widths 1..7 (profiles/r02f, r02h)
    static const double kCost[kMaxOT + 1] = {0.0, 116.8, 84.1, 75.0, 70.0, 68.0, 66.6, 65.6};
    auto split = [n_orb](int ng) {
        std::vector<int> g(ng, n_orb / ng);
        for (int i = 0; i < n_orb % ng; ++i) ++g[i];
        return g;
    };
    if (const char* e = std::getenv("BLTC_ORBITAL_TILE")) {
        const int v = std::atoi(e);
        if (v >= 1 && v <= kMaxOT) return split((n_orb + v - 1) / v);
    }
    int best_ng = (n_orb + kMaxOT - 1) / kMaxOT;
    double best = 1e300;
    for (int ng = best_ng; ng <= n_orb; ++ng) {
        double c = 0.0;
        for (int w : split(ng)) c += kCost[w] * w;
        if (c < best) { best = c; best_ng = ng; }
        if (n_orb / ng < 3) break;                 // narrower tiles only cost more
    }
    return split(best_ng);
}

// direct_convolve has no handle to carry its profiling switch and events: they are per calling thread
thread_local bool g_direct_profiling = false;
thread_local std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_direct_pairs;

}  // namespace

struct bltc_plan_s {
    HostPlan hp;
    bool on_device = false;
    int device = 0;
    double upload_ms = 0, create_ms = 0;
    // static device state
    DevBuf<double4> src_rec, tgt_rec_own;
    const double4* tgt_rec = nullptr;
    DevBuf<int32_t> src_perm, tgt_perm_own;
    const int32_t* tgt_perm = nullptr;
    DevBuf<int32_t> b_begin, b_count, b_nseg, far_slots;
    DevBuf<int64_t> b_partial_base;
    DevBuf<double> slot_nodes, what;
    DevBuf<Range> near_ranges;
    DevBuf<WorkItem> far_items, near_items;
    DevBuf<UpItem> up_items;
    DevBuf<UpReduce> up_reduce;
    DevBuf<C2PItem> c2p_items;
    DevBuf<double> up_chunks;                  // chunk-partial proxy charges (sized for kMaxOT)
    // per-convolve scratch (sized for kMaxOT)
    DevBuf<double> fsrc, ftgt_own, fhat, partial, f_stage, out_stage;
    int last_ot = 0;
    // the scratch above is shared by every call on this handle: a call on another stream waits for the previous one
    cudaEvent_t last_done = nullptr;
    cudaStream_t last_stream = nullptr;
    bool has_last = false;
    // profiling
    bool profiling = false;
    std::vector<cudaEvent_t> events;     // (BLTC_NUM_PHASES + 1) per orbital group
    int events_used = 0;
    ~bltc_plan_s() {
        for (cudaEvent_t e : events) cudaEventDestroy(e);
        if (last_done) cudaEventDestroy(last_done);
    }
};

namespace {

int check_create_args(bltc_handle* h, const double* sources, int64_t N, double theta, int degree,
                      int batch_size, int leaf_size) {
    if (!h) return fail(BLTC_EINVAL, "handle pointer is NULL");
    if (!sources) return fail(BLTC_EINVAL, "sources is NULL");
    if (N <= 0 || N > 2000000000LL) return fail(BLTC_EINVAL, "N must be in [1, 2e9]");
    if (!(theta >= 0.0) || !(theta < 1.0)) return fail(BLTC_EINVAL, "theta must satisfy 0 <= theta < 1");
    if (degree < 1 || degree > 20) return fail(BLTC_EINVAL, "interp_degree must be in [1, 20]");
    if (batch_size < 1 || leaf_size < 1) return fail(BLTC_EINVAL, "batch_size and leaf_size must be >= 1");
    return BLTC_OK;
}

int build_plan_guarded(bltc_plan_s* pl, const double* targets, const double* sources, int64_t N,
                       double theta, int degree, int batch_size, int leaf_size, int sms, int rank, int world,
                       bool upward_children = false) {
    try {
        build_host_plan(pl->hp, targets, sources, N, theta, degree, batch_size, leaf_size, sms, rank, world,
                        upward_children);
    } catch (const std::bad_alloc&) {
        return fail(BLTC_ENOMEM, "host allocation failed while building the plan");
    } catch (const std::exception& e) {
        return fail(BLTC_EINVAL, e.what());
    }
    return BLTC_OK;
}

// A device-built plan keeps its permutations on the device only; the host copies are made on first use.
cudaError_t ensure_host_perm(bltc_plan_s* h) {
    HostPlan& hp = h->hp;
    auto fetch = [&](std::vector<int64_t>& dst, const int32_t* src) -> cudaError_t {
        if (!dst.empty() || !src) return cudaSuccess;
        std::vector<int32_t> tmp((size_t)hp.N);
        cudaError_t e = cudaMemcpy(tmp.data(), src, tmp.size() * sizeof(int32_t), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return e;
        dst.assign(tmp.begin(), tmp.end());
        return cudaSuccess;
    };
    if (!h->on_device) return cudaSuccess;
    cudaError_t e = fetch(hp.src.perm, h->src_perm.p);
    if (e == cudaSuccess && !hp.shared_order) e = fetch(hp.tgt.perm, h->tgt_perm_own.p);
    return e;
}

std::vector<int32_t> to_i32(const std::vector<int64_t>& v) {
    std::vector<int32_t> o(v.size());
    for (size_t i = 0; i < v.size(); ++i) o[i] = (int32_t)v[i];
    return o;
}

}  // namespace

extern "C" {

const char* bltc_last_error(void) { return g_err.c_str(); }
const char* bltc_version(void) { return "bltc-b200 0.2 (sm_100a)"; }

int bltc_orbital_tiles(int n_orb, int* widths, int capacity) {
    if (n_orb < 1 || (capacity > 0 && !widths)) return fail(BLTC_EINVAL, "bltc_orbital_tiles: n_orb >= 1 and a widths array are required");
    const std::vector<int> g = orbital_groups(n_orb);
    for (int i = 0; i < (int)g.size() && i < capacity; ++i) widths[i] = g[i];
    return (int)g.size();
}

int bltc_create_host_plan_sharded(bltc_handle* h, const double* targets, const double* sources,
                                  const double* weights, int64_t N, double theta, int interp_degree,
                                  int batch_size, int leaf_size, int rank, int world) {
    (void)weights;
    int rc = check_create_args(h, sources, N, theta, interp_degree, batch_size, leaf_size);
    if (rc) return rc;
    if (world < 1 || rank < 0 || rank >= world) return fail(BLTC_EINVAL, "need 0 <= rank < world");
    bltc_plan_s* pl = new (std::nothrow) bltc_plan_s;
    if (!pl) return fail(BLTC_ENOMEM, "host allocation failed");
    rc = build_plan_guarded(pl, targets, sources, N, theta, interp_degree, batch_size, leaf_size, 148, rank, world,
                            /*upward_children=*/true);
    if (rc) { delete pl; return rc; }
    *h = pl;
    return BLTC_OK;
}

int bltc_create_host_plan(bltc_handle* h, const double* targets, const double* sources,
                          const double* weights, int64_t N, double theta, int interp_degree,
                          int batch_size, int leaf_size) {
    return bltc_create_host_plan_sharded(h, targets, sources, weights, N, theta, interp_degree, batch_size,
                                         leaf_size, 0, 1);
}

int bltc_create(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                int64_t N, double theta, int interp_degree, int batch_size, int leaf_size) {
    return bltc_create_with_builder(h, targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size, 0, 1,
                                    BLTC_BUILDER_DEVICE);
}

int bltc_create_sharded(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                        int64_t N, double theta, int interp_degree, int batch_size, int leaf_size,
                        int rank, int world) {
    return bltc_create_with_builder(h, targets, sources, weights, N, theta, interp_degree, batch_size, leaf_size, rank,
                                    world, BLTC_BUILDER_DEVICE);
}

int bltc_create_with_builder(bltc_handle* h, const double* targets, const double* sources, const double* weights,
                             int64_t N, double theta, int interp_degree, int batch_size, int leaf_size,
                             int rank, int world, int builder) {
    int rc = check_create_args(h, sources, N, theta, interp_degree, batch_size, leaf_size);
    if (rc) return rc;
    if (world < 1 || rank < 0 || rank >= world) return fail(BLTC_EINVAL, "need 0 <= rank < world");
    if (!weights) return fail(BLTC_EINVAL, "weights is NULL");
    if (builder & ~(BLTC_BUILDER_HOST | BLTC_UPWARD_FROM_CHILDREN | BLTC_UPWARD_FROM_PARTICLES))
        return fail(BLTC_EINVAL, "unknown builder / option bits");
    if ((builder & BLTC_UPWARD_FROM_CHILDREN) && (builder & BLTC_UPWARD_FROM_PARTICLES))
        return fail(BLTC_EINVAL, "BLTC_UPWARD_FROM_CHILDREN and BLTC_UPWARD_FROM_PARTICLES exclude each other");
    const bool upward_children = (builder & BLTC_UPWARD_FROM_PARTICLES) == 0;     // the default
    builder &= BLTC_BUILDER_HOST;
    if (N >= ((int64_t)1 << 28)) builder = BLTC_BUILDER_HOST;     // the device builder's sort keys are 32-bit
    int dev = 0, sms = 0;
    BLTC_CUDA(cudaGetDevice(&dev));
    BLTC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const auto t_begin = std::chrono::steady_clock::now();
    const bool same = (targets == nullptr || targets == sources);

    bltc_plan_s* pl = new (std::nothrow) bltc_plan_s;
    if (!pl) return fail(BLTC_ENOMEM, "host allocation failed");
    pl->device = dev;
    HostPlan& hp = pl->hp;
#define BLTC_TRY_OR_FREE(call)                                                                 \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess) {                                                              \
            cudaGetLastError(); delete pl;                                                     \
            return fail(e__ == cudaErrorMemoryAllocation ? BLTC_ENOMEM : BLTC_ECUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e__));                  \
        }                                                                                      \
    } while (0)

    // device views of the inputs (host arrays are uploaded once; device arrays are used in place)
    DevBuf<double> up_src, up_tgt, up_w;
    const double *d_src = sources, *d_tgt = same ? sources : targets, *d_w = weights;
    if (!is_device_ptr(sources)) {
        BLTC_TRY_OR_FREE(up_src.ensure(3 * (size_t)N));
        BLTC_TRY_OR_FREE(cudaMemcpy(up_src.p, sources, 3 * (size_t)N * sizeof(double), cudaMemcpyHostToDevice));
        d_src = up_src.p;
        if (same) d_tgt = d_src;
    }
    if (!same && !is_device_ptr(targets)) {
        BLTC_TRY_OR_FREE(up_tgt.ensure(3 * (size_t)N));
        BLTC_TRY_OR_FREE(cudaMemcpy(up_tgt.p, targets, 3 * (size_t)N * sizeof(double), cudaMemcpyHostToDevice));
        d_tgt = up_tgt.p;
    }
    if (!is_device_ptr(weights)) {
        BLTC_TRY_OR_FREE(up_w.ensure((size_t)N));
        BLTC_TRY_OR_FREE(cudaMemcpy(up_w.p, weights, (size_t)N * sizeof(double), cudaMemcpyHostToDevice));
        d_w = up_w.p;
    }

    if (builder == BLTC_BUILDER_HOST) {
        // the host builder needs host copies of the coordinates
        std::vector<double> hs, ht;
        try {
            hs.resize(3 * (size_t)N);
            if (!same) ht.resize(3 * (size_t)N);
        } catch (const std::bad_alloc&) { delete pl; return fail(BLTC_ENOMEM, "host allocation failed"); }
        BLTC_TRY_OR_FREE(cudaMemcpy(hs.data(), sources, hs.size() * sizeof(double), cudaMemcpyDefault));
        if (!same) BLTC_TRY_OR_FREE(cudaMemcpy(ht.data(), targets, ht.size() * sizeof(double), cudaMemcpyDefault));
        rc = build_plan_guarded(pl, same ? nullptr : ht.data(), hs.data(), N, theta, interp_degree,
                                batch_size, leaf_size, sms, rank, world, upward_children);
        if (rc) { delete pl; return rc; }
        BLTC_TRY_OR_FREE(pl->src_perm.upload(to_i32(hp.src.perm)));
        if (!hp.shared_order) BLTC_TRY_OR_FREE(pl->tgt_perm_own.upload(to_i32(hp.tgt.perm)));
    } else {
        // NEXT-4a: tree(s) and MAC lists by kernels (plan_device.cu); decisions identical to the host builder's
        Nvtx range_build("bltc_create: device plan build");
        const auto t0 = std::chrono::steady_clock::now();
        auto ms_since = [](std::chrono::steady_clock::time_point a) {
            return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - a).count();
        };
        try {
            plan_begin(hp, N, same, theta, interp_degree, batch_size, leaf_size, upward_children);
            hp.built_on_device = true;
            BLTC_TRY_OR_FREE(pl->src_perm.ensure((size_t)N));
            BLTC_TRY_OR_FREE(build_tree_device(hp.src, d_src, N, leaf_size, pl->src_perm.p, nullptr));
            if (!hp.shared_order) {
                BLTC_TRY_OR_FREE(pl->tgt_perm_own.ensure((size_t)N));
                BLTC_TRY_OR_FREE(build_tree_device(hp.tgt, d_tgt, N, batch_size, pl->tgt_perm_own.p, nullptr));
            }
            plan_set_batches(hp);
            hp.stage_ms[0] = ms_since(t0);
            const auto t1 = std::chrono::steady_clock::now();
            BLTC_TRY_OR_FREE(build_lists_device(hp, rank, world, nullptr));
            hp.stage_ms[1] = ms_since(t1);
            const auto t2 = std::chrono::steady_clock::now();
            plan_finish(hp, sms);
            hp.stage_ms[3] = ms_since(t2);
        } catch (const std::bad_alloc&) {
            delete pl; return fail(BLTC_ENOMEM, "host allocation failed while building the plan");
        } catch (const std::exception& e) {
            delete pl; return fail(BLTC_EINVAL, e.what());
        }
        hp.build_ms = ms_since(t0);
    }

    Nvtx range_upload("bltc_create: upload + proxy weights of w");
    const auto t0 = std::chrono::steady_clock::now();
    // tree-ordered records
    BLTC_TRY_OR_FREE(pl->src_rec.ensure((size_t)N));
    BLTC_TRY_OR_FREE(launch_pack_records(d_src, d_w, pl->src_perm.p, N, pl->src_rec.p, nullptr));
    if (hp.shared_order) {
        pl->tgt_rec = pl->src_rec.p; pl->tgt_perm = pl->src_perm.p;
    } else {
        BLTC_TRY_OR_FREE(pl->tgt_rec_own.ensure((size_t)N));
        BLTC_TRY_OR_FREE(launch_pack_records(d_tgt, nullptr, pl->tgt_perm_own.p, N, pl->tgt_rec_own.p, nullptr));
        pl->tgt_rec = pl->tgt_rec_own.p; pl->tgt_perm = pl->tgt_perm_own.p;
    }
    // batches, lists, work items
    {
        // the epilogue runs over this rank's batches only (all of them unless the plan is sharded)
        const size_t nb = (size_t)(hp.shard_b1 - hp.shard_b0);
        std::vector<int32_t> bb(nb), bc(nb), bs(nb);
        std::vector<int64_t> bp(nb);
        for (size_t i = 0; i < nb; ++i) {
            const size_t b = (size_t)hp.shard_b0 + i;
            bb[i] = (int32_t)hp.b_begin[b]; bc[i] = (int32_t)(hp.b_end[b] - hp.b_begin[b]);
            bs[i] = hp.b_nseg_far[b] + hp.b_nseg_near[b];
            bp[i] = hp.b_partial_base[b];
        }
        BLTC_TRY_OR_FREE(pl->b_begin.upload(bb));
        BLTC_TRY_OR_FREE(pl->b_count.upload(bc));
        BLTC_TRY_OR_FREE(pl->b_nseg.upload(bs));
        BLTC_TRY_OR_FREE(pl->b_partial_base.upload(bp));
        const size_t ns = hp.cluster_of_slot.size();
        BLTC_TRY_OR_FREE(pl->slot_nodes.upload(hp.slot_nodes));
        BLTC_TRY_OR_FREE(pl->far_slots.upload(hp.far_slots));
        BLTC_TRY_OR_FREE(pl->near_ranges.upload(hp.near_ranges));
        BLTC_TRY_OR_FREE(pl->far_items.upload(hp.far_items));
        BLTC_TRY_OR_FREE(pl->near_items.upload(hp.near_items));
        // f-independent proxy weights what_k (Eq. (35) right with q_j = w_j)
        BLTC_TRY_OR_FREE(pl->what.ensure(ns * (size_t)hp.P));
        BLTC_TRY_OR_FREE(pl->up_items.upload(hp.up_items));
        BLTC_TRY_OR_FREE(pl->up_reduce.upload(hp.up_reduce));
        BLTC_TRY_OR_FREE(pl->up_chunks.ensure((size_t)hp.up_partial_chunks * hp.P * kMaxOT));
        BLTC_TRY_OR_FREE(pl->c2p_items.upload(hp.c2p_items));
        BLTC_TRY_OR_FREE(launch_upward(0, pl->up_items.p, (int)hp.up_items.size(), pl->up_reduce.p,
                                       (int)hp.up_reduce.size(), pl->slot_nodes.p, hp.degree, pl->src_rec.p,
                                       nullptr, pl->what.p, pl->up_chunks.p, nullptr));
        for (size_t lv = 0; lv + 1 < hp.c2p_level_ptr.size(); ++lv)
            BLTC_TRY_OR_FREE(launch_upward_children(0, pl->c2p_items.p + hp.c2p_level_ptr[lv],
                                                    hp.c2p_level_ptr[lv + 1] - hp.c2p_level_ptr[lv], pl->slot_nodes.p,
                                                    hp.degree, pl->what.p, nullptr));
        BLTC_TRY_OR_FREE(cudaDeviceSynchronize());
    }
#undef BLTC_TRY_OR_FREE
    pl->upload_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    pl->create_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_begin).count();
    pl->on_device = true;
    *h = pl;
    return BLTC_OK;
}

int bltc_destroy(bltc_handle h) {
    if (!h) return fail(BLTC_EINVAL, "handle is NULL");
    delete h;
    return BLTC_OK;
}

int bltc_get_stats(bltc_handle h, bltc_stats* s) {
    if (!h || !s) return fail(BLTC_EINVAL, "NULL argument");
    const HostPlan& hp = h->hp;
    std::memset(s, 0, sizeof *s);
    s->n_points = hp.N;
    s->n_clusters = (int64_t)hp.src.cl.size();
    s->n_leaves = (int64_t)hp.src.leaves.size();
    s->n_batches = (int64_t)hp.b_begin.size();
    s->n_far = (int64_t)hp.far_idx.size();
    s->n_near = (int64_t)hp.near_idx.size();
    s->far_evals = hp.far_evals;
    s->near_evals = hp.near_evals;
    s->n_proxy_clusters = (int64_t)hp.cluster_of_slot.size();
    s->upward_pairs = hp.upward_pairs;
    s->n_far_items = (int64_t)hp.far_items.size();
    s->n_near_items = (int64_t)hp.near_items.size();
    s->partial_len = hp.partial_len;
    s->n_upward_items = (int64_t)hp.up_items.size();
    s->n_upward_reduce = (int64_t)hp.up_reduce.size();
    s->launches_per_group = 1 /* gather */ + (hp.shared_order ? 0 : 1) + (hp.up_items.empty() ? 0 : 1) +
                            (hp.up_reduce.empty() ? 0 : 1) + (int64_t)(hp.c2p_level_ptr.size() - 1) +
                            (hp.far_items.empty() ? 0 : 1) +
                            (hp.near_items.empty() ? 0 : 1) + 1 /* epilogue */;
    s->shared_batches = hp.shared_order ? 1 : 0;
    s->interp_degree = hp.degree;
    s->theta = hp.theta;
    s->build_ms = hp.build_ms;
    s->upload_ms = h->upload_ms;
    s->shard_rank = hp.shard_rank;
    s->shard_world = hp.shard_world;
    s->shard_batch_begin = hp.shard_b0;
    s->shard_batch_end = hp.shard_b1;
    s->shard_targets = hp.shard_b1 > hp.shard_b0 ? hp.b_end[hp.shard_b1 - 1] - hp.b_begin[hp.shard_b0] : 0;
    s->shard_far_evals = hp.shard_far_evals;
    s->shard_near_evals = hp.shard_near_evals;
    s->tree_ms = hp.stage_ms[0];
    s->lists_ms = hp.stage_ms[1];
    s->decomp_ms = hp.stage_ms[3];
    s->create_ms = h->create_ms;
    s->built_on_device = hp.built_on_device ? 1 : 0;
    s->upward_from_children = hp.upward_children ? 1 : 0;
    return BLTC_OK;
}

int bltc_export_plan(bltc_handle h, int64_t* src_perm, int64_t* tgt_perm,
                     int64_t* cl_begin, int64_t* cl_end, double* cl_lo, double* cl_hi,
                     int32_t* cl_parent, int32_t* cl_nchild, int64_t* b_begin, int64_t* b_end,
                     int64_t* far_ptr, int32_t* far_idx, int64_t* near_ptr, int32_t* near_idx) {
    if (!h) return fail(BLTC_EINVAL, "handle is NULL");
    HostPlan& hp = h->hp;
    BLTC_CUDA(ensure_host_perm(h));
    if (hp.lists_b0 > 0 || hp.lists_b1 < (int)hp.b_begin.size()) {
        // a sharded device-built plan traversed only its own batches: complete the lists on the host (the entries
        // of its own batches come out identical; nothing derived from them changes)
        try {
            std::vector<int64_t> fe, ne;
            plan_lists_host(hp, fe, ne);
        } catch (const std::exception& e) { return fail(BLTC_ENOMEM, e.what()); }
    }
    if (src_perm) std::memcpy(src_perm, hp.src.perm.data(), hp.src.perm.size() * sizeof(int64_t));
    if (tgt_perm) std::memcpy(tgt_perm, hp.tgt_perm().data(), hp.tgt_perm().size() * sizeof(int64_t));
    for (size_t c = 0; c < hp.src.cl.size(); ++c) {
        const Cluster& C = hp.src.cl[c];
        if (cl_begin) cl_begin[c] = C.begin;
        if (cl_end) cl_end[c] = C.end;
        for (int d = 0; d < 3; ++d) {
            if (cl_lo) cl_lo[3 * c + d] = C.lo[d];
            if (cl_hi) cl_hi[3 * c + d] = C.hi[d];
        }
        if (cl_parent) cl_parent[c] = C.parent;
        if (cl_nchild) cl_nchild[c] = C.nchild;
    }
    if (b_begin) std::memcpy(b_begin, hp.b_begin.data(), hp.b_begin.size() * sizeof(int64_t));
    if (b_end) std::memcpy(b_end, hp.b_end.data(), hp.b_end.size() * sizeof(int64_t));
    if (far_ptr) std::memcpy(far_ptr, hp.far_ptr.data(), hp.far_ptr.size() * sizeof(int64_t));
    if (near_ptr) std::memcpy(near_ptr, hp.near_ptr.data(), hp.near_ptr.size() * sizeof(int64_t));
    if (far_idx) std::memcpy(far_idx, hp.far_idx.data(), hp.far_idx.size() * sizeof(int32_t));
    if (near_idx) std::memcpy(near_idx, hp.near_idx.data(), hp.near_idx.size() * sizeof(int32_t));
    return BLTC_OK;
}

int bltc_get_shard_targets(bltc_handle h, int64_t* idx) {
    if (!h || !idx) return fail(BLTC_EINVAL, "NULL argument");
    const HostPlan& hp = h->hp;
    if (hp.shard_b1 <= hp.shard_b0) return BLTC_OK;
    BLTC_CUDA(ensure_host_perm(h));
    const std::vector<int64_t>& perm = hp.tgt_perm();
    const int64_t t0 = hp.b_begin[hp.shard_b0], t1 = hp.b_end[hp.shard_b1 - 1];
    for (int64_t t = t0; t < t1; ++t) idx[t - t0] = perm[t];
    return BLTC_OK;
}

int bltc_export_proxy(bltc_handle h, int32_t* proxy_cluster, double* nodes, double* what,
                      double* fhat, int32_t* ot) {
    if (!h) return fail(BLTC_EINVAL, "handle is NULL");
    if (!h->on_device) return fail(BLTC_ENODEVICE, "plan has no device state");
    const HostPlan& hp = h->hp;
    const size_t ns = hp.cluster_of_slot.size();
    BLTC_CUDA(cudaDeviceSynchronize());
    if (proxy_cluster) std::memcpy(proxy_cluster, hp.cluster_of_slot.data(), ns * sizeof(int32_t));
    if (nodes) std::memcpy(nodes, hp.slot_nodes.data(), hp.slot_nodes.size() * sizeof(double));
    if (what && ns) BLTC_CUDA(cudaMemcpy(what, h->what.p, ns * hp.P * sizeof(double), cudaMemcpyDeviceToHost));
    if (fhat && ns && h->last_ot > 0)
        BLTC_CUDA(cudaMemcpy(fhat, h->fhat.p, ns * hp.P * h->last_ot * sizeof(double), cudaMemcpyDeviceToHost));
    if (ot) *ot = h->last_ot;
    return BLTC_OK;
}

int bltc_set_profiling(bltc_handle h, int enable) {
    if (!h) return fail(BLTC_EINVAL, "handle is NULL");
    h->profiling = enable != 0;
    return BLTC_OK;
}

int bltc_get_phase_ms(bltc_handle h, float ms[BLTC_NUM_PHASES]) {
    if (!h || !ms) return fail(BLTC_EINVAL, "NULL argument");
    for (int p = 0; p < BLTC_NUM_PHASES; ++p) ms[p] = 0.f;
    if (h->events_used == 0) return fail(BLTC_EINVAL, "no profiled convolve has run");
    BLTC_CUDA(cudaEventSynchronize(h->events[h->events_used - 1]));
    const int per = BLTC_NUM_PHASES + 1;
    for (int g = 0; g < h->events_used / per; ++g)
        for (int p = 0; p < BLTC_NUM_PHASES; ++p) {
            float t = 0.f;
            BLTC_CUDA(cudaEventElapsedTime(&t, h->events[g * per + p], h->events[g * per + p + 1]));
            ms[p] += t;
        }
    return BLTC_OK;
}

}  // extern "C"

namespace {

// One convolution through the plan, kind = kYukawa (k: n_orb values) or kCoulomb (alpha; k unused).
int convolve_impl(bltc_handle h, int kind, const double* k, double alpha, const double* f, int n_orb,
                  double* out, int subtract_singularity, bltc_stream stream, double* const* peers = nullptr,
                  int n_peers = 0) {
    if (!h) return fail(BLTC_EINVAL, "handle is NULL");
    if (n_peers < 0 || n_peers > kMaxOuts - 1) return fail(BLTC_EINVAL, "at most 15 additional destinations");
    if (n_peers > 0 && !peers) return fail(BLTC_EINVAL, "peer destination array is NULL");
    for (int r = 0; r < n_peers; ++r)
        if (!peers[r]) return fail(BLTC_EINVAL, "a peer destination is NULL");
    if (n_peers > 0 && out && !is_device_ptr(out)) return fail(BLTC_EINVAL, "bltc_convolve_scatter needs device buffers");
    if (!h->on_device) return fail(BLTC_ENODEVICE, "plan was built with bltc_create_host_plan (no device state)");
    if (!f || !out) return fail(BLTC_EINVAL, "f and out must not be NULL");
    if (n_orb < 1) return fail(BLTC_EINVAL, "n_orb must be >= 1");
    HostPlan& hp = h->hp;
    const bool sub = subtract_singularity != 0;
    if (sub && !hp.same_points) return fail(BLTC_EINVAL, "subtract_singularity requires targets == sources");
    if (kind == kYukawa) {
        if (!k) return fail(BLTC_EINVAL, "k must not be NULL");
        for (int o = 0; o < n_orb; ++o)
            if (!(k[o] > 0.0) || !std::isfinite(k[o])) return fail(BLTC_EINVAL, "every k must be finite and > 0");
    } else if (sub && (!(alpha > 0.0) || !std::isfinite(alpha) || !(hp.max_dist / alpha < 5e5))) {
        return fail(BLTC_EINVAL, "alpha must be finite, > 0 and > 2e-6 x the domain diameter");
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int64_t N = hp.N;
    Nvtx range_call(kind == kYukawa ? "bltc_convolve" : "bltc_convolve_coulomb");
    // per-plan scratch (fsrc, fhat, partial, staging) is reused by every call: order this call after the previous one
    // even if the caller switched streams (same stream: already ordered)
    if (!h->last_done) BLTC_CUDA(cudaEventCreateWithFlags(&h->last_done, cudaEventDisableTiming));
    if (h->has_last && h->last_stream != st) BLTC_CUDA(cudaStreamWaitEvent(st, h->last_done, 0));

    // host buffers are staged through device memory inside the call
    const double* d_f = f;
    double* d_out = out;
    const bool out_on_host = !is_device_ptr(out);
    if (!is_device_ptr(f)) {
        BLTC_CUDA(h->f_stage.ensure((size_t)n_orb * N));
        BLTC_CUDA(cudaMemcpyAsync(h->f_stage.p, f, (size_t)n_orb * N * sizeof(double), cudaMemcpyHostToDevice, st));
        d_f = h->f_stage.p;
    }
    if (out_on_host) {
        BLTC_CUDA(h->out_stage.ensure((size_t)n_orb * N));
        d_out = h->out_stage.p;
        // a sharded plan writes its own targets only: the caller's other elements must survive the copy back
        if (hp.shard_world > 1)
            BLTC_CUDA(cudaMemcpyAsync(d_out, out, (size_t)n_orb * N * sizeof(double), cudaMemcpyHostToDevice, st));
    }

    const size_t ns = hp.cluster_of_slot.size();
    BLTC_CUDA(h->fsrc.ensure((size_t)N * kMaxOT));
    if (!hp.shared_order && sub) BLTC_CUDA(h->ftgt_own.ensure((size_t)N * kMaxOT));
    BLTC_CUDA(h->fhat.ensure(ns * (size_t)hp.P * kMaxOT));
    BLTC_CUDA(h->partial.ensure((size_t)hp.partial_len * kMaxOT));

    const std::vector<int> groups = orbital_groups(n_orb);
    const int per = BLTC_NUM_PHASES + 1;
    if (h->profiling) {
        while (h->events.size() < groups.size() * per) {
            cudaEvent_t e; BLTC_CUDA(cudaEventCreate(&e)); h->events.push_back(e);
        }
    }
    h->events_used = 0;
    int o0 = 0;
    for (size_t g = 0; g < groups.size(); ++g) {
        const int ot = groups[g];
        const KPar nk = kind == kYukawa ? make_kpar(k + o0, ot) : make_kpar_coulomb(sub ? alpha : 1.0);
        const EpiPar ep = kind == kYukawa ? make_epipar(k + o0, ot) : make_epipar_coulomb(sub ? alpha : 1.0);
        // exp underflow guard: not needed when k r < 700 for every pair (max_dist bounds r)
        double kmax = 0.0;
        if (kind == kYukawa) for (int o = 0; o < ot; ++o) kmax = std::max(kmax, k[o0 + o]);
        const bool guard = kind != kYukawa || !(kmax * hp.max_dist < 700.0);
        cudaEvent_t* ev = h->profiling ? &h->events[g * per] : nullptr;
        if (ev) BLTC_CUDA(cudaEventRecord(ev[0], st));
        // a1: gather to tree order
        const double* ftgt = h->fsrc.p;
        {
            Nvtx range_gather("bltc_convolve: a1 gather");
            BLTC_CUDA(launch_gather(d_f, N, o0, ot, h->src_perm.p, N, h->fsrc.p, st));
            if (!hp.shared_order && sub) {
                BLTC_CUDA(launch_gather(d_f, N, o0, ot, h->tgt_perm, N, h->ftgt_own.p, st));
                ftgt = h->ftgt_own.p;
            }
        }
        if (ev) BLTC_CUDA(cudaEventRecord(ev[1], st));
        // a2: upward pass
        Nvtx range_kernels("bltc_convolve: a2 upward, a3 far, a4 near, a5 epilogue");
        BLTC_CUDA(launch_upward(ot, h->up_items.p, (int)hp.up_items.size(), h->up_reduce.p,
                                (int)hp.up_reduce.size(), h->slot_nodes.p, hp.degree, h->src_rec.p, h->fsrc.p,
                                h->fhat.p, h->up_chunks.p, st));
        for (size_t lv = 0; lv + 1 < hp.c2p_level_ptr.size(); ++lv)      // child -> parent levels, deepest first (R23)
            BLTC_CUDA(launch_upward_children(ot, h->c2p_items.p + hp.c2p_level_ptr[lv],
                                             hp.c2p_level_ptr[lv + 1] - hp.c2p_level_ptr[lv], h->slot_nodes.p, hp.degree,
                                             h->fhat.p, st));
        if (ev) BLTC_CUDA(cudaEventRecord(ev[2], st));
        // a3: far field
        BLTC_CUDA(launch_far(kind, ot, sub, guard, h->far_items.p, (int)hp.far_items.size(), h->far_slots.p,
                             h->slot_nodes.p, h->what.p, h->fhat.p, hp.degree, h->tgt_rec, ftgt, nk,
                             h->partial.p, hp.partial_len, st));
        if (ev) BLTC_CUDA(cudaEventRecord(ev[3], st));
        // a4: near field
        BLTC_CUDA(launch_near(kind, ot, sub, guard, false, h->near_items.p, (int)hp.near_items.size(), h->near_ranges.p,
                              h->src_rec.p, h->fsrc.p, h->tgt_rec, ftgt, nk, h->partial.p, hp.partial_len, st));
        if (ev) BLTC_CUDA(cudaEventRecord(ev[4], st));
        // a5: epilogue
        OutSet outs;
        outs.n = 1 + n_peers; outs.p[0] = d_out;
        for (int r = 0; r < n_peers; ++r) outs.p[1 + r] = peers[r];
        BLTC_CUDA(launch_epilogue(ot, sub, hp.shard_b1 - hp.shard_b0, h->b_begin.p, h->b_count.p,
                                  h->b_partial_base.p, h->b_nseg.p, h->partial.p, hp.partial_len, ftgt, ep,
                                  h->tgt_perm, outs, N, o0, st));
        if (ev) { BLTC_CUDA(cudaEventRecord(ev[5], st)); h->events_used += per; }
        h->last_ot = ot;
        o0 += ot;
    }
    if (out_on_host) BLTC_CUDA(cudaMemcpyAsync(out, d_out, (size_t)n_orb * N * sizeof(double), cudaMemcpyDeviceToHost, st));
    BLTC_CUDA(cudaEventRecord(h->last_done, st));
    h->last_stream = st; h->has_last = true;
    if (out_on_host) BLTC_CUDA(cudaStreamSynchronize(st));
    return BLTC_OK;
}

}  // namespace

extern "C" {

int bltc_convolve(bltc_handle h, const double* k, const double* f, int n_orb, double* out,
                  int subtract_singularity, bltc_stream stream) {
    return convolve_impl(h, kYukawa, k, 0.0, f, n_orb, out, subtract_singularity, stream);
}

int bltc_convolve_coulomb(bltc_handle h, const double* f, int n_f, double* out, int subtract_singularity,
                          double alpha, bltc_stream stream) {
    return convolve_impl(h, kCoulomb, nullptr, alpha, f, n_f, out, subtract_singularity, stream);
}

int bltc_convolve_scatter(bltc_handle h, const double* k, const double* f, int n_orb, double* out,
                          double* const* peer_outs, int n_peers, int subtract_singularity, bltc_stream stream) {
    return convolve_impl(h, kYukawa, k, 0.0, f, n_orb, out, subtract_singularity, stream, peer_outs, n_peers);
}

int bltc_convolve_coulomb_scatter(bltc_handle h, const double* f, int n_f, double* out, double* const* peer_outs,
                                  int n_peers, int subtract_singularity, double alpha, bltc_stream stream) {
    return convolve_impl(h, kCoulomb, nullptr, alpha, f, n_f, out, subtract_singularity, stream, peer_outs, n_peers);
}

int bltc_direct_set_profiling(int enable) { g_direct_profiling = enable != 0; return BLTC_OK; }

int bltc_direct_get_kernel_ms(float* ms) {
    if (!ms) return fail(BLTC_EINVAL, "NULL argument");
    *ms = 0.f;
    if (g_direct_pairs.empty()) return fail(BLTC_EINVAL, "no profiled direct_convolve has run");
    for (auto& pr : g_direct_pairs) {
        float t = 0.f;
        BLTC_CUDA(cudaEventSynchronize(pr.second));
        BLTC_CUDA(cudaEventElapsedTime(&t, pr.first, pr.second));
        *ms += t;
    }
    return BLTC_OK;
}

}  // extern "C"

namespace {

int direct_impl(int kind, const double* targets, const double* f_targets, int64_t M,
                const double* sources, const double* weights, const double* f_sources, int64_t N,
                const double* k, double alpha, int n_orb, double* out, int subtract_singularity,
                bltc_stream stream) {
    if (!targets || !sources || !weights || !f_sources || !out)
        return fail(BLTC_EINVAL, "targets, sources, weights, f_sources and out must not be NULL");
    if (M < 0 || N < 0 || M > 2000000000LL || N > 2000000000LL) return fail(BLTC_EINVAL, "M, N must be in [0, 2e9]");
    if (n_orb < 1) return fail(BLTC_EINVAL, "n_orb must be >= 1");
    const bool sub = subtract_singularity != 0;
    if (sub && !f_targets) return fail(BLTC_EINVAL, "subtract_singularity needs f_targets");
    if (kind == kYukawa) {
        if (!k) return fail(BLTC_EINVAL, "k must not be NULL");
        for (int o = 0; o < n_orb; ++o)
            if (!(k[o] > 0.0) || !std::isfinite(k[o])) return fail(BLTC_EINVAL, "every k must be finite and > 0");
    } else if (sub && (!(alpha > 0.0) || !std::isfinite(alpha))) {
        return fail(BLTC_EINVAL, "alpha must be finite and > 0");
    }
    if (M == 0) return BLTC_OK;
    Nvtx range_call(kind == kYukawa ? "direct_convolve" : "direct_convolve_coulomb");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    BLTC_CUDA(cudaGetDevice(&dev));
    BLTC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));

    TempBuf t_tg, t_ft, t_sr, t_w, t_fs, t_out;
    const double *d_tg, *d_ft, *d_sr, *d_w, *d_fs;
    BLTC_CUDA(stage_in(targets, 3 * (size_t)M, t_tg, st, &d_tg));
    BLTC_CUDA(stage_in(sub ? f_targets : nullptr, (size_t)n_orb * M, t_ft, st, &d_ft));
    BLTC_CUDA(stage_in(sources, 3 * (size_t)N, t_sr, st, &d_sr));
    BLTC_CUDA(stage_in(weights, (size_t)N, t_w, st, &d_w));
    BLTC_CUDA(stage_in(f_sources, (size_t)n_orb * N, t_fs, st, &d_fs));
    const bool out_on_host = !is_device_ptr(out);
    double* d_out = out;
    if (out_on_host) { BLTC_CUDA(t_out.alloc((size_t)n_orb * M * sizeof(double), st)); d_out = t_out.as<double>(); }

    // work decomposition: pseudo-batches of 2048 targets, tiles of 8 groups inside them, and
    // nsplit equal source segments so that >= ~16 CTAs exist per resident CTA slot
    constexpr int64_t kPB = 2048;
    std::vector<WorkItem> items;
    std::vector<Range> ranges;
    std::vector<int32_t> pb_begin, pb_count, pb_nseg;
    std::vector<int64_t> pb_base;
    int nsplit = 1;
    const int64_t npb64 = (M + kPB - 1) / kPB;
    {
        const int64_t tiles512 = (M + 511) / 512;
        const int64_t want = (int64_t)sms * 2 * 8;
        nsplit = (int)std::min<int64_t>(64, std::max<int64_t>(1, (want + tiles512 - 1) / tiles512));
        nsplit = (int)std::min<int64_t>(nsplit, std::max<int64_t>(1, N / 256));
    }
    // Bounding boxes of the pseudo-batches and of the source segments (one small kernel each, read back: the one
    // synchronisation of this call): the exp underflow guard is compiled in only if k_max x (the largest possible
    // distance) can reach 700.  The r == 0 test (reading R3) runs for every pair: launch_near below is called with
    // all_zero_safe = true, which ignores Range::flags, so no per-range "may coincide" flag is computed here.
    const int64_t seg_len = std::max<int64_t>(1, (N + nsplit - 1) / nsplit);
    const int nseg_box = (int)((N + seg_len - 1) / seg_len);
    std::vector<double> box_t((size_t)npb64 * 6), box_s((size_t)nseg_box * 6);
    {
        TempBuf t_bt, t_bs;
        BLTC_CUDA(t_bt.alloc(box_t.size() * sizeof(double), st));
        BLTC_CUDA(t_bs.alloc(box_s.size() * sizeof(double), st));
        BLTC_CUDA(launch_chunk_bbox(d_tg, M, kPB, t_bt.as<double>(), st));
        BLTC_CUDA(launch_chunk_bbox(d_sr, N, seg_len, t_bs.as<double>(), st));
        BLTC_CUDA(cudaMemcpyAsync(box_t.data(), t_bt.p, box_t.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        BLTC_CUDA(cudaMemcpyAsync(box_s.data(), t_bs.p, box_s.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        BLTC_CUDA(cudaStreamSynchronize(st));
    }
    bool guard = true;
    if (kind == kYukawa) {
        double lo[3], hi[3], d2 = 0.0, kmax = 0.0;
        for (int d = 0; d < 3; ++d) { lo[d] = INFINITY; hi[d] = -INFINITY; }
        for (int64_t c = 0; c < npb64; ++c)
            for (int d = 0; d < 3; ++d) { lo[d] = std::min(lo[d], box_t[c * 6 + d]); hi[d] = std::max(hi[d], box_t[c * 6 + 3 + d]); }
        for (int c = 0; c < nseg_box; ++c)
            for (int d = 0; d < 3; ++d) { lo[d] = std::min(lo[d], box_s[c * 6 + d]); hi[d] = std::max(hi[d], box_s[c * 6 + 3 + d]); }
        for (int d = 0; d < 3; ++d) d2 += (hi[d] - lo[d]) * (hi[d] - lo[d]);
        for (int o = 0; o < n_orb; ++o) kmax = std::max(kmax, k[o]);
        guard = !(kmax * std::sqrt(d2) < 700.0);
    }
    {
        // ranges[pb * nsplit + s]: source segment s as seen from pseudo-batch pb
        ranges.reserve((size_t)npb64 * nsplit);
        for (int64_t pb = 0; pb < npb64; ++pb) {
            const int64_t b0 = pb * kPB;
            pb_begin.push_back((int32_t)b0);
            pb_count.push_back((int32_t)std::min<int64_t>(kPB, M - b0));
            pb_nseg.push_back(nsplit);
            pb_base.push_back((int64_t)nsplit * b0);
            for (int s = 0; s < nsplit; ++s) {
                const int64_t s0 = std::min<int64_t>(N, (int64_t)s * seg_len), s1 = std::min<int64_t>(N, (int64_t)(s + 1) * seg_len);
                ranges.push_back(Range{(int32_t)s0, (int32_t)s1, kRangeMayCoincide});
            }
        }
        const int unit = 32 * kTargetsPerThread;
        for (int64_t t0 = 0; t0 < M;) {
            const int64_t pb = t0 / kPB, pb_end = std::min<int64_t>(M, (pb + 1) * kPB);
            const int64_t groups = (pb_end - t0 + unit - 1) / unit;
            int g = kTileGroupsMax;
            if (groups < kTileGroupsMax) { g = 1; while (2 * g <= groups) g *= 2; }
            int gs = 0; while ((1 << gs) < g) ++gs;
            const int64_t cnt = std::min<int64_t>((int64_t)g * unit, pb_end - t0);
            for (int s = 0; s < nsplit; ++s)
                items.push_back(WorkItem{(int32_t)t0, (int32_t)cnt, gs, (int32_t)(pb * nsplit + s), (int32_t)(pb * nsplit + s + 1), 0,
                                         pb_base[pb] + (int64_t)s * pb_count[pb] + (t0 - pb * kPB)});
            t0 += cnt;
        }
    }
    const int64_t partial_len = (int64_t)nsplit * M;
    const size_t npb = pb_begin.size();
    TempBuf t_src_rec, t_tgt_rec, t_fsrc, t_ftgt, t_partial, t_items, t_ranges, t_pbb, t_pbc, t_pbn, t_pbs;
    BLTC_CUDA(t_src_rec.alloc((size_t)N * sizeof(double4), st));
    BLTC_CUDA(t_tgt_rec.alloc((size_t)M * sizeof(double4), st));
    BLTC_CUDA(t_fsrc.alloc((size_t)N * kMaxOT * sizeof(double), st));
    BLTC_CUDA(t_ftgt.alloc((size_t)M * kMaxOT * sizeof(double), st));
    BLTC_CUDA(t_partial.alloc((size_t)partial_len * kMaxOT * sizeof(double), st));
    auto put = [&](TempBuf& t, const void* src, size_t bytes) -> cudaError_t {
        cudaError_t e = t.alloc(bytes, st);
        if (e != cudaSuccess) return e;
        return cudaMemcpyAsync(t.p, src, bytes, cudaMemcpyHostToDevice, st);
    };
    BLTC_CUDA(put(t_ranges, ranges.data(), ranges.size() * sizeof(Range)));
    BLTC_CUDA(put(t_pbb, pb_begin.data(), npb * sizeof(int32_t)));
    BLTC_CUDA(put(t_pbc, pb_count.data(), npb * sizeof(int32_t)));
    BLTC_CUDA(put(t_pbn, pb_nseg.data(), npb * sizeof(int32_t)));
    BLTC_CUDA(put(t_pbs, pb_base.data(), npb * sizeof(int64_t)));
    BLTC_CUDA(launch_pack_records(d_sr, d_w, nullptr, N, t_src_rec.as<double4>(), st));
    BLTC_CUDA(launch_pack_records(d_tg, nullptr, nullptr, M, t_tgt_rec.as<double4>(), st));

    BLTC_CUDA(put(t_items, items.data(), items.size() * sizeof(WorkItem)));
    const std::vector<int> groups = orbital_groups(n_orb);
    if (g_direct_profiling) {
        for (auto& pr : g_direct_pairs) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
        g_direct_pairs.clear();
    }
    int o0 = 0;
    for (size_t g = 0; g < groups.size(); ++g) {
        const int ot = groups[g];
        const KPar nk = kind == kYukawa ? make_kpar(k + o0, ot) : make_kpar_coulomb(sub ? alpha : 1.0);
        const EpiPar ep = kind == kYukawa ? make_epipar(k + o0, ot) : make_epipar_coulomb(sub ? alpha : 1.0);
        BLTC_CUDA(launch_gather(d_fs, N, o0, ot, nullptr, N, t_fsrc.as<double>(), st));
        if (sub) BLTC_CUDA(launch_gather(d_ft, M, o0, ot, nullptr, M, t_ftgt.as<double>(), st));
        cudaEvent_t ea = nullptr, eb = nullptr;
        if (g_direct_profiling) {
            BLTC_CUDA(cudaEventCreate(&ea)); BLTC_CUDA(cudaEventCreate(&eb));
            BLTC_CUDA(cudaEventRecord(ea, st));
        }
        BLTC_CUDA(launch_near(kind, ot, sub, guard, true, t_items.as<WorkItem>(), (int)items.size(), t_ranges.as<Range>(),
                              t_src_rec.as<double4>(), t_fsrc.as<double>(), t_tgt_rec.as<double4>(),
                              t_ftgt.as<double>(), nk, t_partial.as<double>(), partial_len, st));
        if (g_direct_profiling) { BLTC_CUDA(cudaEventRecord(eb, st)); g_direct_pairs.emplace_back(ea, eb); }
        OutSet outs;
        outs.n = 1; outs.p[0] = d_out;
        BLTC_CUDA(launch_epilogue(ot, sub, (int)npb, t_pbb.as<int32_t>(), t_pbc.as<int32_t>(),
                                  t_pbs.as<int64_t>(), t_pbn.as<int32_t>(), t_partial.as<double>(), partial_len,
                                  t_ftgt.as<double>(), ep, nullptr, outs, M, o0, st));
        o0 += ot;
    }
    if (out_on_host) {
        BLTC_CUDA(cudaMemcpyAsync(out, d_out, (size_t)n_orb * M * sizeof(double), cudaMemcpyDeviceToHost, st));
        BLTC_CUDA(cudaStreamSynchronize(st));
    }
    return BLTC_OK;
}

}  // namespace

namespace bltc {
int set_last_error(int code, const char* msg) { return fail(code, msg ? msg : ""); }

cudaError_t pool_alloc_async(void** p, size_t bytes, cudaStream_t st) {
    cudaMemPool_t pool = TempBuf::library_pool();
    if (!pool) return cudaMallocAsync(p, bytes ? bytes : 1, st);
    return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, st);
}
}  // namespace bltc

extern "C" {

int direct_convolve(const double* targets, const double* f_targets, int64_t M,
                    const double* sources, const double* weights, const double* f_sources, int64_t N,
                    const double* k, int n_orb, double* out, int subtract_singularity,
                    bltc_stream stream) {
    return direct_impl(kYukawa, targets, f_targets, M, sources, weights, f_sources, N, k, 0.0, n_orb, out,
                       subtract_singularity, stream);
}

int direct_convolve_coulomb(const double* targets, const double* f_targets, int64_t M,
                            const double* sources, const double* weights, const double* f_sources, int64_t N,
                            int n_f, double* out, int subtract_singularity, double alpha, bltc_stream stream) {
    return direct_impl(kCoulomb, targets, f_targets, M, sources, weights, f_sources, N, nullptr, alpha, n_f, out,
                       subtract_singularity, stream);
}

int bltc_gi_update(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                   const double* phi, int n_prev, int64_t N, double eps_old, double* result,
                   bltc_stream stream) {
    if (!w || !psi_old || !f_old || !psi_new || !result) return fail(BLTC_EINVAL, "NULL argument");
    if (N < 1 || N > 2000000000LL) return fail(BLTC_EINVAL, "N must be in [1, 2e9]");
    if (n_prev < 0 || n_prev > 4096) return fail(BLTC_EINVAL, "n_prev must be in [0, 4096]");
    if (n_prev > 0 && !phi) return fail(BLTC_EINVAL, "phi is NULL but n_prev > 0");
    if (!std::isfinite(eps_old)) return fail(BLTC_EINVAL, "eps_old must be finite");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    BLTC_CUDA(cudaGetDevice(&dev));
    BLTC_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    TempBuf t_w, t_po, t_f, t_phi, t_pn, t_res, t_scratch;
    const double *d_w, *d_po, *d_f, *d_phi;
    BLTC_CUDA(stage_in(w, (size_t)N, t_w, st, &d_w));
    BLTC_CUDA(stage_in(psi_old, (size_t)N, t_po, st, &d_po));
    BLTC_CUDA(stage_in(f_old, (size_t)N, t_f, st, &d_f));
    BLTC_CUDA(stage_in(n_prev ? phi : nullptr, (size_t)n_prev * N, t_phi, st, &d_phi));
    const bool psi_on_host = !is_device_ptr(psi_new), res_on_host = !is_device_ptr(result);
    double* d_pn = psi_new;
    if (psi_on_host) {
        BLTC_CUDA(t_pn.alloc((size_t)N * sizeof(double), st));
        d_pn = t_pn.as<double>();
        BLTC_CUDA(cudaMemcpyAsync(d_pn, psi_new, (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    double* d_res = result;
    const size_t nres = 4 + (size_t)n_prev;
    if (res_on_host) { BLTC_CUDA(t_res.alloc(nres * sizeof(double), st)); d_res = t_res.as<double>(); }
    const int nblk = gi_grid_blocks(N, sms);
    BLTC_CUDA(t_scratch.alloc(gi_scratch_doubles(n_prev, nblk) * sizeof(double), st));
    BLTC_CUDA(launch_gi_update(d_w, d_po, d_f, d_pn, d_phi, n_prev, N, eps_old, d_res, t_scratch.as<double>(), nblk, st));
    if (psi_on_host) BLTC_CUDA(cudaMemcpyAsync(psi_new, d_pn, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (res_on_host) BLTC_CUDA(cudaMemcpyAsync(result, d_res, nres * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (psi_on_host || res_on_host) BLTC_CUDA(cudaStreamSynchronize(st));
    return BLTC_OK;
}

int bltc_probe_fp64_form(int form, int iters, double* tflops, bltc_stream stream) {
    if (!tflops || iters < 1 || form < 0 || form > 1) return fail(BLTC_EINVAL, "bad argument");
    float ms = 0.f; double dfma = 0.0;
    BLTC_CUDA(launch_fp64_probe(form, iters, &ms, &dfma, static_cast<cudaStream_t>(stream)));
    *tflops = 2.0 * dfma / (ms * 1e-3) / 1e12;
    return BLTC_OK;
}

int bltc_probe_fp64(int iters, double* tflops, bltc_stream stream) { return bltc_probe_fp64_form(0, iters, tflops, stream); }

}  // extern "C"
