// Built by tests/test_sanitizers.py with -fsanitize=address,undefined: the host plan builder (plan_host.cpp) and the
// CPU oracle (oracle/*.c) on small clouds that hit the odd paths -- duplicates, planar points, leaf size 1, a second
// (batch) tree, sharding, empty far lists; the work decomposition's invariants are checked on the way.  Prints "sanitize ok"; any ASan / UBSan report makes the run fail.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../paper_2003_01833_b200/csrc/plan_host.hpp"

extern "C" {
struct oracle_plan;
oracle_plan* oracle_plan_create(int64_t N, const double* sx, const double* sy, const double* sz, int64_t M,
                                const double* tx, const double* ty, const double* tz, double theta, int degree,
                                int leaf_size, int batch_size);
void oracle_plan_destroy(oracle_plan* p);
void oracle_plan_sizes(const oracle_plan* p, int64_t* s);
int oracle_bltc_eval(const oracle_plan* p, int kind, const double* w, const double* f_src, const double* f_tgt, double k,
                     int subtract, int finalize, int64_t nsel, const int64_t* sel, double* out, double* parts);
int oracle_bltc_eval_coulomb(const oracle_plan* p, const double* w, const double* f_src, const double* f_tgt,
                             double alpha, int subtract, int64_t nsel, const int64_t* sel, double* out, double* parts);
int oracle_direct(int kind, int64_t M, const double* tx, const double* ty, const double* tz, const double* tf, int64_t N,
                  const double* sx, const double* sy, const double* sz, const double* sw, const double* sf, double k,
                  int subtract, int finalize, double* out);
int oracle_coulomb_direct(int64_t M, const double* tx, const double* ty, const double* tz, const double* tf, int64_t N,
                          const double* sx, const double* sy, const double* sz, const double* sw, const double* sf,
                          double alpha, int subtract, double* out);
}

// Invariants of the B200 work decomposition (plan_host.cpp plan_finish): for every batch and every list segment the
// tiles cover each target exactly once, a tile is 2^gshift full groups (or one narrower tail group), every item's list
// slice is valid, and the items' slices of the partial-sum buffer are disjoint and fill [0, partial_len).
static bool check_decomposition(const bltc::HostPlan& p) {
    using namespace bltc;
    std::vector<char> used((size_t)p.partial_len, 0);
    auto check_items = [&](const std::vector<WorkItem>& items, size_t list_size) {
        for (const WorkItem& w : items) {
            if (w.list_begin < 0 || w.list_end > (int32_t)list_size || w.list_begin >= w.list_end) return false;
            if (w.gshift < 0 || (1 << w.gshift) > kTileGroupsMax || w.rshift < 0 || (kTargetsPerThread >> w.rshift) < 1) return false;
            const int cap = 32 * (kTargetsPerThread >> w.rshift) << w.gshift;
            if (w.tgt_count < 1 || w.tgt_count > cap) return false;
            if (w.rshift > 0 && w.gshift != 0) return false;
            if (w.gshift > 0 && w.tgt_count <= cap / 2) return false;            // no empty groups in a tile
            if (w.partial_off < 0 || w.partial_off + w.tgt_count > p.partial_len) return false;
            for (int32_t i = 0; i < w.tgt_count; ++i) {
                if (used[(size_t)w.partial_off + i]) return false;                // slices are disjoint
                used[(size_t)w.partial_off + i] = 1;
            }
        }
        return true;
    };
    if (!check_items(p.far_items, p.far_slots.size()) || !check_items(p.near_items, p.near_ranges.size())) return false;
    for (char u : used) if (!u) return false;                                     // ... and cover the buffer
    int64_t expect = 0;
    for (int b = p.shard_b0; b < p.shard_b1; ++b) {
        if (p.b_partial_base[b] != expect) return false;
        expect += (int64_t)(p.b_nseg_far[b] + p.b_nseg_near[b]) * (p.b_end[b] - p.b_begin[b]);
    }
    if (expect != p.partial_len) return false;
    // near segments of a batch: their ranges add up to the batch's near sources, each source once
    int64_t near_src = 0, listed = 0;
    for (const Range& r : p.near_ranges) { if (r.end <= r.begin) return false; near_src += r.end - r.begin; }
    for (int b = p.shard_b0; b < p.shard_b1; ++b)
        for (int64_t q = p.near_ptr[b]; q < p.near_ptr[b + 1]; ++q) listed += p.src.cl[p.near_idx[q]].end - p.src.cl[p.near_idx[q]].begin;
    return near_src == listed && (int64_t)p.far_slots.size() == p.far_ptr[p.shard_b1] - p.far_ptr[p.shard_b0];
}

static uint64_t rng_state = 20030183;
static double urand() {                      // splitmix64
    uint64_t z = (rng_state += 0x9e3779b97f4a7c15ull);
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
    z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
    return (double)((z ^ (z >> 31)) >> 11) / 9007199254740992.0;
}

int main() {
    struct Case { int64_t N; int leaf, batch, degree, shape, world; double theta; };
    const Case cases[] = {
        {1, 1, 1, 1, 0, 1, 0.5},       {3, 1, 2, 2, 0, 2, 0.7},      {257, 7, 7, 3, 1, 3, 0.7},   {1000, 32, 5, 4, 2, 1, 0.95},
        {2500, 100, 100, 5, 3, 4, 0.3}, {4000, 300, 300, 2, 0, 1, 0.0}, {6000, 50, 200, 3, 0, 8, 0.8},
    };
    for (const Case& c : cases) {
        const int64_t N = c.N;
        std::vector<double> X(3 * N), w(N), f(N), out(N), out2(N);
        for (int64_t i = 0; i < 3 * N; ++i) X[i] = urand();
        if (c.shape == 1) for (int64_t i = 0; i < N; ++i) X[2 * N + i] = 0.25;                       // planar
        if (c.shape == 2) for (int64_t i = 0; i < N; ++i) { X[N + i] = X[i]; X[2 * N + i] = 0.5; }   // collinear
        if (c.shape == 3) for (int64_t i = N / 2; i < N; ++i)                                        // duplicates
            for (int d = 0; d < 3; ++d) X[d * N + i] = X[d * N + i - N / 2];
        for (int64_t i = 0; i < N; ++i) { w[i] = urand() / (double)N; f[i] = 2.0 * urand() - 1.0; }
        int64_t far_evals = -1, near_evals = -1;
        for (int r = 0; r < 2 * c.world; ++r) {             // both upward-pass modes (slots of the child -> parent pass)
            bltc::HostPlan p;
            bltc::build_host_plan(p, nullptr, X.data(), N, c.theta, c.degree, c.batch, c.leaf, 148, r % c.world, c.world,
                                  r >= c.world);
            for (size_t lv = 0; lv + 1 < p.c2p_level_ptr.size(); ++lv)
                for (int32_t i = p.c2p_level_ptr[lv]; i < p.c2p_level_ptr[lv + 1]; ++i) {
                    const bltc::C2PItem& it = p.c2p_items[i];
                    const int level = p.src.cl[p.cluster_of_slot[it.parent]].level;
                    if (it.nchild < 2 || it.nchild > 8) { std::printf("bad child count\n"); return 1; }
                    for (int q = 0; q < it.nchild; ++q)          // children have slots, one level deeper, and come earlier
                        if (it.child[q] < 0 || p.src.cl[p.cluster_of_slot[it.child[q]]].level != level + 1 ||
                            p.src.cl[p.cluster_of_slot[it.child[q]]].parent != p.cluster_of_slot[it.parent]) {
                            std::printf("child -> parent item inconsistent\n"); return 1;
                        }
                    if (i > p.c2p_level_ptr[lv] && p.src.cl[p.cluster_of_slot[p.c2p_items[i - 1].parent]].level != level) {
                        std::printf("levels mixed\n"); return 1;
                    }
                }
            far_evals = p.far_evals; near_evals = p.near_evals;
            if (!check_decomposition(p)) { std::printf("work decomposition invariant broken, N=%lld rank %d\n", (long long)N, r); return 1; }
        }
        oracle_plan* op = oracle_plan_create(N, X.data(), X.data() + N, X.data() + 2 * N, 0, nullptr, nullptr, nullptr,
                                             c.theta, c.degree, c.leaf, c.batch);
        if (!op) { std::printf("oracle_plan_create failed\n"); return 1; }
        int64_t s[8];
        oracle_plan_sizes(op, s);
        if (s[5] != far_evals || s[6] != near_evals) { std::printf("plan mismatch N=%lld\n", (long long)N); return 1; }
        if (oracle_bltc_eval(op, 0, w.data(), f.data(), f.data(), 1.3, 1, 1, 0, nullptr, out.data(), nullptr)) return 1;
        if (oracle_bltc_eval_coulomb(op, w.data(), f.data(), f.data(), 0.4, 1, 0, nullptr, out2.data(), nullptr)) return 1;
        oracle_plan_destroy(op);
        if (N <= 2500) {
            std::vector<double> ds(N);
            if (oracle_direct(0, N, X.data(), X.data() + N, X.data() + 2 * N, f.data(), N, X.data(), X.data() + N,
                              X.data() + 2 * N, w.data(), f.data(), 1.3, 1, 1, ds.data())) return 1;
            if (c.theta == 0.0 || c.N <= 3) {      // all-direct lists: the treecode is the definition
                for (int64_t i = 0; i < N; ++i)
                    if (std::fabs(ds[i] - out[i]) > 1e-12 * (1.0 + std::fabs(ds[i]))) { std::printf("value mismatch\n"); return 1; }
            }
            if (oracle_coulomb_direct(N, X.data(), X.data() + N, X.data() + 2 * N, f.data(), N, X.data(), X.data() + N,
                                      X.data() + 2 * N, w.data(), f.data(), 0.4, 1, ds.data())) return 1;
        }
    }
    std::printf("sanitize ok\n");
    return 0;
}
