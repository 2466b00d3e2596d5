// plan_host.cpp -- see plan_host.hpp.  Compiled with -ffp-contract=off: every MAC and
// midpoint expression below is evaluated in plain IEEE double, in the written order, so that
// the decisions are reproducible (readings R4-R8).
#include "plan_host.hpp"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <future>
#include <numeric>
#include <stdexcept>
#include <thread>

namespace bltc {
namespace {

constexpr double kSqrt2 = 1.4142135623730951;
constexpr double kPi = 3.14159265358979323846;

// Sub-trees of different children touch disjoint ranges of perm / tmp / code, so the children of the top
// kParLevels levels are built by concurrent tasks into private cluster vectors (local ids, DFS pre-order) and
// spliced behind their parent in child order: the result is identical to the sequential build, cluster for
// cluster (stage 1 "scales worst ... due to some serial computation").
struct TreeBuilder {
    static constexpr int kParLevels = 2;                 // up to 64 concurrent sub-tree tasks
    static constexpr int64_t kParMin = 100000;           // smaller clusters are not worth a thread
    const double* c[3];
    int64_t max_leaf;
    std::vector<int64_t>& perm;
    std::vector<int64_t> tmp;
    std::vector<uint8_t> code;

    TreeBuilder(std::vector<int64_t>& perm_, const double* x, const double* y, const double* z, int64_t n, int64_t ml)
        : c{x, y, z}, max_leaf(ml), perm(perm_), tmp(n), code(n) {
        perm.resize(n);
        std::iota(perm.begin(), perm.end(), int64_t(0));
    }

    // Appends the cluster of [b, e) to `out` and returns its id; fills count/first with the split (all counts 0:
    // the cluster is a leaf).  PAPER.md:378: bisection at the box midpoint, children shrunk to their particles.
    int make_cluster(int64_t b, int64_t e, int parent, int level, std::vector<Cluster>& out, int64_t count[8],
                     int64_t first[8]) {
        const int id = (int)out.size();
        out.emplace_back();
        Cluster& C = out.back();
        C.begin = b; C.end = e; C.parent = parent; C.level = level;
        for (int d = 0; d < 3; ++d) {
            double lo = c[d][perm[b]], hi = lo;
            for (int64_t i = b + 1; i < e; ++i) {
                const double v = c[d][perm[i]];
                lo = v < lo ? v : lo;
                hi = v > hi ? v : hi;
            }
            C.lo[d] = lo; C.hi[d] = hi;
        }
        for (int q = 0; q < 8; ++q) count[q] = 0;
        if (e - b <= max_leaf) return id;                         // R4: leaf iff count <= N_L
        double ext[3], longest = 0.0, mid[3];
        bool cut[3];
        int ncut = 0;
        for (int d = 0; d < 3; ++d) {
            ext[d] = C.hi[d] - C.lo[d];
            longest = ext[d] > longest ? ext[d] : longest;
        }
        for (int d = 0; d < 3; ++d) {                             // R5: aspect-ratio rule sqrt(2)
            cut[d] = ext[d] > 0.0 && ext[d] * kSqrt2 >= longest;
            ncut += cut[d];
            mid[d] = 0.5 * (C.lo[d] + C.hi[d]);
        }
        if (ncut == 0) return id;                                 // all particles coincide
        for (int64_t i = b; i < e; ++i) {
            const int64_t p = perm[i];
            uint8_t k = 0;
            if (cut[0] && c[0][p] > mid[0]) k |= 1;               // bit0 x, bit1 y, bit2 z
            if (cut[1] && c[1][p] > mid[1]) k |= 2;
            if (cut[2] && c[2][p] > mid[2]) k |= 4;
            code[i] = k;
            ++count[k];
        }
        int live = 0;
        for (int q = 0; q < 8; ++q) live += count[q] != 0;
        if (live < 2) {                                           // midpoint rounded onto a face
            for (int q = 0; q < 8; ++q) count[q] = 0;
            return id;
        }
        int64_t cur[8];
        int64_t at = b;
        for (int q = 0; q < 8; ++q) { first[q] = cur[q] = at; at += count[q]; }
        for (int64_t i = b; i < e; ++i) tmp[cur[code[i]]++] = perm[i];     // stable
        std::copy(tmp.begin() + b, tmp.begin() + e, perm.begin() + b);
        return id;
    }

    int subdivide(int64_t b, int64_t e, int parent, int level, int par_levels, std::vector<Cluster>& out) {
        int64_t count[8], first[8];
        const int id = make_cluster(b, e, parent, level, out, count, first);
        if (par_levels > 0 && e - b >= kParMin) {
            std::vector<Cluster> frag[8];
            std::vector<std::future<void>> tasks;
            for (int q = 0; q < 8; ++q) {
                if (!count[q]) continue;                          // empty children dropped
                tasks.push_back(std::async(std::launch::async, [this, &frag, q, &first, &count, level, par_levels] {
                    subdivide(first[q], first[q] + count[q], -1, level + 1, par_levels - 1, frag[q]);
                }));
            }
            for (auto& t : tasks) t.get();
            for (int q = 0; q < 8; ++q) {
                if (!count[q]) continue;
                const int base = (int)out.size();
                for (Cluster C : frag[q]) {
                    C.parent = C.parent < 0 ? id : C.parent + base;
                    for (int k = 0; k < C.nchild; ++k) C.child[k] += base;
                    out.push_back(C);
                }
                Cluster& P = out[id];
                P.child[P.nchild++] = base;
            }
            return id;
        }
        for (int q = 0; q < 8; ++q) {
            if (!count[q]) continue;                              // empty children dropped
            const int ch = subdivide(first[q], first[q] + count[q], id, level + 1, 0, out);
            Cluster& C = out[id];
            C.child[C.nchild++] = ch;
        }
        return id;
    }
};

void gather_leaves(const Tree& t, int id, std::vector<int>& out) {
    if (t.cl[id].nchild == 0) { out.push_back(id); return; }
    for (int q = 0; q < t.cl[id].nchild; ++q) gather_leaves(t, t.cl[id].child[q], out);
}

}  // namespace

void build_tree(Tree& t, const double* x, const double* y, const double* z, int64_t n, int64_t max_leaf) {
    t.cl.clear();
    TreeBuilder tb(t.perm, x, y, z, n, max_leaf);
    tb.subdivide(0, n, -1, 0, TreeBuilder::kParLevels, t.cl);
    t.leaves.clear();
    gather_leaves(t, 0, t.leaves);
}

namespace {

inline double half_diagonal(const double* lo, const double* hi) {
    const double ex = hi[0] - lo[0], ey = hi[1] - lo[1], ez = hi[2] - lo[2];
    return 0.5 * std::sqrt((ex * ex + ey * ey) + ez * ez);
}

// Algorithm 3 ComputePotential, decision part only (text PAPER.md:434).
struct Traversal {
    const HostPlan& p;
    const double* blo; const double* bhi;
    double rB;
    std::vector<int32_t>& far; std::vector<int32_t>& near;

    void visit(int c) {
        const Cluster& C = p.src.cl[c];
        const double rC = half_diagonal(C.lo, C.hi);
        const double dx = 0.5 * (blo[0] + bhi[0]) - 0.5 * (C.lo[0] + C.hi[0]);
        const double dy = 0.5 * (blo[1] + bhi[1]) - 0.5 * (C.lo[1] + C.hi[1]);
        const double dz = 0.5 * (blo[2] + bhi[2]) - 0.5 * (C.lo[2] + C.hi[2]);
        const double R = std::sqrt((dx * dx + dy * dy) + dz * dz);
        const bool separated = (rB + rC) < p.theta * R;           // Eq. (36) left, R6
        bool big = (int64_t)p.P < (C.end - C.begin);              // Eq. (36) right
        if (C.hi[0] == C.lo[0] || C.hi[1] == C.lo[1] || C.hi[2] == C.lo[2]) big = false;   // R8
        if (separated && big) { far.push_back(c); return; }
        if (!separated) {
            if (C.nchild == 0) { near.push_back(c); return; }
            for (int q = 0; q < C.nchild; ++q) visit(C.child[q]);
            return;
        }
        near.push_back(c);                                        // R10: whole cluster, no descent
    }
};

int ilog2_floor(int v) { int s = 0; while ((2 << s) <= v) ++s; return s; }

// Tiles of a batch: binary decomposition of its target groups into tiles of 8/4/2/1 groups,
// so every warp of a CTA has work (S = kPairWarps / groups source-split ways).
void make_tiles(int64_t tb, int64_t te, std::vector<std::pair<int32_t, int32_t>>& tiles,
                std::vector<int>& gshift, std::vector<int>& rshift) {
    tiles.clear(); gshift.clear(); rshift.clear();
    constexpr int unit = 32 * kTargetsPerThread;
    // The ragged tail (rem < unit targets) is covered by single narrower groups of 32 (R >> rs) targets, the widest
    // first, so that fewer than 32 lanes are wasted; a tail that needs the full width anyway is just the last
    // (partial) group of the regular tiles.
    const int64_t rem0 = (te - tb) % unit;
    int64_t pos = tb;
    int groups = (int)((te - tb) / unit) + ((rem0 > unit - 32) ? 1 : 0);      // full groups (+ a tail wasting < 32 lanes)
    while (groups > 0) {
        const int g = std::min(kTileGroupsMax, 1 << ilog2_floor(groups));
        const int64_t cnt = std::min<int64_t>((int64_t)g * unit, te - pos);
        tiles.emplace_back((int32_t)pos, (int32_t)cnt);
        gshift.push_back(ilog2_floor(g));
        rshift.push_back(0);
        pos += cnt; groups -= g;
    }
    int64_t rem = te - pos;
    while (rem > 0) {
        int rs = 0;                                               // narrowest group that still holds rem
        while ((kTargetsPerThread >> (rs + 1)) >= 1 && (int64_t)(unit >> (rs + 1)) >= rem) ++rs;
        int64_t cap = unit >> rs;
        if (cap - rem >= 32 && (kTargetsPerThread >> (rs + 1)) >= 1) { ++rs; cap = unit >> rs; }   // fill a narrower one first
        const int64_t cnt = std::min(cap, rem);
        tiles.emplace_back((int32_t)pos, (int32_t)cnt);
        gshift.push_back(0);
        rshift.push_back(rs);
        pos += cnt; rem -= cnt;
    }
}

}  // namespace

std::vector<int> shard_cuts(const std::vector<int64_t>& batch_cost, int world) {
    const int nb = (int)batch_cost.size();
    long double total = 0;
    for (int64_t c : batch_cost) total += (long double)c;
    std::vector<int> cut(world + 1, nb);
    cut[0] = 0;
    long double acc = 0;
    int r = 1;
    for (int b = 0; b < nb && r < world; ++b) {
        // batch b goes to the slice in which the midpoint of its cost interval falls
        const long double mid = acc + 0.5L * (long double)batch_cost[b];
        while (r < world && mid >= total * (long double)r / (long double)world) cut[r++] = b;
        acc += (long double)batch_cost[b];
    }
    for (int i = 1; i <= world; ++i) cut[i] = std::max(cut[i], cut[i - 1]);
    return cut;
}

void plan_begin(HostPlan& p, int64_t N, bool same_points, double theta, int degree, int batch_size, int leaf_size,
                bool upward_children) {
    if (N <= 0 || N > (int64_t)2000000000) throw std::invalid_argument("N must be in [1, 2e9]");
    if (!(theta >= 0.0) || !(theta < 1.0)) throw std::invalid_argument("theta must be in [0, 1)");
    if (degree < 1 || degree > 20) throw std::invalid_argument("interp_degree must be in [1, 20]");
    if (batch_size < 1 || leaf_size < 1) throw std::invalid_argument("batch_size and leaf_size must be >= 1");
    p = HostPlan();
    p.N = N; p.M = N; p.theta = theta; p.degree = degree;
    p.P = (degree + 1) * (degree + 1) * (degree + 1);
    p.leaf_size = leaf_size; p.batch_size = batch_size;
    p.same_points = same_points;
    p.shared_order = same_points && batch_size == leaf_size;
    p.upward_children = upward_children;
}

void plan_set_batches(HostPlan& p) {
    const Tree* bt = p.shared_order ? &p.src : &p.tgt;
    {   // bound of |target - source|: farthest corners of the two root boxes
        const Cluster& A = p.src.cl[0];
        const Cluster& B = bt->cl[0];
        double d2 = 0.0;
        for (int d = 0; d < 3; ++d) {
            const double e = std::max(A.hi[d], B.hi[d]) - std::min(A.lo[d], B.lo[d]);
            d2 += e * e;
        }
        p.max_dist = std::sqrt(d2);
    }
    const int nb = (int)bt->leaves.size();
    p.b_begin.resize(nb); p.b_end.resize(nb); p.b_lo.resize(3 * (size_t)nb); p.b_hi.resize(3 * (size_t)nb);
    for (int b = 0; b < nb; ++b) {
        const Cluster& L = bt->cl[bt->leaves[b]];
        p.b_begin[b] = L.begin; p.b_end[b] = L.end;
        for (int d = 0; d < 3; ++d) { p.b_lo[3 * b + d] = L.lo[d]; p.b_hi[3 * b + d] = L.hi[d]; }
    }
}

// Algorithm 3 line 3, decisions: per-batch interaction lists ("precomputed for each target batch")
// for the batches [b0, b1), written at the CSR offsets far_ptr / near_ptr (which must be set).  Batches are
// independent: contiguous chunks of them are traversed by concurrent tasks.

void plan_lists_host(HostPlan& p, std::vector<int64_t>& b_far_evals, std::vector<int64_t>& b_near_evals) {
    const int nb = (int)p.b_begin.size();
    p.far_ptr.assign(nb + 1, 0); p.near_ptr.assign(nb + 1, 0);
    b_far_evals.assign(nb, 0); b_near_evals.assign(nb, 0);
    const int hw = (int)std::max(1u, std::thread::hardware_concurrency());
    const int nchunk = std::max(1, std::min(hw, nb / 64));
    std::vector<std::vector<int32_t>> cfar(nchunk), cnear(nchunk);
    std::vector<int64_t> nfar(nb, 0), nnear(nb, 0);
    auto work = [&](int ch) {
        const int b0 = (int)((int64_t)nb * ch / nchunk), b1 = (int)((int64_t)nb * (ch + 1) / nchunk);
        for (int b = b0; b < b1; ++b) {
            const size_t f0 = cfar[ch].size(), n0 = cnear[ch].size();
            Traversal tr{p, &p.b_lo[3 * b], &p.b_hi[3 * b], half_diagonal(&p.b_lo[3 * b], &p.b_hi[3 * b]),
                         cfar[ch], cnear[ch]};
            tr.visit(0);
            nfar[b] = (int64_t)(cfar[ch].size() - f0); nnear[b] = (int64_t)(cnear[ch].size() - n0);
            const int64_t nt = p.b_end[b] - p.b_begin[b];
            b_far_evals[b] = nt * p.P * nfar[b];
            for (size_t q = n0; q < cnear[ch].size(); ++q)
                b_near_evals[b] += nt * (p.src.cl[cnear[ch][q]].end - p.src.cl[cnear[ch][q]].begin);
        }
    };
    if (nchunk == 1) work(0);
    else {
        std::vector<std::future<void>> tasks;
        for (int ch = 0; ch < nchunk; ++ch) tasks.push_back(std::async(std::launch::async, work, ch));
        for (auto& t : tasks) t.get();
    }
    for (int b = 0; b < nb; ++b) {
        p.far_ptr[b + 1] = p.far_ptr[b] + nfar[b]; p.near_ptr[b + 1] = p.near_ptr[b] + nnear[b];
    }
    p.far_idx.clear(); p.near_idx.clear();
    p.far_idx.reserve((size_t)p.far_ptr[nb]); p.near_idx.reserve((size_t)p.near_ptr[nb]);
    for (int ch = 0; ch < nchunk; ++ch) {
        p.far_idx.insert(p.far_idx.end(), cfar[ch].begin(), cfar[ch].end());
        p.near_idx.insert(p.near_idx.end(), cnear[ch].begin(), cnear[ch].end());
    }
    p.lists_b0 = 0; p.lists_b1 = nb;
}

void plan_set_shard(HostPlan& p, const std::vector<int64_t>& b_far_evals, const std::vector<int64_t>& b_near_evals,
                    int shard_rank, int shard_world) {
    if (shard_world < 1 || shard_rank < 0 || shard_rank >= shard_world)
        throw std::invalid_argument("shard rank/world must satisfy 0 <= rank < world");
    const int nb = (int)p.b_begin.size();
    p.far_evals = p.near_evals = 0;
    std::vector<int64_t> cost(nb);
    for (int b = 0; b < nb; ++b) {
        p.far_evals += b_far_evals[b]; p.near_evals += b_near_evals[b];
        cost[b] = b_far_evals[b] + b_near_evals[b];
    }
    // batch slice of this rank: equal shares of the kernel evaluations (the batches are independent given
    // the sources and the proxy charges)
    p.shard_rank = shard_rank; p.shard_world = shard_world;
    const std::vector<int> cut = shard_cuts(cost, shard_world);
    p.shard_b0 = cut[shard_rank]; p.shard_b1 = cut[shard_rank + 1];
    p.shard_far_evals = p.shard_near_evals = 0;
    for (int b = p.shard_b0; b < p.shard_b1; ++b) {
        p.shard_far_evals += b_far_evals[b]; p.shard_near_evals += b_near_evals[b];
    }
}

// Everything after the lists of the batches [shard_b0, shard_b1) are known: proxy slots with their Chebyshev grids,
// upward-pass work items, and the B200 work decomposition.
void plan_finish(HostPlan& p, int sm_count) {
    const int nb = (int)p.b_begin.size();
    const int B0 = p.shard_b0, B1 = p.shard_b1;
    const int degree = p.degree;
    if (B0 < p.lists_b0 || B1 > p.lists_b1) throw std::logic_error("plan_finish: lists of the shard's batches are missing");

    // proxy slots: clusters that appear in some far list (R9), with their Chebyshev grids Eq. (37).  With the
    // child -> parent upward pass (R23) an internal cluster's charges come from its children's, so the children get
    // slots too (recursively); a cluster with a child whose box is flat on an axis (R8: no grid) and every leaf
    // take their charges from their own particles.
    const int ncl = (int)p.src.cl.size();
    const int n1 = degree + 1;
    p.slot_of_cluster.assign(ncl, -1);
    for (int64_t q = p.far_ptr[B0]; q < p.far_ptr[B1]; ++q) p.slot_of_cluster[p.far_idx[q]] = 0;   // local batches' far lists
    auto flat = [&](const Cluster& C) { return C.hi[0] == C.lo[0] || C.hi[1] == C.lo[1] || C.hi[2] == C.lo[2]; };
    auto from_children = [&](int c) {
        const Cluster& C = p.src.cl[c];
        if (!p.upward_children || C.nchild == 0) return false;
        for (int q = 0; q < C.nchild; ++q) if (flat(p.src.cl[C.child[q]])) return false;
        return true;
    };
    if (p.upward_children)
        for (int c = 0; c < ncl; ++c)                              // pre-order: parents before children
            if (p.slot_of_cluster[c] == 0 && from_children(c))
                for (int q = 0; q < p.src.cl[c].nchild; ++q) p.slot_of_cluster[p.src.cl[c].child[q]] = 0;
    int max_level = 0;
    for (int c = 0; c < ncl; ++c)
        if (p.slot_of_cluster[c] == 0) {
            p.slot_of_cluster[c] = (int32_t)p.cluster_of_slot.size();
            p.cluster_of_slot.push_back(c);
            if (!from_children(c)) p.upward_pairs += p.src.cl[c].end - p.src.cl[c].begin;
            max_level = std::max(max_level, p.src.cl[c].level);
        }
    p.c2p_level_ptr.assign(1, 0);
    if (p.upward_children)
        for (int level = max_level; level >= 0; --level) {
            for (size_t s = 0; s < p.cluster_of_slot.size(); ++s) {
                const int c = p.cluster_of_slot[s];
                const Cluster& C = p.src.cl[c];
                if (C.level != level || !from_children(c)) continue;
                C2PItem it{(int32_t)s, C.nchild, {0, 0, 0, 0, 0, 0, 0, 0}};
                for (int q = 0; q < C.nchild; ++q) it.child[q] = p.slot_of_cluster[C.child[q]];
                p.c2p_items.push_back(it);
            }
            if ((int32_t)p.c2p_items.size() > p.c2p_level_ptr.back()) p.c2p_level_ptr.push_back((int32_t)p.c2p_items.size());
        }
    p.slot_nodes.resize(p.cluster_of_slot.size() * 3 * (size_t)n1);
    for (size_t s = 0; s < p.cluster_of_slot.size(); ++s) {
        const Cluster& C = p.src.cl[p.cluster_of_slot[s]];
        for (int d = 0; d < 3; ++d) {
            const double mid = 0.5 * (C.lo[d] + C.hi[d]);
            const double half = 0.5 * (C.hi[d] - C.lo[d]);
            for (int k = 0; k < n1; ++k)
                p.slot_nodes[(s * 3 + d) * n1 + k] = mid + half * std::cos((kPi * k) / degree);
        }
    }

    // upward-pass work items: clusters are cut into chunks so that ~16 CTAs exist per SM and no CTA
    // carries a root-level cluster alone; chunk partials are summed in chunk order (deterministic)
    {
        const int64_t want = (int64_t)std::max(1, sm_count) * 16;
        const int64_t chunk = std::min<int64_t>(8192, std::max<int64_t>(512, (p.upward_pairs + want - 1) / want));
        for (size_t s = 0; s < p.cluster_of_slot.size(); ++s) {
            if (from_children(p.cluster_of_slot[s])) continue;     // filled by the child -> parent pass
            const Cluster& C = p.src.cl[p.cluster_of_slot[s]];
            const int64_t n = C.end - C.begin;
            const int64_t nch = std::max<int64_t>(1, (n + chunk - 1) / chunk);
            if (nch == 1) {
                p.up_items.push_back(UpItem{(int32_t)s, (int32_t)C.begin, (int32_t)C.end, -1});
                continue;
            }
            p.up_reduce.push_back(UpReduce{(int32_t)s, (int32_t)p.up_partial_chunks, (int32_t)nch});
            for (int64_t c = 0; c < nch; ++c)
                p.up_items.push_back(UpItem{(int32_t)s, (int32_t)(C.begin + n * c / nch),
                                            (int32_t)(C.begin + n * (c + 1) / nch), (int32_t)p.up_partial_chunks++});
        }
        std::stable_sort(p.up_items.begin(), p.up_items.end(), [](const UpItem& a, const UpItem& c) {
            return (a.end - a.begin) > (c.end - c.begin);
        });
    }

    // ---- B200 work decomposition -------------------------------------------------------
    // Per batch: near clusters -> merged contiguous source ranges; far clusters -> slot ids.
    // Lists are cut into segments so that (tiles x segments) gives >= ~32 work items per
    // resident CTA slot (2 CTAs/SM), each CTA slot then sees many items sorted by cost.
    // Batches are independent: chunks of them are decomposed by concurrent tasks into private vectors
    // (indices relative to the chunk) that are spliced in batch order afterwards.
    const int cta_slots = std::max(1, sm_count) * 2;
    double near_cost = 0, far_cost = 0;            // in (target group of 64) x (source) units
    std::vector<int64_t> near_src(nb, 0);
    for (int b = B0; b < B1; ++b) {
        for (int64_t q = p.near_ptr[b]; q < p.near_ptr[b + 1]; ++q)
            near_src[b] += p.src.cl[p.near_idx[q]].end - p.src.cl[p.near_idx[q]].begin;
        const double groups = (double)((p.b_end[b] - p.b_begin[b] + 63) / 64);      // cost unit: 64 targets x 1 source
        near_cost += groups * (double)near_src[b];
        far_cost += groups * (double)(p.far_ptr[b + 1] - p.far_ptr[b]) * p.P;
    }
    const double near_cap = std::max(512.0, near_cost / (cta_slots * 32.0 * 8.0));
    const double far_cap = std::max((double)p.P, far_cost / (cta_slots * 32.0 * 8.0));

    p.b_nseg_far.assign(nb, 0); p.b_nseg_near.assign(nb, 0); p.b_partial_base.assign(nb, 0);
    struct Chunk {
        std::vector<Range> ranges; std::vector<int32_t> slots; std::vector<WorkItem> far_items, near_items;
        std::vector<int64_t> near_key; int64_t partial = 0;
    };
    const int hw = (int)std::max(1u, std::thread::hardware_concurrency());
    const int nchunk = std::max(1, std::min(hw, (B1 - B0) / 32));
    std::vector<Chunk> chunks(nchunk);
    auto decompose = [&](int ch) {
        Chunk& K = chunks[ch];
        const int c0 = B0 + (int)((int64_t)(B1 - B0) * ch / nchunk), c1 = B0 + (int)((int64_t)(B1 - B0) * (ch + 1) / nchunk);
        std::vector<Range> r;
        std::vector<std::pair<int32_t, int32_t>> tiles, nseg_slices, fseg_slices; std::vector<int> gsh, hf;
        for (int b = c0; b < c1; ++b) {
            r.clear();
            for (int64_t q = p.near_ptr[b]; q < p.near_ptr[b + 1]; ++q) {
                const Cluster& C = p.src.cl[p.near_idx[q]];
                // can a source of C coincide with a target of the batch?  Only if the (closed, minimal)
                // bounding boxes intersect; otherwise the kernel skips the r == 0 test (reading R3).
                bool touch = true;
                for (int d = 0; d < 3; ++d)
                    touch = touch && C.lo[d] <= p.b_hi[3 * b + d] && p.b_lo[3 * b + d] <= C.hi[d];
                r.push_back(Range{(int32_t)C.begin, (int32_t)C.end, touch ? kRangeMayCoincide : 0});
            }
            std::sort(r.begin(), r.end(), [](const Range& a, const Range& c) { return a.begin < c.begin; });
            size_t o = 0;
            for (size_t i = 0; i < r.size(); ++i) {
                if (o > 0 && r[o - 1].end == r[i].begin && r[o - 1].flags == r[i].flags) r[o - 1].end = r[i].end;
                else r[o++] = r[i];
            }
            r.resize(o);
            const int64_t nt = p.b_end[b] - p.b_begin[b];
            // near segments: equal source counts, ranges may be cut anywhere
            nseg_slices.clear();    // [begin, end) into the chunk's ranges
            if (near_src[b] > 0) {
                int nseg = (int)std::min<int64_t>(64, (int64_t)std::ceil((double)near_src[b] / near_cap));
                nseg = std::max(1, nseg);
                const int64_t per = (near_src[b] + nseg - 1) / nseg;
                int64_t room = per;
                int32_t seg_start = (int32_t)K.ranges.size();
                for (const Range& g : r) {
                    int32_t at = g.begin;
                    while (at < g.end) {
                        const int32_t take = (int32_t)std::min<int64_t>(room, g.end - at);
                        K.ranges.push_back(Range{at, at + take, g.flags});
                        at += take; room -= take;
                        if (room == 0) {
                            nseg_slices.emplace_back(seg_start, (int32_t)K.ranges.size());
                            seg_start = (int32_t)K.ranges.size(); room = per;
                        }
                    }
                }
                if ((int32_t)K.ranges.size() > seg_start)
                    nseg_slices.emplace_back(seg_start, (int32_t)K.ranges.size());
            }
            // far segments: whole clusters
            fseg_slices.clear();
            const int64_t nfar = p.far_ptr[b + 1] - p.far_ptr[b];
            if (nfar > 0) {
                const int64_t per = std::max<int64_t>(1, (int64_t)(far_cap / p.P));
                int64_t nseg = std::min<int64_t>(64, (nfar + per - 1) / per);
                const int64_t per2 = (nfar + nseg - 1) / nseg;
                for (int64_t q = 0; q < nfar; q += per2) {
                    const int32_t s0 = (int32_t)K.slots.size();
                    for (int64_t u = q; u < std::min(nfar, q + per2); ++u)
                        K.slots.push_back(p.slot_of_cluster[p.far_idx[p.far_ptr[b] + u]]);
                    fseg_slices.emplace_back(s0, (int32_t)K.slots.size());
                }
            }
            p.b_nseg_far[b] = (int32_t)fseg_slices.size();
            p.b_nseg_near[b] = (int32_t)nseg_slices.size();
            p.b_partial_base[b] = K.partial;                      // relative to the chunk
            make_tiles(p.b_begin[b], p.b_end[b], tiles, gsh, hf);
            for (size_t ti = 0; ti < tiles.size(); ++ti) {
                const int64_t local = tiles[ti].first - p.b_begin[b];
                for (size_t s = 0; s < fseg_slices.size(); ++s)
                    K.far_items.push_back(WorkItem{tiles[ti].first, tiles[ti].second, gsh[ti],
                        fseg_slices[s].first, fseg_slices[s].second, hf[ti],
                        K.partial + (int64_t)s * nt + local});
                for (size_t s = 0; s < nseg_slices.size(); ++s) {
                    K.near_items.push_back(WorkItem{tiles[ti].first, tiles[ti].second, gsh[ti],
                        nseg_slices[s].first, nseg_slices[s].second, hf[ti],
                        K.partial + (int64_t)(fseg_slices.size() + s) * nt + local});
                    int64_t key = 0;
                    for (int32_t q = nseg_slices[s].first; q < nseg_slices[s].second; ++q)
                        key += K.ranges[q].end - K.ranges[q].begin;
                    K.near_key.push_back(key << gsh[ti]);
                }
            }
            K.partial += (int64_t)(fseg_slices.size() + nseg_slices.size()) * nt;
        }
    };
    if (nchunk == 1) decompose(0);
    else {
        std::vector<std::future<void>> tasks;
        for (int ch = 0; ch < nchunk; ++ch) tasks.push_back(std::async(std::launch::async, decompose, ch));
        for (auto& t : tasks) t.get();
    }
    // splice the chunks in batch order: chunk-relative indices become global ones
    std::vector<int64_t> near_key;
    {
        size_t nr = 0, nsl = 0, nfi = 0, nni = 0;
        for (const Chunk& K : chunks) { nr += K.ranges.size(); nsl += K.slots.size(); nfi += K.far_items.size(); nni += K.near_items.size(); }
        p.near_ranges.reserve(nr); p.far_slots.reserve(nsl); p.far_items.reserve(nfi); p.near_items.reserve(nni);
        near_key.reserve(nni);
        int64_t partial = 0;
        for (int ch = 0; ch < nchunk; ++ch) {
            Chunk& K = chunks[ch];
            const int32_t rbase = (int32_t)p.near_ranges.size(), sbase = (int32_t)p.far_slots.size();
            const int c0 = B0 + (int)((int64_t)(B1 - B0) * ch / nchunk), c1 = B0 + (int)((int64_t)(B1 - B0) * (ch + 1) / nchunk);
            for (int b = c0; b < c1; ++b) p.b_partial_base[b] += partial;
            for (WorkItem w : K.far_items) {
                w.list_begin += sbase; w.list_end += sbase; w.partial_off += partial;
                p.far_items.push_back(w);
            }
            for (WorkItem w : K.near_items) {
                w.list_begin += rbase; w.list_end += rbase; w.partial_off += partial;
                p.near_items.push_back(w);
            }
            p.near_ranges.insert(p.near_ranges.end(), K.ranges.begin(), K.ranges.end());
            p.far_slots.insert(p.far_slots.end(), K.slots.begin(), K.slots.end());
            near_key.insert(near_key.end(), K.near_key.begin(), K.near_key.end());
            partial += K.partial;
            K = Chunk();
        }
        p.partial_len = partial;
    }

    // longest-processing-time-first: the hardware block scheduler hands out CTAs in order
    auto far_cost_of = [&](const WorkItem& w) { return (int64_t)(w.list_end - w.list_begin) << w.gshift; };
    {
        std::vector<size_t> ord(near_key.size());
        std::iota(ord.begin(), ord.end(), size_t(0));
        std::stable_sort(ord.begin(), ord.end(), [&](size_t a, size_t c) { return near_key[a] > near_key[c]; });
        std::vector<WorkItem> sorted(near_key.size());
        for (size_t i = 0; i < ord.size(); ++i) sorted[i] = p.near_items[ord[i]];
        p.near_items.swap(sorted);
        std::stable_sort(p.far_items.begin(), p.far_items.end(),
                         [&](const WorkItem& a, const WorkItem& c) { return far_cost_of(a) > far_cost_of(c); });
    }
}

void build_host_plan(HostPlan& p, const double* targets, const double* sources, int64_t N,
                     double theta, int degree, int batch_size, int leaf_size, int sm_count,
                     int shard_rank, int shard_world, bool upward_children) {
    const auto t0 = std::chrono::steady_clock::now();
    if (shard_world < 1 || shard_rank < 0 || shard_rank >= shard_world)
        throw std::invalid_argument("shard rank/world must satisfy 0 <= rank < world");
    if (!sources) throw std::invalid_argument("sources is NULL");
    plan_begin(p, N, targets == nullptr || targets == sources, theta, degree, batch_size, leaf_size, upward_children);
    auto lap = [&, last = t0](int stage) mutable {
        const auto now = std::chrono::steady_clock::now();
        p.stage_ms[stage] += std::chrono::duration<double, std::milli>(now - last).count();
        last = now;
    };
    // Algorithm 3 line 1: tree of source clusters and set of target batches
    build_tree(p.src, sources, sources + N, sources + 2 * N, N, leaf_size);
    if (!p.shared_order) {
        const double* t = p.same_points ? sources : targets;
        build_tree(p.tgt, t, t + N, t + 2 * N, N, batch_size);
    }
    plan_set_batches(p);
    lap(0);
    std::vector<int64_t> b_far_evals, b_near_evals;
    plan_lists_host(p, b_far_evals, b_near_evals);
    lap(1);
    plan_set_shard(p, b_far_evals, b_near_evals, shard_rank, shard_world);
    plan_finish(p, sm_count);
    lap(3);
    p.build_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
}

}  // namespace bltc
