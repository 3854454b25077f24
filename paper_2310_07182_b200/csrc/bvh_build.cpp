// a0: host-side BVH construction for libcrt ("acceleration structures such as bounding volume
// hierarchies"; the paper leaves width, leaf size and builder open -- DESIGN.md D:R11).
// Binary tree, binned surface-area heuristic evaluated on all three axes per split, built top-down by a
// small thread pool (large ranges are split one at a time, subtrees below a size threshold run as tasks).
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <cstdlib>
#include <cstring>
#include <deque>
#include <functional>
#include <limits>
#include <mutex>
#include <thread>
#include "crt_internal.h"

namespace {

constexpr int kMaxBins = 64;

struct Box {
    float mn[3], mx[3];
    void reset() { for (int k = 0; k < 3; ++k) { mn[k] = std::numeric_limits<float>::infinity(); mx[k] = -mn[k]; } }
    void grow(const float* a, const float* b) { for (int k = 0; k < 3; ++k) { mn[k] = std::min(mn[k], a[k]); mx[k] = std::max(mx[k], b[k]); } }
    void grow(const Box& o) { grow(o.mn, o.mx); }
    double half_area() const
    {
        double dx = (double)mx[0] - mn[0], dy = (double)mx[1] - mn[1], dz = (double)mx[2] - mn[2];
        return dx * dy + dy * dz + dz * dx;
    }
};

class Pool {
public:
    explicit Pool(int n)
    {
        for (int i = 0; i < n; ++i) workers_.emplace_back([this] { run(); });
    }
    ~Pool()
    {
        { std::lock_guard<std::mutex> g(m_); stop_ = true; }
        cv_.notify_all();
        for (auto& t : workers_) t.join();
    }
    void submit(std::function<void()> f)
    {
        { std::lock_guard<std::mutex> g(m_); q_.push_back(std::move(f)); ++pending_; }
        cv_.notify_one();
    }
    void wait()
    {
        std::unique_lock<std::mutex> g(m_);
        done_.wait(g, [this] { return pending_ == 0; });
    }
private:
    void run()
    {
        for (;;) {
            std::function<void()> f;
            {
                std::unique_lock<std::mutex> g(m_);
                cv_.wait(g, [this] { return stop_ || !q_.empty(); });
                if (stop_ && q_.empty()) return;
                f = std::move(q_.front()); q_.pop_front();
            }
            f();
            { std::lock_guard<std::mutex> g(m_); if (--pending_ == 0) done_.notify_all(); }
        }
    }
    std::vector<std::thread> workers_;
    std::deque<std::function<void()>> q_;
    std::mutex m_;
    std::condition_variable cv_, done_;
    int64_t pending_ = 0;
    bool stop_ = false;
};

struct Builder {
    const float* verts; int64_t n; int max_leaf, bins; float ct, ci;
    std::vector<float> tmn, tmx, cen;      // per-triangle box and centroid
    std::vector<int32_t>& prim;
    std::vector<BuildNode>& nodes;
    std::atomic<int64_t> n_nodes{0};
    std::atomic<int> max_depth{0};
    Pool* pool;

    Builder(std::vector<int32_t>& p, std::vector<BuildNode>& nd) : prim(p), nodes(nd) {}

    int64_t alloc2() { return n_nodes.fetch_add(2); }

    void make_leaf(BuildNode& nd, int64_t lo, int64_t hi) { nd.left = nd.right = -1; nd.first = (int32_t)lo; nd.count = (int32_t)(hi - lo); }

    // builds the subtree of `node` over prim[lo,hi)
    void subtree(int64_t node, int64_t lo, int64_t hi, int depth)
    {
        for (;;) {
            Box bb, cb; bb.reset(); cb.reset();
            for (int64_t i = lo; i < hi; ++i) {
                int64_t p = prim[i];
                bb.grow(&tmn[3 * p], &tmx[3 * p]); cb.grow(&cen[3 * p], &cen[3 * p]);
            }
            BuildNode& nd = nodes[node];
            std::memcpy(nd.bmin, bb.mn, 12); std::memcpy(nd.bmax, bb.mx, 12);
            int d0 = max_depth.load(std::memory_order_relaxed);
            while (depth > d0 && !max_depth.compare_exchange_weak(d0, depth)) {}
            int64_t cnt = hi - lo;
            if (cnt <= max_leaf) { make_leaf(nd, lo, hi); return; }

            // binned SAH on the three axes in one pass
            int best_axis = -1, best_bin = -1; double best = std::numeric_limits<double>::infinity();
            int64_t bc[3][kMaxBins]; Box bx[3][kMaxBins]; float scale[3];
            for (int a = 0; a < 3; ++a) {
                float ext = cb.mx[a] - cb.mn[a];
                scale[a] = ext > 0.f ? (float)bins / ext : 0.f;
                for (int j = 0; j < bins; ++j) { bc[a][j] = 0; bx[a][j].reset(); }
            }
            for (int64_t i = lo; i < hi; ++i) {
                int64_t p = prim[i];
                for (int a = 0; a < 3; ++a) {
                    if (scale[a] == 0.f) continue;
                    int j = std::min(bins - 1, std::max(0, (int)((cen[3 * p + a] - cb.mn[a]) * scale[a])));
                    ++bc[a][j]; bx[a][j].grow(&tmn[3 * p], &tmx[3 * p]);
                }
            }
            for (int a = 0; a < 3; ++a) {
                if (scale[a] == 0.f) continue;
                double ra[kMaxBins]; int64_t rc[kMaxBins]; Box acc; acc.reset(); int64_t c = 0;
                for (int j = bins - 1; j >= 1; --j) { acc.grow(bx[a][j]); c += bc[a][j]; rc[j] = c; ra[j] = c ? acc.half_area() : 0.0; }
                acc.reset(); c = 0;
                for (int j = 0; j + 1 < bins; ++j) {
                    acc.grow(bx[a][j]); c += bc[a][j];
                    if (c == 0 || rc[j + 1] == 0) continue;
                    double cost = acc.half_area() * (double)c + ra[j + 1] * (double)rc[j + 1];
                    if (cost < best) { best = cost; best_axis = a; best_bin = j; }
                }
            }
            int64_t mid;
            if (best_axis < 0) {
                mid = lo + cnt / 2;
            } else {
                const int a = best_axis; const float c0 = cb.mn[a], sc = scale[a];
                auto it = std::partition(prim.begin() + lo, prim.begin() + hi, [&](int32_t p) {
                    int j = std::min(bins - 1, std::max(0, (int)((cen[3 * (int64_t)p + a] - c0) * sc)));
                    return j <= best_bin;
                });
                mid = it - prim.begin();
                if (mid == lo || mid == hi) mid = lo + cnt / 2;
            }
            int64_t c = alloc2();
            nd.left = (int32_t)c; nd.right = (int32_t)(c + 1); nd.count = 0; nd.first = 0;
            int64_t rlo = mid, rhi = hi; int rd = depth + 1;
            if (pool && (rhi - rlo) >= 4096) {
                pool->submit([this, c, rlo, rhi, rd] { subtree(c + 1, rlo, rhi, rd); });
            } else {
                subtree(c + 1, rlo, rhi, rd);
            }
            node = c; hi = mid; ++depth;       // continue with the left child in this thread
        }
    }
};

// ---- triangle pre-splitting (crt_bvh_params.presplit; "early split clipping", Ernst & Greiner 2007) ------------------------------------
// A triangle much larger than the scene's detail (a wall, a floor) has a box that overlaps thousands of small objects: every ray that passes
// near it tests it and the nodes above it cannot separate what lies on its two sides.  Such a triangle is given SEVERAL references, each with the
// box of the part of the triangle inside one cell of a recursive midpoint split of its box; the tree is built over references.  The triangle
// itself is unchanged (same record, same id, tested whole), so the result of a traversal is the same nearest hit; only which boxes lead to it.
struct Ref { float mn[3], mx[3]; int32_t prim; };

float round_down(double d) { float f = (float)d; return (double)f > d ? std::nextafterf(f, -std::numeric_limits<float>::infinity()) : f; }
float round_up(double d) { float f = (float)d; return (double)f < d ? std::nextafterf(f, std::numeric_limits<float>::infinity()) : f; }

struct Poly { int n; double v[10][3]; };      // a triangle clipped by axis-aligned planes: convex, at most 3 + 6 vertices

// the part of `in` on the side s * (x[axis] - pos) <= 0 (Sutherland-Hodgman against one plane)
void clip(const Poly& in, int axis, double pos, double s, Poly& out)
{
    out.n = 0;
    for (int i = 0; i < in.n; ++i) {
        const double* a = in.v[i]; const double* b = in.v[(i + 1) % in.n];
        const double da = s * (a[axis] - pos), db = s * (b[axis] - pos);
        if (da <= 0 && out.n < 10) std::memcpy(out.v[out.n++], a, 24);
        if ((da < 0 && db > 0) || (da > 0 && db < 0)) {
            const double t = da / (da - db);
            if (out.n < 10) { double* c = out.v[out.n++]; for (int k = 0; k < 3; ++k) c[k] = a[k] + t * (b[k] - a[k]); c[axis] = pos; }
        }
    }
}

// references of triangle `prim`: one if its box is no longer than `limit` on any axis, else the cells of a recursive midpoint split (at most `budget` more)
void presplit_triangle(const float* tv, int32_t prim, double limit, int64_t& budget, std::vector<Ref>& refs)
{
    struct Item { Poly p; double mn[3], mx[3]; int depth; };
    auto box_of = [](Item& it) {
        for (int k = 0; k < 3; ++k) { it.mn[k] = std::numeric_limits<double>::infinity(); it.mx[k] = -it.mn[k]; }
        for (int i = 0; i < it.p.n; ++i) for (int k = 0; k < 3; ++k) { it.mn[k] = std::min(it.mn[k], it.p.v[i][k]); it.mx[k] = std::max(it.mx[k], it.p.v[i][k]); }
    };
    std::vector<Item> work(1);
    work[0].p.n = 3; work[0].depth = 0;
    for (int i = 0; i < 3; ++i) for (int k = 0; k < 3; ++k) work[0].p.v[i][k] = tv[3 * i + k];
    box_of(work[0]);
    while (!work.empty()) {
        Item it = work.back(); work.pop_back();
        int axis = 0;
        for (int k = 1; k < 3; ++k) if (it.mx[k] - it.mn[k] > it.mx[axis] - it.mn[axis]) axis = k;
        if (!(it.mx[axis] - it.mn[axis] > limit) || it.depth >= 16 || budget <= 0) {
            Ref r; r.prim = prim;
            for (int k = 0; k < 3; ++k) { r.mn[k] = round_down(it.mn[k]); r.mx[k] = round_up(it.mx[k]); }
            refs.push_back(r);
            continue;
        }
        const double pos = 0.5 * (it.mn[axis] + it.mx[axis]);
        Item lo, hi; lo.depth = hi.depth = it.depth + 1;
        clip(it.p, axis, pos, 1.0, lo.p); clip(it.p, axis, pos, -1.0, hi.p);
        if (lo.p.n == 0 || hi.p.n == 0) {      // cannot happen for pos strictly inside the box; keep the piece whole rather than lose it
            Ref r; r.prim = prim;
            for (int k = 0; k < 3; ++k) { r.mn[k] = round_down(it.mn[k]); r.mx[k] = round_up(it.mx[k]); }
            refs.push_back(r);
            continue;
        }
        box_of(lo); box_of(hi);
        --budget;
        work.push_back(hi); work.push_back(lo);
    }
}

int tree_depth(const std::vector<BuildNode>& nd)
{
    std::vector<std::pair<int32_t, int>> st{{0, 1}}; int md = 0;
    while (!st.empty()) {
        const std::pair<int32_t, int> t = st.back(); st.pop_back(); md = std::max(md, t.second);
        const BuildNode& x = nd[t.first];
        if (x.left >= 0) { st.push_back({x.left, t.second + 1}); st.push_back({x.right, t.second + 1}); }
    }
    return md;
}

// ---- insertion-based optimisation of a built tree (crt_bvh_params.optimize; Bittner, Hapala & Havran 2013, restated) -------------------------------
// Repeatedly: take the inner nodes that look worst (large, with children much smaller than themselves), detach the two children of each, close the gap
// (the node's sibling takes its parent's place), and put each child back at the position of the whole tree where it adds the least surface area, found by a
// best-first search bounded by the best total so far.  Leaves keep their ranges, the node count stays, the root stays node 0.
struct TreeOpt {
    struct Cand { double induced; int32_t node; bool operator<(const Cand& o) const { return induced > o.induced; } };      // min-heap on the induced cost
    std::vector<BuildNode>& nd;
    std::vector<int32_t> parent;
    std::vector<Cand> heap_;
    explicit TreeOpt(std::vector<BuildNode>& n) : nd(n), parent(n.size(), -1)
    {
        for (size_t i = 0; i < nd.size(); ++i) if (nd[i].left >= 0) { parent[nd[i].left] = (int32_t)i; parent[nd[i].right] = (int32_t)i; }
    }
    static double area(const BuildNode& x)
    {
        const double dx = (double)x.bmax[0] - x.bmin[0], dy = (double)x.bmax[1] - x.bmin[1], dz = (double)x.bmax[2] - x.bmin[2];
        return dx * dy + dy * dz + dz * dx;
    }
    static double union_area(const BuildNode& x, const BuildNode& y)
    {
        double d[3];
        for (int k = 0; k < 3; ++k) d[k] = (double)std::max(x.bmax[k], y.bmax[k]) - (double)std::min(x.bmin[k], y.bmin[k]);
        return d[0] * d[1] + d[1] * d[2] + d[2] * d[0];
    }
    void refit(int32_t i)
    {
        const BuildNode& l = nd[nd[i].left]; const BuildNode& r = nd[nd[i].right];
        for (int k = 0; k < 3; ++k) { nd[i].bmin[k] = std::min(l.bmin[k], r.bmin[k]); nd[i].bmax[k] = std::max(l.bmax[k], r.bmax[k]); }
    }
    void refit_up(int32_t i) { for (; i >= 0; i = parent[i]) refit(i); }
    // total inner-node area (the part of the SAH cost the optimisation can change)
    double inner_area() const { double a = 0; for (const BuildNode& x : nd) if (x.left >= 0) a += area(x); return a; }

    // where to hang the detached subtree `sub`: the node X minimising area(X u sub) + the growth of X's ancestors
    int32_t best_position(int32_t sub)
    {
        const double a_sub = area(nd[sub]);
        std::vector<Cand>& heap = heap_; heap.clear();
        heap.push_back({0.0, 0});
        double best = std::numeric_limits<double>::infinity(); int32_t best_node = nd[0].left;      // (never the root itself: the root stays node 0)
        while (!heap.empty()) {
            std::pop_heap(heap.begin(), heap.end()); const Cand c = heap.back(); heap.pop_back();
            if (c.induced + a_sub >= best) break;                     // nothing below can beat the best: its cost is at least induced + area(sub)
            const double direct = union_area(nd[c.node], nd[sub]);
            if (c.node != 0 && c.induced + direct < best) { best = c.induced + direct; best_node = c.node; }
            if (nd[c.node].left >= 0) {
                const double ind = c.induced + direct - area(nd[c.node]);      // what node c grows by if `sub` goes somewhere below it
                if (ind + a_sub < best) {
                    heap.push_back({ind, nd[c.node].left}); std::push_heap(heap.begin(), heap.end());
                    heap.push_back({ind, nd[c.node].right}); std::push_heap(heap.begin(), heap.end());
                }
            }
        }
        return best_node;
    }
    // hangs `sub` beside x under the free node `link`, which takes x's place
    void insert(int32_t sub, int32_t x, int32_t link)
    {
        const int32_t px = parent[x];
        nd[link].left = x; nd[link].right = sub; nd[link].first = 0; nd[link].count = 0;
        parent[x] = link; parent[sub] = link; parent[link] = px;
        if (nd[px].left == x) nd[px].left = link; else nd[px].right = link;
        refit_up(link);
    }
    // one node: detach its children, close the gap, reinsert both.  Needs a grandparent (root 0 and its children stay).
    bool reinsert_children(int32_t n)
    {
        if (nd[n].left < 0) return false;
        const int32_t p = parent[n]; if (p <= 0) return false;          // n is the root or a child of the root
        const int32_t g = parent[p];
        const int32_t sib = nd[p].left == n ? nd[p].right : nd[p].left;
        int32_t l = nd[n].left, r = nd[n].right;
        if (nd[g].left == p) nd[g].left = sib; else nd[g].right = sib;
        parent[sib] = g; refit_up(g);
        parent[l] = parent[r] = -1;
        if (area(nd[l]) < area(nd[r])) std::swap(l, r);                   // the larger subtree first
        insert(l, best_position(l), p);
        insert(r, best_position(r), n);
        return true;
    }
};

}  // namespace

// Insertion-based optimisation of b->nodes (TreeOpt above; crt_bvh_params.optimize iterations; boxes unpadded or padded alike).  Returns the tree's depth
// afterwards (built_depth when nothing was done).  Used by the host builder and by builder 2 (device clustering + host layout).
int crt_bvh_optimize_tree(crt_bvh* b, const crt_bvh_params& pr, int built_depth)
{
    b->opt_iters = 0;
    if (pr.optimize > 0 && b->nodes.size() >= 16) {
        // insertion-based optimisation (TreeOpt above): per iteration the worst-looking 2 % of the inner nodes (at most 20,000), ranked by area x
        // (area / smaller child) x (area / mean child); four consecutive windows of that ranking take turns, so that nodes which are already placed
        // as well as the search can place them are not picked over and over
        TreeOpt T(b->nodes);
        std::vector<std::pair<double, int32_t>> rank;
        const auto worse = [](const std::pair<double, int32_t>& a, const std::pair<double, int32_t>& c) { return a.first > c.first || (a.first == c.first && a.second < c.second); };
        std::vector<double> total{T.inner_area()};        // summed inner-node area after each iteration
        for (int it = 0; it < pr.optimize; ++it) {
            // no progress worth the time (a terrain grid, say, is as good as it gets after the build): less than 0.2 % over the last four iterations
            if (it >= 4 && total[it - 4] - total[it] < 0.002 * total[it]) break;
            if (it == 1 && total[0] - total[1] < 0.0005 * total[1]) break;      // the most promising 2 % gained next to nothing
            rank.clear();
            for (size_t i = 1; i < b->nodes.size(); ++i) {
                const BuildNode& x = b->nodes[i];
                if (x.left < 0 || T.parent[i] <= 0) continue;
                const double a = TreeOpt::area(x), al = TreeOpt::area(b->nodes[x.left]), ar = TreeOpt::area(b->nodes[x.right]);
                const double mn = std::max(std::min(al, ar), 1e-300), sum = std::max(al + ar, 1e-300);
                rank.emplace_back(a * (a / mn) * (2.0 * a / sum), (int32_t)i);
            }
            if (rank.empty()) break;
            const size_t batch = std::min<size_t>(rank.size(), std::max<size_t>(64, std::min<size_t>(rank.size() / 50, 20000)));
            const size_t off = std::min(rank.size() - batch, (size_t)(it % 4) * batch);
            std::nth_element(rank.begin(), rank.begin() + off, rank.end(), worse);
            std::nth_element(rank.begin() + off, rank.begin() + off + batch - 1, rank.end(), worse);
            std::sort(rank.begin() + off, rank.begin() + off + batch, worse);      // a fixed processing order for a given tree
            // (putting two children back one after the other is not guaranteed to pay: an iteration that loses is undone; so is one that makes the tree
            // deeper than the traversal stack allows -- many identical boxes can be chained into a list -- and the optimisation ends there)
            const std::vector<BuildNode> before_nodes = b->nodes; const std::vector<int32_t> before_parent = T.parent;
            for (size_t k = off; k < off + batch; ++k) T.reinsert_children(rank[k].second);
            total.push_back(T.inner_area());
            const bool too_deep = tree_depth(b->nodes) > std::max(56, built_depth);
            if (too_deep || total.back() > total[total.size() - 2]) { b->nodes = before_nodes; T.parent = before_parent; total.back() = total[total.size() - 2]; }
            if (too_deep) break;
            if (total.back() < total[total.size() - 2]) ++b->opt_iters;
        }
        return tree_depth(b->nodes);
    }
    return built_depth;
}

// Builds the host tree.  Returns false on failure.
bool crt_bvh_build_host(crt_bvh* b, const float* verts, int64_t n, const crt_bvh_params& pr, bool presplit_single)
{
    auto t0 = std::chrono::steady_clock::now();
    b->n_tris = n; b->max_leaf = pr.max_leaf;
    b->verts.assign(verts, verts + 9 * n);
    // references: one per triangle, several for a triangle much longer than the scene's detail (pre-splitting; not with one triangle per leaf,
    // where the 8-wide layout shares the triangle order and wants every triangle exactly once)
    std::vector<Ref> refs; refs.reserve((size_t)n);
    float maxabs = 0.f;
    Box root; root.reset();
    for (int64_t i = 0; i < n; ++i) {
        const float* tv = verts + 9 * i;
        Ref r; r.prim = (int32_t)i;
        for (int k = 0; k < 3; ++k) {
            r.mn[k] = std::min(tv[k], std::min(tv[3 + k], tv[6 + k])); r.mx[k] = std::max(tv[k], std::max(tv[3 + k], tv[6 + k]));
            maxabs = std::max(maxabs, std::max(std::fabs(r.mn[k]), std::fabs(r.mx[k])));
        }
        root.grow(r.mn, r.mx);
        refs.push_back(r);
    }
    for (int k = 0; k < 3; ++k) { b->bounds[k] = n ? root.mn[k] : 0.f; b->bounds[3 + k] = n ? root.mx[k] : 0.f; }
    if (pr.presplit > 0.f && (pr.max_leaf > 1 || presplit_single) && n > 0) {
        double diag = 0; for (int k = 0; k < 3; ++k) diag += ((double)root.mx[k] - root.mn[k]) * ((double)root.mx[k] - root.mn[k]);
        const double limit = (double)pr.presplit * std::sqrt(diag);
        int64_t budget = std::max<int64_t>(n / 4, 4096);         // at most this many additional references in all
        if (n + budget >= ((int64_t)1 << 28)) budget = std::max<int64_t>(0, ((int64_t)1 << 28) - 1 - n);
        std::vector<Ref> out; out.reserve((size_t)n + 1024);
        for (int64_t i = 0; i < n; ++i) {
            const Ref& r = refs[i];
            if (limit > 0 && std::max(r.mx[0] - r.mn[0], std::max(r.mx[1] - r.mn[1], r.mx[2] - r.mn[2])) > limit && budget > 0) presplit_triangle(verts + 9 * i, (int32_t)i, limit, budget, out);
            else out.push_back(r);
        }
        refs.swap(out);
    }
    const int64_t nr = (int64_t)refs.size();
    b->n_refs = nr;
    b->prim.resize((size_t)nr);
    b->nodes.assign((size_t)std::max<int64_t>(2 * nr, 1), BuildNode());
    Builder B(b->prim, b->nodes);
    B.verts = b->verts.data(); B.n = nr; B.max_leaf = pr.max_leaf; B.bins = std::min(kMaxBins, std::max(4, pr.sah_bins));
    B.ct = pr.cost_traversal; B.ci = pr.cost_intersect;
    B.tmn.resize(3 * (size_t)nr); B.tmx.resize(3 * (size_t)nr); B.cen.resize(3 * (size_t)nr);
    for (int64_t i = 0; i < nr; ++i) {
        b->prim[i] = (int32_t)i;      // reference ids while building; the caller's triangle ids afterwards
        for (int k = 0; k < 3; ++k) { B.tmn[3 * i + k] = refs[i].mn[k]; B.tmx[3 * i + k] = refs[i].mx[k]; B.cen[3 * i + k] = 0.5f * refs[i].mn[k] + 0.5f * refs[i].mx[k]; }
    }
    if (n > 0) {
        int nt = pr.n_threads > 0 ? pr.n_threads : (int)std::max(1u, std::thread::hardware_concurrency());
        nt = std::min(nt, 64);
        B.n_nodes = 1;
        if (nt > 1 && nr > 65536) {
            Pool pool(nt);
            B.pool = &pool;
            pool.submit([&] { B.subtree(0, 0, nr, 1); });
            pool.wait();
        } else {
            B.pool = nullptr;
            B.subtree(0, 0, nr, 1);
        }
        b->nodes.resize((size_t)B.n_nodes.load());
        for (int64_t i = 0; i < nr; ++i) b->prim[i] = refs[b->prim[i]].prim;
        b->depth = crt_bvh_optimize_tree(b, pr, B.max_depth.load());
        // SAH cost (relative to the root area) before padding
        double ra = root.half_area(), cost = 0;
        for (const BuildNode& nd : b->nodes) {
            Box x; std::memcpy(x.mn, nd.bmin, 12); std::memcpy(x.mx, nd.bmax, 12);
            cost += x.half_area() * (nd.left >= 0 ? (double)pr.cost_traversal : (double)pr.cost_intersect * nd.count);
        }
        b->sah = ra > 0 ? cost / ra : 0;
        // Conservative padding (D:R10): the triangle test in fp32 may accept a hit a few ulps of the scene's
        // coordinate range outside the triangle's exact box; boxes grow by 2^-17 of the largest |coordinate|.
        float pad = maxabs * (1.0f / 131072.0f);
        for (BuildNode& nd : b->nodes)
            for (int k = 0; k < 3; ++k) { nd.bmin[k] -= pad; nd.bmax[k] += pad; }
    } else {
        b->nodes.clear(); b->depth = 0; b->sah = 0;
    }
    b->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return true;
}

int32_t crt_bvh_check_host(const crt_bvh* b)
{
    int32_t bad = 0;
    if (b->n_tris == 0) return 0;
    std::vector<uint8_t> seen((size_t)b->n_tris, 0);
    // pre-split trees (n_refs > n_tris): a triangle may sit in several leaves, each holding the part of it inside that leaf's box; for those triangles
    // the invariant is that the leaves' boxes together cover the triangle (checked below on a lattice of points of the triangle)
    const bool split = b->n_refs > b->n_tris;
    std::vector<int32_t> n_leaves; std::vector<std::pair<int32_t, int32_t>> leaf_of;      // (triangle, node) of every reference of a multiply referenced triangle
    if (split) {
        n_leaves.assign((size_t)b->n_tris, 0);
        for (int32_t p : b->prim) if (p >= 0 && p < b->n_tris) ++n_leaves[p];
    }
    for (const BuildNode& nd : b->nodes) {
        if (nd.left >= 0) {
            for (int32_t c : {nd.left, nd.right}) {
                const BuildNode& ch = b->nodes[c];
                for (int k = 0; k < 3; ++k) if (ch.bmin[k] < nd.bmin[k] || ch.bmax[k] > nd.bmax[k]) bad |= 1;
            }
        } else {
            if (nd.count < 1 || nd.count > b->max_leaf) bad |= 2;
            for (int j = 0; j < nd.count; ++j) {
                int32_t p = b->prim[nd.first + j];
                if (p < 0 || p >= b->n_tris) { bad |= 32; continue; }
                if (seen[p] && !split) bad |= 4;
                seen[p] = 1;
                if (split && n_leaves[p] > 1) { leaf_of.emplace_back(p, (int32_t)(&nd - b->nodes.data())); continue; }
                const float* tv = b->verts.data() + 9 * (int64_t)p;
                for (int v = 0; v < 3; ++v) for (int k = 0; k < 3; ++k)
                    if (tv[3 * v + k] < nd.bmin[k] || tv[3 * v + k] > nd.bmax[k]) bad |= 8;
            }
        }
    }
    for (uint8_t s : seen) if (!s) bad |= 16;
    if (split) {
        std::sort(leaf_of.begin(), leaf_of.end());
        for (size_t i = 0; i < leaf_of.size();) {
            size_t j = i; while (j < leaf_of.size() && leaf_of[j].first == leaf_of[i].first) ++j;
            const float* tv = b->verts.data() + 9 * (int64_t)leaf_of[i].first;
            const int G = 12;         // barycentric lattice: 91 points including the corners and edge points
            for (int a = 0; a <= G; ++a) for (int c = 0; a + c <= G; ++c) {
                const double wa = (double)a / G, wc = (double)c / G, wb = 1.0 - wa - wc;
                double q[3]; for (int k = 0; k < 3; ++k) q[k] = wb * tv[k] + wa * tv[3 + k] + wc * tv[6 + k];
                bool in = false;
                for (size_t m = i; m < j && !in; ++m) {
                    const BuildNode& nd = b->nodes[leaf_of[m].second];
                    in = q[0] >= nd.bmin[0] && q[0] <= nd.bmax[0] && q[1] >= nd.bmin[1] && q[1] <= nd.bmax[1] && q[2] >= nd.bmin[2] && q[2] <= nd.bmax[2];
                }
                if (!in) bad |= 8;
            }
            i = j;
        }
    }
    return bad;
}

// Flattens the host tree into the binary traversal layout (host vectors; the caller uploads them).
// tri_order: caller's triangle id stored at position j of the device triangle array; empty = the tree's own leaf order.
// A non-empty order (the wide layout's) requires one triangle per leaf, so that every leaf is still one contiguous range.
void crt_bvh_flatten(const crt_bvh* b, const std::vector<int32_t>& tri_order, std::vector<GpuNode>& gn, std::vector<GpuTri>& gt, std::vector<int32_t>& slot_of_prim)
{
    const float inf = std::numeric_limits<float>::infinity();
    const int64_t n = b->n_refs;         // records of the device triangle array: one per reference (== triangles unless the build pre-split some)
    const bool own = tri_order.empty();
    gt.resize((size_t)n); slot_of_prim.assign((size_t)b->n_tris, -1);      // slot_of_prim: any one of a triangle's records (they are identical)
    for (int64_t j = 0; j < n; ++j) {
        int32_t p = own ? b->prim[j] : tri_order[j];
        const float* tv = b->verts.data() + 9 * (int64_t)p;
        GpuTri t;
        t.v0p = make_float4(tv[0], tv[1], tv[2], 0.f);
        std::memcpy(&t.v0p.w, &p, 4);
        t.e1 = make_float4(tv[3] - tv[0], tv[4] - tv[1], tv[5] - tv[2], 0.f);
        t.e2 = make_float4(tv[6] - tv[0], tv[7] - tv[1], tv[8] - tv[2], 0.f);
        t.pad = make_float4(0.f, 0.f, 0.f, 0.f);
        gt[j] = t; slot_of_prim[p] = (int32_t)j;
    }
    auto leaf_ref = [&](const BuildNode& nd) {
        const int32_t first = own ? nd.first : slot_of_prim[b->prim[nd.first]];
        return ~((first << 3) | (nd.count - 1));
    };
    // a box at +infinity on every axis: the slab test fails for every ray (an inverted box would NOT fail, because the
    // test takes min/max of the two plane distances)
    auto empty_child = [&] { GpuChild c; c.min_x = c.max_x = c.min_y = c.max_y = c.min_z = c.max_z = inf; c.ref = ~0; c.pad = 0; return c; };
    auto child_of = [&](const BuildNode& nd, int32_t ref) {
        GpuChild c; c.min_x = nd.bmin[0]; c.max_x = nd.bmax[0]; c.min_y = nd.bmin[1]; c.max_y = nd.bmax[1]; c.min_z = nd.bmin[2]; c.max_z = nd.bmax[2];
        c.ref = ref; c.pad = 0; return c;
    };
    gn.clear();
    if (n == 0) { GpuNode g; g.c[0] = g.c[1] = empty_child(); gn.push_back(g); return; }
    if (b->nodes[0].left < 0) {      // the whole scene is one leaf: a root whose second child is empty
        GpuNode g; g.c[0] = child_of(b->nodes[0], leaf_ref(b->nodes[0])); g.c[1] = empty_child(); gn.push_back(g); return;
    }
    // numbering of inner nodes: the top of the tree breadth-first (the first 512 indices are the top levels, which every ray visits: they
    // share cache lines, and an experiment stages them in shared memory), then depth-first, left child next to its parent
    std::vector<int32_t> gpu_index(b->nodes.size(), -1), stack, order;
    {
        std::deque<int32_t> frontier{0};
        while (!frontier.empty() && order.size() + frontier.size() < 512) {
            int32_t i = frontier.front(); frontier.pop_front();
            gpu_index[i] = (int32_t)order.size(); order.push_back(i);
            const BuildNode& nd = b->nodes[i];
            if (b->nodes[nd.left].left >= 0) frontier.push_back(nd.left);
            if (b->nodes[nd.right].left >= 0) frontier.push_back(nd.right);
        }
        for (auto it = frontier.rbegin(); it != frontier.rend(); ++it) stack.push_back(*it);      // the rest depth-first, in breadth-first order of their roots
    }
    while (!stack.empty()) {
        int32_t i = stack.back(); stack.pop_back();
        gpu_index[i] = (int32_t)order.size(); order.push_back(i);
        const BuildNode& nd = b->nodes[i];
        if (b->nodes[nd.right].left >= 0) stack.push_back(nd.right);
        if (b->nodes[nd.left].left >= 0) stack.push_back(nd.left);
    }
    gn.resize(order.size());
    for (size_t k = 0; k < order.size(); ++k) {
        const BuildNode& nd = b->nodes[order[k]];
        const BuildNode& l = b->nodes[nd.left]; const BuildNode& r = b->nodes[nd.right];
        GpuNode g;
        g.c[0] = child_of(l, l.left >= 0 ? gpu_index[nd.left] : leaf_ref(l));
        g.c[1] = child_of(r, r.left >= 0 ? gpu_index[nd.right] : leaf_ref(r));
        gn[k] = g;
    }
}

// grid of the 16-bit layout over the (padded) scene box [lo, hi]
void crt_qgrid_for_box(const double lo[3], const double hi[3], QGrid* grid)
{
    double maxext = 0;
    for (int k = 0; k < 3; ++k) maxext = std::max(maxext, hi[k] - lo[k]);
    if (!(maxext > 0)) maxext = 1;
    for (int k = 0; k < 3; ++k) {
        // margin on either side: 8 grid steps, or 4 ulps of the box's coordinates when the scene sits far from the origin (gmin is a
        // float: its rounding must not eat the margin, or planes clamp inward); gmin is rounded DOWN so the low side only gains
        const double e = std::max(hi[k] - lo[k], maxext * (1.0 / 4096.0));
        const double ulp = std::max(std::fabs(lo[k]), std::fabs(hi[k])) * (1.0 / 8388608.0);
        const double margin = std::max(8.0 * e / (65535.0 - 16.0), 4.0 * ulp);
        const float scale = (float)(65535.0 / (e + 2.0 * margin) * (1.0 - 1e-6));
        grid->scale[k] = scale;
        grid->gmin[k] = std::nextafterf((float)(lo[k] - margin), -std::numeric_limits<float>::infinity());
        grid->inv_scale[k] = (float)(1.0 / (double)scale);
    }
}

// 16-bit layout of the flattened nodes (trace_kernel 3): every box plane becomes a position on a 65536-step grid over the
// scene box, rounded OUTWARD (min planes down, max planes up) and then moved ONE more step outward: the traversal kernel
// evaluates a plane distance as one FMA in grid units whose rounding error stays below one step of position for ray
// origins within 16 scene extents (trace.cu: QRay), so the box test stays conservative (D:R10: it never decides the result, only which subtrees are
// visited).  Returns 0, or 1 if a plane had to be clamped / is less than one step outside its box.
int32_t crt_bvh_quantise(const crt_bvh* b, const std::vector<GpuNode>& gn, std::vector<QNode>& qn, QGrid* grid, double* inflation)
{
    (void)b;
    double area_f = 0, area_q = 0;       // summed half-areas of the fp32 boxes and of the boxes the 16-bit planes decode to
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    auto planes = [](const GpuChild& c, int k, double& mn, double& mx) {
        const float* p = &c.min_x; mn = p[2 * k]; mx = p[2 * k + 1];
    };
    if (!gn.empty())
        for (int c = 0; c < 2; ++c)
            for (int k = 0; k < 3; ++k) {
                double mn, mx; planes(gn[0].c[c], k, mn, mx);
                if (std::isfinite(mn) && std::isfinite(mx)) { lo[k] = std::min(lo[k], mn); hi[k] = std::max(hi[k], mx); }
            }
    for (int k = 0; k < 3; ++k) if (lo[k] > hi[k]) { lo[k] = 0; hi[k] = 1; }
    crt_qgrid_for_box(lo, hi, grid);
    int32_t bad = 0;
    qn.resize(gn.size());
    for (size_t i = 0; i < gn.size(); ++i) {
        QNode q;
        for (int c = 0; c < 2; ++c) {
            q.ref[c] = gn[i].c[c].ref;
            for (int k = 0; k < 3; ++k) {
                double mn, mx; planes(gn[i].c[c], k, mn, mx);
                uint32_t qlo = 65535u, qhi = 0u;           // empty child: inverted on every axis, fails for every ray
                if (std::isfinite(mn) && std::isfinite(mx)) {
                    const double g = (double)grid->gmin[k], s = (double)grid->scale[k];
                    double a = std::floor((mn - g) * s), z = std::ceil((mx - g) * s);
                    if (g + a / s > mn) a -= 1.0;          // the products above are rounded: re-check in the direction that matters
                    if (g + z / s < mx) z += 1.0;
                    a -= 1.0; z += 1.0;
                    if (a < 0.0) { a = 0.0; bad |= 1; }
                    if (z > 65535.0) { z = 65535.0; bad |= 1; }
                    if (!(g + (a + 1.0) / s <= mn) || !(g + (z - 1.0) / s >= mx)) bad |= 1;
                    qlo = (uint32_t)a; qhi = (uint32_t)z;
                }
                q.planes[3 * c + k] = qlo | (qhi << 16);
            }
            double ef[3], eq[3]; bool finite = true;
            for (int k = 0; k < 3; ++k) {
                double mn, mx; planes(gn[i].c[c], k, mn, mx);
                if (!std::isfinite(mn) || !std::isfinite(mx)) { finite = false; break; }
                ef[k] = mx - mn; eq[k] = (double)((q.planes[3 * c + k] >> 16) - (q.planes[3 * c + k] & 0xffffu)) / (double)grid->scale[k];
            }
            if (finite) { area_f += ef[0] * ef[1] + ef[1] * ef[2] + ef[2] * ef[0]; area_q += eq[0] * eq[1] + eq[1] * eq[2] + eq[2] * eq[0]; }
        }
        qn[i] = q;
    }
    if (inflation) *inflation = area_f > 0 ? area_q / area_f : 1.0;
    return bad;
}

// 4-wide form of the 16-bit layout (trace_kernel 7): node j = TWO consecutive 32-byte records, 2j holding the boxes and references of the children of
// binary node i's first child, 2j + 1 those of its second child, i.e. the four GRANDCHILDREN of i; a child of i that is a leaf stands for itself
// (its own planes, second slot empty: planes inverted, never hit).  The planes are copied from the binary 16-bit nodes, so the layout inherits their
// outward rounding; inner references are renumbered to 4-wide nodes (breadth-first from the root).  One visit = two independent 256-bit loads and four
// box tests: the same bytes and about 17 % fewer box tests per ray than two binary levels, and half as many DEPENDENT fetches (the kernel is bound by
// their latency, profiles/r02a).
void crt_bvh_collapse4(const std::vector<GpuNode>& gn, const std::vector<QNode>& qn, std::vector<QNode>& q4)
{
    q4.clear();
    if (gn.empty()) return;
    const uint32_t EMPTY_PLANES = 65535u;            // lo = 65535, hi = 0
    std::vector<int32_t> map4(gn.size(), -1), order;
    map4[0] = 0; order.push_back(0);
    for (size_t h = 0; h < order.size(); ++h) {       // breadth-first over the binary nodes that head a 4-wide node
        const int32_t i = order[h];
        for (int c = 0; c < 2; ++c) {
            const int32_t cr = gn[i].c[c].ref;
            if (cr < 0 || !std::isfinite(gn[i].c[c].min_x)) continue;          // leaf or empty child: stands for itself
            for (int g = 0; g < 2; ++g) {
                const int32_t gr = gn[cr].c[g].ref;
                if (gr >= 0 && std::isfinite(gn[cr].c[g].min_x) && map4[gr] < 0) { map4[gr] = (int32_t)order.size(); order.push_back(gr); }
            }
        }
    }
    q4.resize(2 * order.size());
    for (size_t h = 0; h < order.size(); ++h) {
        const int32_t i = order[h];
        for (int c = 0; c < 2; ++c) {
            QNode rec;
            const int32_t cr = gn[i].c[c].ref;
            const bool empty = !std::isfinite(gn[i].c[c].min_x);
            if (!empty && cr >= 0) {
                rec = qn[cr];
                for (int g = 0; g < 2; ++g) if (rec.ref[g] >= 0 && std::isfinite(gn[cr].c[g].min_x)) rec.ref[g] = map4[rec.ref[g]];
            } else {
                for (int k = 0; k < 3; ++k) { rec.planes[k] = empty ? EMPTY_PLANES : qn[i].planes[3 * c + k]; rec.planes[3 + k] = EMPTY_PLANES; }
                rec.ref[0] = empty ? ~0 : cr; rec.ref[1] = ~0;
            }
            q4[2 * h + c] = rec;
        }
    }
}

// Invariants of the DEVICE traversal layouts themselves (whichever builder wrote them): downloads the fp32 nodes, the 16-bit nodes, the
// triangle records and slot_of_prim and walks the tree from node 0.  Bits as crt_bvh_check_host (1 child box not inside its parent's,
// 2 leaf size, 4 triangle in two leaves, 8 triangle outside its leaf's box, 16 triangle in no leaf, 32 bad index / record) and 0x10000
// (a 16-bit plane less than one grid step outside the fp32 box it stands for, or different child references).
int32_t crt_layout_check_device(const crt_bvh* b)
{
    if (b->n_tris == 0 || !b->d_nodes || !b->d_tris) return 0;
    const int64_t nn = b->n_gpu_nodes, nt = b->n_tris, nrec = b->n_refs;
    const bool split = nrec > nt;        // pre-split build: a triangle may have several records; the coverage of such triangles is crt_bvh_check_host's
    std::vector<GpuNode> gn((size_t)nn); std::vector<QNode> qn((size_t)nn); std::vector<GpuTri> gt((size_t)nrec); std::vector<int32_t> sop((size_t)nt);
    if (cudaMemcpy(gn.data(), b->d_nodes, gn.size() * sizeof(GpuNode), cudaMemcpyDeviceToHost) != cudaSuccess) return 32;
    if (b->d_qnodes && cudaMemcpy(qn.data(), b->d_qnodes, qn.size() * sizeof(QNode), cudaMemcpyDeviceToHost) != cudaSuccess) return 32;
    if (cudaMemcpy(gt.data(), b->d_tris, gt.size() * sizeof(GpuTri), cudaMemcpyDeviceToHost) != cudaSuccess) return 32;
    if (cudaMemcpy(sop.data(), b->d_slot_of_prim, sop.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return 32;
    int32_t bad = 0;
    std::vector<uint8_t> seen_node((size_t)nn, 0), seen_tri((size_t)nt, 0);
    auto inside = [](const GpuChild& in, const GpuChild& out) {
        return in.min_x >= out.min_x && in.max_x <= out.max_x && in.min_y >= out.min_y && in.max_y <= out.max_y && in.min_z >= out.min_z && in.max_z <= out.max_z;
    };
    std::vector<int32_t> stack{0};
    seen_node[0] = 1;
    while (!stack.empty()) {
        const int32_t i = stack.back(); stack.pop_back();
        for (int c = 0; c < 2; ++c) {
            const GpuChild& ch = gn[i].c[c];
            if (!std::isfinite(ch.min_x)) continue;                     // the empty second child of a one-leaf scene
            if (b->d_qnodes) {
                if (qn[i].ref[c] != ch.ref) bad |= 0x10000;
                const float* pl = &ch.min_x;
                for (int k = 0; k < 3; ++k) {
                    const double g = b->qgrid.gmin[k], s = b->qgrid.scale[k];
                    const uint32_t w = qn[i].planes[3 * c + k];
                    const double a = (double)(w & 0xffffu), z = (double)(w >> 16);
                    if (!(g + (a + 1.0) / s <= (double)pl[2 * k]) || !(g + (z - 1.0) / s >= (double)pl[2 * k + 1])) bad |= 0x10000;
                }
            }
            if (ch.ref >= 0) {
                if (ch.ref >= nn) { bad |= 32; continue; }
                if (seen_node[ch.ref]) { bad |= 4; continue; }
                seen_node[ch.ref] = 1;
                for (int g2 = 0; g2 < 2; ++g2) if (std::isfinite(gn[ch.ref].c[g2].min_x) && !inside(gn[ch.ref].c[g2], ch)) bad |= 1;
                stack.push_back(ch.ref);
            } else {
                const int32_t leaf = ~ch.ref; const int64_t first = leaf >> 3; const int cnt = (leaf & 7) + 1;
                if (cnt > b->max_leaf) bad |= 2;
                if (first + cnt > nrec) { bad |= 32; continue; }
                for (int64_t j = first; j < first + cnt; ++j) {
                    int32_t prim; std::memcpy(&prim, &gt[j].v0p.w, 4);
                    if (prim < 0 || prim >= nt) { bad |= 32; continue; }
                    if (seen_tri[prim] && !split) bad |= 4;
                    seen_tri[prim] = 1;
                    if (split) { int32_t q = -1; if (sop[prim] >= 0 && sop[prim] < nrec) std::memcpy(&q, &gt[sop[prim]].v0p.w, 4); if (q != prim) bad |= 32; }
                    else if (sop[prim] != (int32_t)j) bad |= 32;
                    const float* tv = b->verts.data() + 9 * (int64_t)prim;
                    if (gt[j].v0p.x != tv[0] || gt[j].v0p.y != tv[1] || gt[j].v0p.z != tv[2] || gt[j].e1.x != tv[3] - tv[0] || gt[j].e2.z != tv[8] - tv[2]) bad |= 32;
                    for (int v = 0; v < 3 && !split; ++v)
                        if (tv[3 * v] < ch.min_x || tv[3 * v] > ch.max_x || tv[3 * v + 1] < ch.min_y || tv[3 * v + 1] > ch.max_y || tv[3 * v + 2] < ch.min_z || tv[3 * v + 2] > ch.max_z) bad |= 8;
                }
            }
        }
    }
    for (uint8_t s2 : seen_tri) if (!s2) bad |= 16;
    for (uint8_t s2 : seen_node) if (!s2) bad |= 32;
    return bad;
}
