// a0 (part): collapses the binary SAH tree (max_leaf = 1) into the 8-wide compressed layout that the alternative traversal
// kernel (trace_kernel = 2, trace_wide.cu) reads.  The paper leaves the acceleration structure open (D:R11); the result
// of crt_trace does not depend on it (D:R10), so this layout is purely a B200 design choice: the traversal kernel is bound
// by the L1 data pipe (profiles/r01a), and a 128-byte node that holds eight child boxes is one dependent fetch where the
// binary layout needs several.  Measured result: profiles/r01b.
//
// WNode (128 bytes, four 32-byte sectors, each fetched by one 256-bit load):
//   sector 0: p.xyz (box origin), E.x (fp32 power of two), E.y | E.z (bf16 halves), child_base, tri_base, imask | lmask << 8
//   sectors 1-3: per axis 16 bytes of LO planes then 16 bytes of HI planes; each 32-bit word = two children (2k in the low
//   half, 2k+1 in the high half), a plane being the bf16 bit pattern of r = (x - p) / E in [0, 1].
// Conservative rounding: LO planes round down, HI planes round up; the kernel reads the high-half entry WITHOUT masking the
// low half (it only enlarges the value by less than one bf16 ulp), so LO planes stored in a high half are lowered one more ulp.
// Child j of a node is an inner node (bit j of imask), a single triangle (bit j of lmask) or empty.  Inner children are
// contiguous from child_base in slot order, triangles contiguous from tri_base in slot order.  Slots are assigned so that
// slot s lies towards the octant s of the node (bit 2 = +x, bit 1 = +y, bit 0 = +z): a ray visits hit children in the order
// of descending (slot XOR octinv), which approximates front-to-back order without sorting distances.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include "crt_internal.h"

namespace {

inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
inline float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

// bf16 bit pattern of the largest bf16 <= r (r >= 0)
inline uint16_t bf16_down(double r)
{
    if (!(r > 0.0)) return 0;
    float f = (float)r;
    if ((double)f > r) f = std::nextafter(f, 0.0f);
    return (uint16_t)(f2u(f) >> 16);                       // truncation of a positive float rounds down
}
// bf16 bit pattern of the smallest bf16 >= r (r >= 0)
inline uint16_t bf16_up(double r)
{
    if (!(r > 0.0)) return 0;
    float f = (float)r;
    if ((double)f < r) f = std::nextafter(f, std::numeric_limits<float>::infinity());
    uint32_t u = f2u(f);
    return (uint16_t)((u >> 16) + ((u & 0xffffu) ? 1u : 0u));
}

struct Item { int32_t bnode; double area; };

}  // namespace

// Builds the wide layout from b->nodes (binary, every leaf holding exactly one triangle).
// tri_order[j] = caller's triangle id stored at position j of the device triangle array.
void crt_bvh_build_wide(const crt_bvh* b, std::vector<WNode>& wn, std::vector<int32_t>& tri_order, int* depth_out)
{
    const std::vector<BuildNode>& bn = b->nodes;
    wn.clear(); tri_order.clear(); *depth_out = 0;
    if (b->n_tris == 0) {
        WNode w; std::memset(&w, 0, sizeof w);
        for (int a = 0; a < 3; ++a) for (int k = 0; k < 4; ++k) { w.planes[a][k] = 0x40004000u; w.planes[a][4 + k] = 0u; }
        w.ex = 1.0f; w.eyz = (f2u(1.0f) & 0xffff0000u) | (f2u(1.0f) >> 16);
        wn.push_back(w);
        return;
    }
    auto half_area = [&](int32_t i) {
        const BuildNode& n = bn[i];
        double dx = (double)n.bmax[0] - n.bmin[0], dy = (double)n.bmax[1] - n.bmin[1], dz = (double)n.bmax[2] - n.bmin[2];
        return dx * dy + dy * dz + dz * dx;
    };
    struct Pending { int32_t broot; int32_t windex; int depth; };
    std::vector<Pending> queue; queue.push_back({0, 0, 1});
    wn.resize(1);
    tri_order.reserve((size_t)b->n_tris);
    for (size_t qi = 0; qi < queue.size(); ++qi) {
        const Pending pd = queue[qi];
        *depth_out = std::max(*depth_out, pd.depth);
        // ---- greedy collapse: open the inner child of largest surface area until eight children
        Item items[8]; int n = 0;
        if (bn[pd.broot].left < 0) items[n++] = {pd.broot, 0.0};
        else { items[n++] = {bn[pd.broot].left, 0.0}; items[n++] = {bn[pd.broot].right, 0.0}; }
        for (int i = 0; i < n; ++i) items[i].area = half_area(items[i].bnode);
        while (n < 8) {
            int best = -1;
            for (int i = 0; i < n; ++i) if (bn[items[i].bnode].left >= 0 && (best < 0 || items[i].area > items[best].area)) best = i;
            if (best < 0) break;
            const BuildNode& o = bn[items[best].bnode];
            items[best] = {o.left, half_area(o.left)};
            items[n++] = {o.right, half_area(o.right)};
        }
        // ---- node box and child slots (greedy assignment maximising the octant score)
        double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
        for (int i = 0; i < n; ++i) for (int a = 0; a < 3; ++a) { mn[a] = std::min(mn[a], (double)bn[items[i].bnode].bmin[a]); mx[a] = std::max(mx[a], (double)bn[items[i].bnode].bmax[a]); }
        double score[8][8];
        for (int i = 0; i < n; ++i)
            for (int s = 0; s < 8; ++s) {
                double sc = 0;
                for (int a = 0; a < 3; ++a) {
                    const BuildNode& c = bn[items[i].bnode];
                    double d = 0.5 * ((double)c.bmin[a] + c.bmax[a]) - 0.5 * (mn[a] + mx[a]);
                    sc += ((s >> (2 - a)) & 1) ? d : -d;
                }
                score[i][s] = sc;
            }
        int slot_of[8]; bool slot_used[8] = {false, false, false, false, false, false, false, false}; bool done[8] = {false, false, false, false, false, false, false, false};
        for (int r = 0; r < n; ++r) {
            int bi = -1, bs = -1;
            for (int i = 0; i < n; ++i) if (!done[i]) for (int s = 0; s < 8; ++s) if (!slot_used[s] && (bi < 0 || score[i][s] > score[bi][bs])) { bi = i; bs = s; }
            slot_of[bi] = bs; slot_used[bs] = true; done[bi] = true;
        }
        int child_at[8]; for (int s = 0; s < 8; ++s) child_at[s] = -1;
        for (int i = 0; i < n; ++i) child_at[slot_of[i]] = i;
        // ---- encode
        WNode w; std::memset(&w, 0, sizeof w);
        double E[3];
        for (int a = 0; a < 3; ++a) {
            double ext = mx[a] - mn[a];
            int e = ext > 0 ? (int)std::ceil(std::log2(ext)) : -100;
            if (ext > 0 && std::ldexp(1.0, e) < ext) ++e;
            e = std::max(-100, std::min(100, e));
            E[a] = std::ldexp(1.0, e);
        }
        w.px = (float)mn[0]; w.py = (float)mn[1]; w.pz = (float)mn[2];        // exact: the minima are fp32 values
        w.ex = (float)E[0];
        w.eyz = (f2u((float)E[1]) & 0xffff0000u) | (f2u((float)E[2]) >> 16);  // powers of two: exact in bf16
        uint32_t imask = 0, lmask = 0;
        int n_inner = 0, n_leaf = 0;
        for (int s = 0; s < 8; ++s) if (child_at[s] >= 0) { if (bn[items[child_at[s]].bnode].left >= 0) { imask |= 1u << s; ++n_inner; } else { lmask |= 1u << s; ++n_leaf; } }
        w.child_base = (uint32_t)wn.size();
        w.tri_base = (uint32_t)tri_order.size();
        w.masks = imask | (lmask << 8);
        for (int a = 0; a < 3; ++a)
            for (int s = 0; s < 8; ++s) {
                uint16_t lo = 0x4000, hi = 0;                       // empty child: lo = 2 > hi = 0, never hit
                if (child_at[s] >= 0) {
                    const BuildNode& c = bn[items[child_at[s]].bnode];
                    lo = bf16_down(((double)c.bmin[a] - mn[a]) / E[a]);
                    hi = bf16_up(((double)c.bmax[a] - mn[a]) / E[a]);
                    if ((s & 1) && lo > 0) --lo;                    // high-half entry is read with the low half as extra mantissa bits
                }
                const int word = s >> 1, sh = (s & 1) * 16;
                w.planes[a][word] |= (uint32_t)lo << sh;
                w.planes[a][4 + word] |= (uint32_t)hi << sh;
            }
        // ---- children: inner nodes get consecutive indices, triangles consecutive positions, both in slot order
        const size_t first_child = wn.size();
        wn.resize(first_child + (size_t)n_inner);
        int k = 0;
        for (int s = 0; s < 8; ++s) {
            if (child_at[s] < 0) continue;
            const int32_t bi = items[child_at[s]].bnode;
            if (bn[bi].left >= 0) queue.push_back({bi, (int32_t)(first_child + (size_t)k++), pd.depth + 1});
            else tri_order.push_back(b->prim[bn[bi].first]);
        }
        wn[(size_t)pd.windex] = w;
    }
}

// Conservativeness of the encoding, evaluated in double: every triangle must lie inside the box that the kernel reconstructs
// for each of its ancestors (including the enlargement of high-half entries), every triangle must appear exactly once and
// empty slots must be unhittable.  Returns a bit set of violations (0 = sound).
int32_t crt_bvh_check_wide(const crt_bvh* b, const std::vector<WNode>& wn, const std::vector<int32_t>& tri_order)
{
    int32_t bad = 0;
    if (b->n_tris == 0) return 0;
    std::vector<uint8_t> seen((size_t)b->n_tris, 0);
    struct Ent { uint32_t node; double mn[3], mx[3]; };
    std::vector<Ent> stack;
    Ent root; root.node = 0; for (int a = 0; a < 3; ++a) { root.mn[a] = -1e300; root.mx[a] = 1e300; }
    stack.push_back(root);
    while (!stack.empty()) {
        Ent e = stack.back(); stack.pop_back();
        if (e.node >= wn.size()) { bad |= 32; continue; }
        const WNode& w = wn[e.node];
        const double p[3] = {w.px, w.py, w.pz};
        const double E[3] = {w.ex, u2f(w.eyz & 0xffff0000u), u2f(w.eyz << 16)};
        const uint32_t imask = w.masks & 0xff, lmask = (w.masks >> 8) & 0xff;
        if (imask & lmask) bad |= 2;
        int ki = 0, kl = 0;
        for (int s = 0; s < 8; ++s) {
            double lo[3], hi[3];
            for (int a = 0; a < 3; ++a) {
                const uint32_t wl = w.planes[a][s >> 1], wh = w.planes[a][4 + (s >> 1)];
                // what the kernel sees: low-half entries exactly, high-half entries with the low half as extra mantissa bits
                const float flo = (s & 1) ? u2f(wl) : u2f(wl << 16), fhi = (s & 1) ? u2f(wh) : u2f(wh << 16);
                lo[a] = p[a] + (double)flo * E[a]; hi[a] = p[a] + (double)fhi * E[a];
            }
            const bool inner = (imask >> s) & 1, leaf = (lmask >> s) & 1;
            if (!inner && !leaf) { if (!(lo[0] > hi[0])) bad |= 64; continue; }
            // a ray reaches this child only through every ancestor's box: keep the intersection of them
            for (int a = 0; a < 3; ++a) { lo[a] = std::max(lo[a], e.mn[a]); hi[a] = std::min(hi[a], e.mx[a]); }
            if (inner) {
                Ent c; c.node = w.child_base + (uint32_t)ki++;
                for (int a = 0; a < 3; ++a) { c.mn[a] = lo[a]; c.mx[a] = hi[a]; }
                stack.push_back(c);
            } else {
                const size_t pos = (size_t)w.tri_base + (size_t)kl++;
                if (pos >= tri_order.size()) { bad |= 32; continue; }
                const int32_t prim = tri_order[pos];
                if (prim < 0 || prim >= b->n_tris) { bad |= 32; continue; }
                if (seen[prim]) bad |= 4;
                seen[prim] = 1;
                const float* tv = b->verts.data() + 9 * (int64_t)prim;
                for (int v = 0; v < 3; ++v) for (int a = 0; a < 3; ++a) if (tv[3 * v + a] < lo[a] || tv[3 * v + a] > hi[a]) bad |= 8;
            }
        }
    }
    for (uint8_t s : seen) if (!s) bad |= 16;
    return bad;
}
