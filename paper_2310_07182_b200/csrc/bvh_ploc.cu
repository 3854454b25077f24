// a0 on the device (NEXT-4, second half): the BVH built by the GPU ("acceleration structures such as bounding volume
// hierarchies"; the paper leaves the builder open, D:R11).  crt_bvh_params.builder = 1 (everything on the device) or 2 (hierarchy on
// the device, layout by the host code the host builder uses: the cross-check of 1).
//
// Method: parallel locally-ordered clustering (PLOC, Meister & Bittner 2018), restated from the publication:
//   1. triangle boxes and centroids; 30-bit Morton code of the centroid on a cubic grid over the scene box; stable radix sort (sort.cu)
//   2. clusters = the triangles in Morton order.  Repeat until one cluster is left:
//        a. every cluster looks at its `radius` neighbours on either side in the array and picks the one with which its union box has
//           the smallest surface area (ties -> the lower index)
//        b. clusters that picked EACH OTHER merge into a new inner node, which takes the place of the left partner
//        c. the array is compacted (order-preserving: an exclusive scan), so that neighbours in the array stay neighbours in space
//      Node indices are a pure function of the input (rank of the dropped partner in its round, no atomics), children always have lower
//      indices than their parent, the root is the last node.
//   3. subtrees of at most max_leaf triangles become leaves (the same forced-split rule as the host builder).
//   4. (builder 1) the traversal layouts are written on the device: inner nodes numbered top-down (descending creation order, the root
//      first), every leaf gets a contiguous run of triangle records ordered by the Morton position of its first triangle, fp32 64-byte
//      nodes and 16-bit 32-byte nodes (the quantisation rule of crt_bvh_quantise: planes rounded outward plus one grid step) in one pass.
// Agglomerative clustering driven by the surface area of the merged box is a bottom-up surface-area heuristic; the trees trace within
// 3-10 % of the host's binned-SAH trees and build two orders of magnitude faster (profiles/r02b).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include "crt_internal.h"

void crt_qgrid_for_box(const double lo[3], const double hi[3], QGrid* grid);

namespace {

constexpr int PB = 256;                 // threads per block
constexpr int MAX_RADIUS = 128;

struct Box2 { float4 lo, hi; };        // lo.xyz = min, hi.xyz = max (w unused)

__device__ __forceinline__ unsigned ord_f(float f) { const unsigned b = __float_as_uint(f); return b ^ ((unsigned)((int)b >> 31) | 0x80000000u); }
__device__ __forceinline__ float unord_f(unsigned u) { return __uint_as_float(u ^ ((u >> 31) ? 0x80000000u : 0xffffffffu)); }

// bounds[0..2] = ordered(min), bounds[3..5] = ordered(max) of all vertices
__global__ void __launch_bounds__(PB) ploc_bounds_kernel(const float* __restrict__ verts, int64_t n, unsigned* __restrict__ bounds)
{
    float mn[3] = {3.0e38f, 3.0e38f, 3.0e38f}, mx[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float* tv = verts + 9 * i;
#pragma unroll
        for (int v = 0; v < 3; ++v)
#pragma unroll
            for (int k = 0; k < 3; ++k) { const float x = __ldg(tv + 3 * v + k); mn[k] = fminf(mn[k], x); mx[k] = fmaxf(mx[k], x); }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { mn[k] = fminf(mn[k], __shfl_xor_sync(0xffffffffu, mn[k], d)); mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xffffffffu, mx[k], d)); }
    if ((threadIdx.x & 31) == 0)
        for (int k = 0; k < 3; ++k) { atomicMin(bounds + k, ord_f(mn[k])); atomicMax(bounds + 3 + k, ord_f(mx[k])); }
}

__device__ __forceinline__ unsigned spread10(unsigned v)      // bit l of v -> bit 3*l
{
    v = (v | (v << 16)) & 0x030000FFu; v = (v | (v << 8)) & 0x0300F00Fu; v = (v | (v << 4)) & 0x030C30C3u; v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__global__ void __launch_bounds__(PB) ploc_prims_kernel(const float* __restrict__ verts, int64_t n, const unsigned* __restrict__ bounds,
                                                        Box2* __restrict__ tri_box, uint32_t* __restrict__ keys, int32_t* __restrict__ vals)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float* tv = verts + 9 * i;
    float mn[3], mx[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float a = __ldg(tv + k), b = __ldg(tv + 3 + k), c = __ldg(tv + 6 + k);
        mn[k] = fminf(a, fminf(b, c)); mx[k] = fmaxf(a, fmaxf(b, c));
    }
    Box2 bx; bx.lo = make_float4(mn[0], mn[1], mn[2], 0.f); bx.hi = make_float4(mx[0], mx[1], mx[2], 0.f);
    tri_box[i] = bx;
    // one CUBIC grid of 1024^3 cells over the largest extent: per-axis normalisation makes the cells of a flat scene thin slabs (landscape:
    // 2 x 0.2 x 2 units) and lets tiny height differences reorder horizontal neighbours (measured: SAH cost 56.7 -> 50.2, profiles/r02b)
    unsigned q[3];
    float maxext = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) maxext = fmaxf(maxext, unord_f(bounds[3 + k]) - unord_f(bounds[k]));
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float lo = unord_f(bounds[k]);
        const float c = 0.5f * mn[k] + 0.5f * mx[k];
        const float t = maxext > 0.f ? (c - lo) / maxext * 1024.0f : 0.f;
        q[k] = (unsigned)fminf(fmaxf(t, 0.f), 1023.f);
    }
    keys[i] = (spread10(q[0]) << 2) | (spread10(q[1]) << 1) | spread10(q[2]);
    vals[i] = (int32_t)i;
}

// the hierarchy, node-indexed (2n - 1 nodes; node k < n = the leaf of the k-th triangle in Morton order)
struct Tree {
    Box2* box; int32_t *left, *right, *cnt, *parent, *first, *height;
};

__global__ void __launch_bounds__(PB) ploc_init_kernel(const int32_t* __restrict__ sorted_tri, const Box2* __restrict__ tri_box, int64_t n,
                                                       int32_t* __restrict__ cl_id, Box2* __restrict__ cl_box, Tree T)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const Box2 b = tri_box[sorted_tri[k]];
    cl_id[k] = (int32_t)k; cl_box[k] = b; T.box[k] = b;
    T.left[k] = -1; T.right[k] = -1; T.cnt[k] = 1; T.parent[k] = -1; T.first[k] = (int32_t)k; T.height[k] = 1;
}

__device__ __forceinline__ float union_area(const Box2& a, const Box2& b)
{
    const float dx = fmaxf(a.hi.x, b.hi.x) - fminf(a.lo.x, b.lo.x), dy = fmaxf(a.hi.y, b.hi.y) - fminf(a.lo.y, b.lo.y), dz = fmaxf(a.hi.z, b.hi.z) - fminf(a.lo.z, b.lo.z);
    return dx * dy + dy * dz + dz * dx;
}

// 2a: nearest neighbour (by the surface area of the union box) within `radius` positions on either side
__global__ void __launch_bounds__(PB) ploc_nn_kernel(const Box2* __restrict__ cl_box, int n, int radius, int32_t* __restrict__ nn)
{
    __shared__ Box2 s_box[PB + 2 * MAX_RADIUS];
    const int b0 = blockIdx.x * PB;
    for (int t = threadIdx.x; t < PB + 2 * radius; t += PB) {
        const int j = b0 - radius + t;
        if (j >= 0 && j < n) s_box[t] = cl_box[j];
    }
    __syncthreads();
    const int i = b0 + threadIdx.x;
    if (i >= n) return;
    const Box2 me = s_box[threadIdx.x + radius];
    float best = 3.0e38f; int best_j = -1;
    const int j0 = max(0, i - radius), j1 = min(n - 1, i + radius);
    for (int j = j0; j <= j1; ++j) {
        if (j == i) continue;
        const float a = union_area(me, s_box[j - b0 + radius]);
        if (a < best) { best = a; best_j = j; }
    }
    nn[i] = best_j;
}

// 2b: a cluster stays in the array unless it is the RIGHT partner of a mutual pair
__global__ void __launch_bounds__(PB) ploc_mark_kernel(const int32_t* __restrict__ nn, int n, int32_t* __restrict__ keep)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    if (i >= n) return;
    const int j = nn[i];
    keep[i] = !(j >= 0 && nn[j] == i && j < i);
}

// ---- exclusive scan of n ints (block sums, one-block scan of the sums, per-block scan + offset)
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = PB * SCAN_ITEMS;
__global__ void __launch_bounds__(PB) scan_blocksum_kernel(const int32_t* __restrict__ in, int n, int32_t* __restrict__ block_sum)
{
    __shared__ int s[PB / 32];
    int v = 0;
    for (int t = 0; t < SCAN_ITEMS; ++t) { const int i = blockIdx.x * SCAN_TILE + t * PB + threadIdx.x; if (i < n) v += in[i]; }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) { int t = 0; for (int w = 0; w < PB / 32; ++w) t += s[w]; block_sum[blockIdx.x] = t; }
}
__global__ void __launch_bounds__(1024) scan_sums_kernel(int32_t* __restrict__ block_sum, int nb, int32_t* __restrict__ total)
{
    __shared__ int warp_s[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = i < nb ? block_sum[i] : 0;
        int incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += t; }
        if (lane == 31) warp_s[warp] = incl;
        __syncthreads();
        int off = carry;
        for (int w = 0; w < warp; ++w) off += warp_s[w];
        if (i < nb) block_sum[i] = off + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = off + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry;
}
__global__ void __launch_bounds__(PB) scan_write_kernel(const int32_t* __restrict__ in, int n, const int32_t* __restrict__ block_off, int32_t* __restrict__ out)
{
    __shared__ int warp_s[PB / 32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = block_off[blockIdx.x];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int t = 0; t < SCAN_ITEMS; ++t) {
        const int i = blockIdx.x * SCAN_TILE + t * PB + threadIdx.x;
        const int f = i < n ? in[i] : 0;
        int incl = f;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int x = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += x; }
        if (lane == 31) warp_s[warp] = incl;
        __syncthreads();
        int off = carry;
        for (int w = 0; w < warp; ++w) off += warp_s[w];
        if (i < n) out[i] = off + incl - f;
        __syncthreads();
        if (threadIdx.x == PB - 1) carry = off + incl;
        __syncthreads();
    }
}
// out[i] = sum of in[0..i); *total (device) = sum of all.  bsum: scratch of ceil(n / SCAN_TILE) + 1 ints.
void exclusive_scan(const int32_t* in, int32_t* out, int n, int32_t* bsum, int32_t* total)
{
    const int nb = (n + SCAN_TILE - 1) / SCAN_TILE;
    scan_blocksum_kernel<<<nb, PB>>>(in, n, bsum);
    scan_sums_kernel<<<1, 1024>>>(bsum, nb, total);
    scan_write_kernel<<<nb, PB>>>(in, n, bsum, out);
}

// 2b + 2c: a merged pair (i < j) becomes node base + (number of dropped clusters before j): a pure function of the input.  The new node,
// or the unmerged cluster, goes to position pos[i] = (number of kept clusters before i) of the next array.
__global__ void __launch_bounds__(PB) ploc_build_kernel(const int32_t* __restrict__ nn, const int32_t* __restrict__ keep, const int32_t* __restrict__ pos,
                                                        const int32_t* __restrict__ cl_id, const Box2* __restrict__ cl_box, int n, int32_t node_base,
                                                        int32_t* __restrict__ new_id, Box2* __restrict__ new_box, Tree T)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    if (i >= n || !keep[i]) return;
    const int j = nn[i];
    int32_t id = cl_id[i]; Box2 b = cl_box[i];
    if (j >= 0 && nn[j] == i) {          // i < j, or i would not have been kept
        const Box2 o = cl_box[j]; const int32_t oid = cl_id[j];
        Box2 u;
        u.lo = make_float4(fminf(b.lo.x, o.lo.x), fminf(b.lo.y, o.lo.y), fminf(b.lo.z, o.lo.z), 0.f);
        u.hi = make_float4(fmaxf(b.hi.x, o.hi.x), fmaxf(b.hi.y, o.hi.y), fmaxf(b.hi.z, o.hi.z), 0.f);
        const int32_t idx = node_base + (j - pos[j]);
        T.box[idx] = u; T.left[idx] = id; T.right[idx] = oid; T.cnt[idx] = T.cnt[id] + T.cnt[oid]; T.parent[idx] = -1;
        T.first[idx] = min(T.first[id], T.first[oid]); T.height[idx] = 1 + max(T.height[id], T.height[oid]);
        T.parent[id] = idx; T.parent[oid] = idx;
        id = idx; b = u;
    }
    new_id[pos[i]] = id; new_box[pos[i]] = b;
}

// ---- 4. traversal layouts on the device
// inner[i] = 1 for nodes that stay inner nodes; w[first triangle position] = triangle count for the roots of collapsed subtrees (leaves)
__global__ void __launch_bounds__(PB) layout_classify_kernel(Tree T, int n_nodes, int max_leaf, int32_t* __restrict__ inner, int32_t* __restrict__ w)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    if (i >= n_nodes) return;
    const int c = T.cnt[i];
    inner[i] = c > max_leaf;
    const int p = T.parent[i];
    if (c <= max_leaf && (p < 0 || T.cnt[p] > max_leaf)) w[T.first[i]] = c;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// leaves: triangle records in the leaf's run of slots, left to right; ref[i] = the child reference a parent stores for node i
__global__ void __launch_bounds__(PB) layout_leaves_kernel(Tree T, int n_nodes, int max_leaf, const int32_t* __restrict__ inner_before, int n_inner,
                                                           const int32_t* __restrict__ slot_start, const int32_t* __restrict__ sorted_tri,
                                                           const float* __restrict__ verts, GpuTri* __restrict__ tris, int32_t* __restrict__ slot_of_prim,
                                                           int32_t* __restrict__ ref, double cost_intersect, double* __restrict__ sums)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    double area = 0.0;
    if (i < n_nodes) {
        const int c = T.cnt[i];
        const int p = T.parent[i];
        if (c > max_leaf) ref[i] = n_inner - 1 - inner_before[i];                 // inner nodes are numbered in descending creation order: the root is node 0
        else if (p < 0 || T.cnt[p] > max_leaf) {
            const int slot = slot_start[T.first[i]];
            ref[i] = ~((slot << 3) | (c - 1));
            int stack[16]; int sp = 0, k = 0; stack[sp++] = i;
            while (sp) {
                const int s = stack[--sp];
                if (T.left[s] < 0) {
                    const int tri = sorted_tri[s];
                    const float* tv = verts + 9 * (int64_t)tri;
                    GpuTri t;
                    t.v0p = make_float4(tv[0], tv[1], tv[2], __int_as_float(tri));
                    t.e1 = make_float4(tv[3] - tv[0], tv[4] - tv[1], tv[5] - tv[2], 0.f);
                    t.e2 = make_float4(tv[6] - tv[0], tv[7] - tv[1], tv[8] - tv[2], 0.f);
                    t.pad = make_float4(0.f, 0.f, 0.f, 0.f);
                    tris[slot + k] = t; slot_of_prim[tri] = slot + k; ++k;
                } else { stack[sp++] = T.right[s]; stack[sp++] = T.left[s]; }
            }
            const Box2 b = T.box[i];
            const double dx = (double)b.hi.x - b.lo.x, dy = (double)b.hi.y - b.lo.y, dz = (double)b.hi.z - b.lo.z;
            area = (dx * dy + dy * dz + dz * dx) * cost_intersect * c;
        }
    }
    area = warp_sum(area);
    if ((threadIdx.x & 31) == 0 && area != 0.0) atomicAdd(sums + 0, area);
}

// inner nodes: fp32 node and 16-bit node (crt_bvh_quantise's rule) of both children
__global__ void __launch_bounds__(PB) layout_nodes_kernel(Tree T, int n_nodes, int max_leaf, const int32_t* __restrict__ ref, float pad, QGrid grid,
                                                          GpuNode* __restrict__ gn, QNode* __restrict__ qn, double cost_traversal, double* __restrict__ sums, int32_t* __restrict__ q_bad)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    double cost = 0.0, area_f = 0.0, area_q = 0.0;
    if (i < n_nodes && T.cnt[i] > max_leaf) {
        const int g = ref[i];
        GpuNode N; QNode Q; int bad = 0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const int ch = c ? T.right[i] : T.left[i];
            const Box2 b = T.box[ch];
            const float mn[3] = {b.lo.x - pad, b.lo.y - pad, b.lo.z - pad}, mx[3] = {b.hi.x + pad, b.hi.y + pad, b.hi.z + pad};
            N.c[c].min_x = mn[0]; N.c[c].max_x = mx[0]; N.c[c].min_y = mn[1]; N.c[c].max_y = mx[1]; N.c[c].min_z = mn[2]; N.c[c].max_z = mx[2];
            N.c[c].ref = ref[ch]; N.c[c].pad = 0;
            Q.ref[c] = ref[ch];
            double ef[3], eq[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double gm = (double)grid.gmin[k], s = (double)grid.scale[k];
                double a = floor(((double)mn[k] - gm) * s), z = ceil(((double)mx[k] - gm) * s);
                if (gm + a / s > (double)mn[k]) a -= 1.0;
                if (gm + z / s < (double)mx[k]) z += 1.0;
                a -= 1.0; z += 1.0;
                if (a < 0.0) { a = 0.0; bad = 1; }
                if (z > 65535.0) { z = 65535.0; bad = 1; }
                if (!(gm + (a + 1.0) / s <= (double)mn[k]) || !(gm + (z - 1.0) / s >= (double)mx[k])) bad = 1;
                Q.planes[3 * c + k] = (uint32_t)a | ((uint32_t)z << 16);
                ef[k] = (double)mx[k] - mn[k]; eq[k] = (z - a) / s;
            }
            area_f += ef[0] * ef[1] + ef[1] * ef[2] + ef[2] * ef[0]; area_q += eq[0] * eq[1] + eq[1] * eq[2] + eq[2] * eq[0];
        }
        gn[g] = N; qn[g] = Q;
        if (bad) atomicOr(q_bad, 1);
        const Box2 b = T.box[i];
        const double dx = (double)b.hi.x - b.lo.x, dy = (double)b.hi.y - b.lo.y, dz = (double)b.hi.z - b.lo.z;
        cost = (dx * dy + dy * dz + dz * dx) * cost_traversal;
    }
    cost = warp_sum(cost); area_f = warp_sum(area_f); area_q = warp_sum(area_q);
    if ((threadIdx.x & 31) == 0 && area_f != 0.0) { atomicAdd(sums + 0, cost); atomicAdd(sums + 1, area_f); atomicAdd(sums + 2, area_q); }
}

// ---- 2d. parallel re-insertion on the device (crt_bvh_params.optimize iterations; Meister & Bittner 2018, "Parallel reinsertion for bounding
// volume hierarchy optimization", restated).  Per iteration, on the binary clustering tree (before leaves are collapsed):
//   search : every node x (not the root, not a child of the root) looks for the node y beside which its subtree would add the least surface area:
//            removing x deletes its parent p (the sibling s takes p's place) and shrinks the ancestors; the search walks the ancestors a_k of x
//            ("pivots") upwards and descends, with a bound on the best gain so far, into the child of each pivot that does not contain x
//   lock   : a move touches x, p, s, the grandparent g, y and y's parent: each candidate writes (gain, x) into those six nodes with atomicMax
//   win    : x wins if it owns all six; a winner whose target y lies inside the subtree of ANOTHER winner steps back (two such moves could
//            hang each subtree under the other one: a cycle)
//   apply  : g adopts s; p becomes the parent of (y, x) in y's old place
//   refit  : boxes, triangle counts, first positions and heights bottom-up from the leaves (atomic arrival counters)
// A losing iteration cannot be told apart cheaply, so the summed inner area is reduced after each one and the loop stops when it no longer falls.
__device__ __forceinline__ float box_area(const Box2& a)
{
    const float dx = a.hi.x - a.lo.x, dy = a.hi.y - a.lo.y, dz = a.hi.z - a.lo.z;
    return dx * dy + dy * dz + dz * dx;
}
__device__ __forceinline__ Box2 box_union(const Box2& a, const Box2& b)
{
    Box2 u;
    u.lo = make_float4(fminf(a.lo.x, b.lo.x), fminf(a.lo.y, b.lo.y), fminf(a.lo.z, b.lo.z), 0.f);
    u.hi = make_float4(fmaxf(a.hi.x, b.hi.x), fmaxf(a.hi.y, b.hi.y), fmaxf(a.hi.z, b.hi.z), 0.f);
    return u;
}

constexpr int REINS_STACK = 72;          // per-thread search stack (the tree's height is checked against 60 after every iteration)
constexpr int REINS_MAX_VISITS = 768;    // nodes one search may look at

__global__ void __launch_bounds__(128) reins_search_kernel(Tree T, int n_nodes, int32_t* __restrict__ target, float* __restrict__ gain_out)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= n_nodes) return;
    target[x] = -1; gain_out[x] = 0.f;
    const int root = n_nodes - 1;
    const int p = T.parent[x];
    if (x == root || p < 0 || p == root) return;
    const Box2 bx = T.box[x];
    const float ax = box_area(bx);
    const int s = T.left[p] == x ? T.right[p] : T.left[p];
    int st_node[REINS_STACK]; float st_ind[REINS_STACK];
    float best = 0.f; int best_y = -1;
    float d_rem = box_area(T.box[p]);         // removal gain so far: p disappears; ancestors below the pivot shrink
    Box2 shrunk = T.box[s];                    // box of the path node below the pivot once x is gone
    int below = x, pivot = p, visits = 0;
    while (pivot >= 0 && visits < REINS_MAX_VISITS) {
        const int other = T.left[pivot] == below ? T.right[pivot] : T.left[pivot];
        int sp = 0;
        st_node[sp] = other; st_ind[sp] = 0.f; ++sp;
        while (sp > 0 && visits < REINS_MAX_VISITS) {
            --sp; const int y = st_node[sp]; const float ind = st_ind[sp];
            ++visits;
            const Box2 by = T.box[y];
            const float c = box_area(box_union(by, bx));
            const float g = d_rem - ind - c;
            if (g > best && y != s) { best = g; best_y = y; }
            const int l = T.left[y];
            if (l >= 0 && sp + 2 <= REINS_STACK) {
                const float ind_c = ind + (c - box_area(by));          // y itself grows by x when x goes below it
                if (d_rem - ind_c - ax > best) { st_node[sp] = T.right[y]; st_ind[sp] = ind_c; ++sp; st_node[sp] = l; st_ind[sp] = ind_c; ++sp; }
            }
        }
        // the pivot moves up: the old pivot (unless it is p, which is gone) keeps the shrunk box
        const int up = T.parent[pivot];
        if (up < 0) break;
        if (pivot != p) {
            shrunk = box_union(shrunk, T.box[other]);
            d_rem += box_area(T.box[pivot]) - box_area(shrunk);
        }
        below = pivot; pivot = up;
    }
    // a move must pay for the staleness of its estimate (other moves of the same iteration change the boxes it was computed on)
    if (best_y >= 0 && best > 1e-6f * ax) { target[x] = best_y; gain_out[x] = best; }
}

__device__ __forceinline__ unsigned long long reins_key(float gain, int x) { return ((unsigned long long)__float_as_uint(gain) << 32) | (unsigned)x; }

__global__ void __launch_bounds__(PB) reins_lock_kernel(Tree T, int n_nodes, const int32_t* __restrict__ target, const float* __restrict__ gain, unsigned long long* __restrict__ lock)
{
    const int x = blockIdx.x * PB + threadIdx.x;
    if (x >= n_nodes) return;
    const int y = target[x];
    if (y < 0) return;
    const int p = T.parent[x], s = T.left[p] == x ? T.right[p] : T.left[p], g = T.parent[p], yp = T.parent[y];
    const unsigned long long k = reins_key(gain[x], x);
    atomicMax(lock + x, k); atomicMax(lock + p, k); atomicMax(lock + s, k); atomicMax(lock + g, k); atomicMax(lock + y, k); atomicMax(lock + yp, k);
}

__global__ void __launch_bounds__(PB) reins_win_kernel(Tree T, int n_nodes, const int32_t* __restrict__ target, const float* __restrict__ gain, const unsigned long long* __restrict__ lock,
                                                       int32_t* __restrict__ win)
{
    const int x = blockIdx.x * PB + threadIdx.x;
    if (x >= n_nodes) return;
    const int y = target[x];
    int w = 0;
    if (y >= 0) {
        const int p = T.parent[x], s = T.left[p] == x ? T.right[p] : T.left[p], g = T.parent[p], yp = T.parent[y];
        const unsigned long long k = reins_key(gain[x], x);
        w = lock[x] == k && lock[p] == k && lock[s] == k && lock[g] == k && lock[y] == k && lock[yp] == k;
    }
    win[x] = w;
}

// a winner goes ahead unless an ancestor of its target is itself a winner (that subtree is about to move): decided for all winners BEFORE any pointer changes
__global__ void __launch_bounds__(PB) reins_filter_kernel(Tree T, int n_nodes, const int32_t* __restrict__ target, const int32_t* __restrict__ win, int32_t* __restrict__ go)
{
    const int x = blockIdx.x * PB + threadIdx.x;
    if (x >= n_nodes) return;
    int ok = win[x];
    if (ok) {
        int steps = 0;
        for (int a = T.parent[target[x]]; a >= 0; a = T.parent[a]) if (win[a] || ++steps > 4096) { ok = 0; break; }      // (4096: far beyond any height this file accepts)
    }
    go[x] = ok;
}

// the moves: every node a thread writes is one of the six it owns, so the writes of different threads never meet
__global__ void __launch_bounds__(PB) reins_apply_kernel(Tree T, int n_nodes, const int32_t* __restrict__ target, const int32_t* __restrict__ go, int32_t* __restrict__ n_applied)
{
    const int x = blockIdx.x * PB + threadIdx.x;
    if (x >= n_nodes || !go[x]) return;
    const int y = target[x];
    const int p = T.parent[x], s = T.left[p] == x ? T.right[p] : T.left[p], g = T.parent[p];
    if (T.left[g] == p) T.left[g] = s; else T.right[g] = s;          // g adopts s
    T.parent[s] = g;
    const int yp = T.parent[y];                                        // (may be g, or s)
    if (T.left[yp] == y) T.left[yp] = p; else T.right[yp] = p;         // p takes y's place ...
    T.parent[p] = yp;
    T.left[p] = y; T.right[p] = x; T.parent[y] = p;                   // ... as the parent of y and x
    atomicAdd(n_applied, 1);
}

// boxes, counts, first positions and heights of all inner nodes, bottom-up: the second thread to arrive at a node computes it and goes on
__global__ void __launch_bounds__(PB) reins_refit_kernel(Tree T, int n, int32_t* __restrict__ arrive)
{
    const int k = blockIdx.x * PB + threadIdx.x;
    if (k >= n) return;
    int i = k;
    for (;;) {
        const int p = T.parent[i];
        if (p < 0) break;
        __threadfence();
        if (atomicAdd(arrive + p, 1) != 1) break;          // the first arrival stops; the second goes on (anything else would mean a malformed tree: stop)
        const int l = T.left[p], r = T.right[p];
        Box2 a, b;
        a.lo = __ldcg(&T.box[l].lo); a.hi = __ldcg(&T.box[l].hi); b.lo = __ldcg(&T.box[r].lo); b.hi = __ldcg(&T.box[r].hi);
        T.box[p] = box_union(a, b);
        T.cnt[p] = __ldcg(T.cnt + l) + __ldcg(T.cnt + r);
        T.first[p] = min(__ldcg(T.first + l), __ldcg(T.first + r));
        T.height[p] = 1 + max(__ldcg(T.height + l), __ldcg(T.height + r));
        i = p;
    }
}

// summed surface area of the inner nodes (what the re-insertion lowers)
__global__ void __launch_bounds__(PB) reins_area_kernel(Tree T, int n, int n_nodes, double* __restrict__ total)
{
    const int i = n + blockIdx.x * PB + threadIdx.x;
    double a = i < n_nodes ? (double)box_area(T.box[i]) : 0.0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) a += __shfl_xor_sync(0xffffffffu, a, d);
    if ((threadIdx.x & 31) == 0 && a != 0.0) atomicAdd(total, a);
}

struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 256); }
    template <class T> T* as() { return static_cast<T*>(p); }
    void* release() { void* r = p; p = nullptr; return r; }
};

}  // namespace

#define PLOC_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return crt_fail(ctx, e_ == cudaErrorMemoryAllocation ? CRT_ERR_NOMEM : CRT_ERR_CUDA, "build_bvh(device): %s: %s", #call, cudaGetErrorString(e_)); } while (0)

// The re-insertion iterations on a device tree of n_leaves leaves (nodes [0, n_leaves)) and n_leaves - 1 inner nodes, the root last; boxes, counts, first
// positions and heights of the inner nodes are (re)computed by the refit.  *kept = iterations that lowered the summed inner area and were kept.
struct ReinsBufs {
    DevBuf d_target, d_gain, d_lock, d_win, d_go, d_arrive, d_bk[3], d_acc;
    cudaError_t alloc(int n_nodes)
    {
        cudaError_t e = cudaSuccess;
        for (DevBuf* d : {&d_target, &d_gain, &d_win, &d_go, &d_arrive, &d_bk[0], &d_bk[1], &d_bk[2]}) if (e == cudaSuccess) e = d->alloc((size_t)n_nodes * 4);
        if (e == cudaSuccess) e = d_lock.alloc((size_t)n_nodes * 8);
        if (e == cudaSuccess) e = d_acc.alloc(64);
        return e;
    }
};

static crt_status reinsertion_loop(crt_ctx* ctx, Tree T, int n_leaves, int n_nodes, int iterations, int* kept, ReinsBufs& R)
{
    *kept = 0;
    DevBuf &d_target = R.d_target, &d_gain = R.d_gain, &d_lock = R.d_lock, &d_win = R.d_win, &d_go = R.d_go, &d_arrive = R.d_arrive, &d_acc = R.d_acc;
    DevBuf* const d_bk = R.d_bk;
    const unsigned gnodes = (unsigned)((n_nodes + PB - 1) / PB), ginner = (unsigned)((n_nodes - n_leaves + PB - 1) / PB), gleaves = (unsigned)((n_leaves + PB - 1) / PB);
    int32_t* const topo[3] = {T.left, T.right, T.parent};
    struct Acc { double area; int32_t applied, pad; } acc;
    auto measure = [&](Acc* out) -> cudaError_t {
        cudaError_t e = cudaMemsetAsync(d_acc.p, 0, 64, 0); if (e != cudaSuccess) return e;
        reins_area_kernel<<<ginner, PB>>>(T, n_leaves, n_nodes, d_acc.as<double>());
        return cudaMemcpy(out, d_acc.p, sizeof(Acc), cudaMemcpyDeviceToHost);
    };
    auto refit = [&]() -> cudaError_t {
        cudaError_t e = cudaMemsetAsync(d_arrive.p, 0, (size_t)n_nodes * 4, 0); if (e != cudaSuccess) return e;
        reins_refit_kernel<<<gleaves, PB>>>(T, n_leaves, d_arrive.as<int32_t>());
        return cudaGetLastError();
    };
    PLOC_CUDA(measure(&acc));
    double prev_area = acc.area;
    for (int it = 0; it < iterations; ++it) {
        for (int k = 0; k < 3; ++k) PLOC_CUDA(cudaMemcpyAsync(d_bk[k].p, topo[k], (size_t)n_nodes * 4, cudaMemcpyDeviceToDevice, 0));
        reins_search_kernel<<<(unsigned)((n_nodes + 127) / 128), 128>>>(T, n_nodes, d_target.as<int32_t>(), d_gain.as<float>());
        PLOC_CUDA(cudaMemsetAsync(d_lock.p, 0, (size_t)n_nodes * 8, 0));
        reins_lock_kernel<<<gnodes, PB>>>(T, n_nodes, d_target.as<int32_t>(), d_gain.as<float>(), d_lock.as<unsigned long long>());
        reins_win_kernel<<<gnodes, PB>>>(T, n_nodes, d_target.as<int32_t>(), d_gain.as<float>(), d_lock.as<unsigned long long>(), d_win.as<int32_t>());
        reins_filter_kernel<<<gnodes, PB>>>(T, n_nodes, d_target.as<int32_t>(), d_win.as<int32_t>(), d_go.as<int32_t>());
        PLOC_CUDA(cudaMemsetAsync(d_acc.p, 0, 64, 0));
        reins_apply_kernel<<<gnodes, PB>>>(T, n_nodes, d_target.as<int32_t>(), d_go.as<int32_t>(), d_acc.as<int32_t>() + 2);
        int32_t applied = 0;
        PLOC_CUDA(cudaMemcpy(&applied, d_acc.as<int32_t>() + 2, 4, cudaMemcpyDeviceToHost));
        PLOC_CUDA(refit());
        PLOC_CUDA(measure(&acc));
        int32_t h = 0;
        PLOC_CUDA(cudaMemcpy(&h, T.height + (n_nodes - 1), 4, cudaMemcpyDeviceToHost));
        if (h > 56 || !(acc.area < prev_area)) {          // too deep for the traversal stack, or no gain: this iteration is undone
            for (int k = 0; k < 3; ++k) PLOC_CUDA(cudaMemcpyAsync(topo[k], d_bk[k].p, (size_t)n_nodes * 4, cudaMemcpyDeviceToDevice, 0));
            PLOC_CUDA(refit());
            break;
        }
        ++*kept;
        const bool small = prev_area - acc.area < 0.002 * prev_area;
        prev_area = acc.area;
        if (applied == 0 || small) break;
    }
    return CRT_OK;
}

// Builds the BVH of verts (HOST array; uploaded here) on the device `ctx` lives on.
//  full_device (builder 1): fills b->d_nodes, d_qnodes, d_tris, d_slot_of_prim, qgrid, q_violations, q_inflation, n_gpu_nodes, n_tree_nodes,
//                           bounds, depth, sah; no host tree (crt_bvh_check verifies the device layouts themselves).
//  otherwise (builder 2):   fills b->nodes / b->prim / bounds / depth / sah; the caller runs the host layout code.
crt_status crt_bvh_build_device(crt_ctx* ctx, crt_bvh* b, const float* verts, int64_t n, const crt_bvh_params& pr, bool full_device)
{
    auto t0 = std::chrono::steady_clock::now();
    b->n_tris = n; b->n_refs = n; b->max_leaf = pr.max_leaf;
    b->verts.assign(verts, verts + 9 * n);
    b->nodes.clear(); b->prim.clear(); b->depth = 0; b->sah = 0; b->builder = full_device ? 1 : 2;
    for (int k = 0; k < 6; ++k) b->bounds[k] = 0.f;
    if (n >= ((int64_t)1 << 27)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "build_bvh(device): too many triangles");
    const int radius = std::min(MAX_RADIUS, std::max(1, pr.ploc_radius > 0 ? pr.ploc_radius : 8));
    const int n_nodes = (int)(2 * n - 1);
    DevBuf d_verts, d_bounds, d_tri_box, d_keys, d_vals, d_keys2, d_vals2, d_sort, d_cl_id[2], d_cl_box[2], d_keep, d_pos, d_nn,
           d_box, d_left, d_right, d_cnt, d_parent, d_first, d_height, d_total, d_bsum;
    const size_t sort_bytes = radix_sort_scratch_bytes(n);
    const int nb_max = (int)((2 * n + SCAN_TILE - 1) / SCAN_TILE);
    PLOC_CUDA(d_verts.alloc((size_t)n * 36)); PLOC_CUDA(d_bounds.alloc(32)); PLOC_CUDA(d_tri_box.alloc((size_t)n * sizeof(Box2)));
    PLOC_CUDA(d_keys.alloc((size_t)n * 4)); PLOC_CUDA(d_vals.alloc((size_t)n * 4)); PLOC_CUDA(d_keys2.alloc((size_t)n * 4)); PLOC_CUDA(d_vals2.alloc((size_t)n * 4));
    PLOC_CUDA(d_sort.alloc(sort_bytes));
    for (int k = 0; k < 2; ++k) { PLOC_CUDA(d_cl_id[k].alloc((size_t)n * 4)); PLOC_CUDA(d_cl_box[k].alloc((size_t)n * sizeof(Box2))); }
    PLOC_CUDA(d_keep.alloc((size_t)2 * n * 4)); PLOC_CUDA(d_pos.alloc((size_t)2 * n * 4)); PLOC_CUDA(d_nn.alloc((size_t)n * 4));
    PLOC_CUDA(d_box.alloc((size_t)2 * n * sizeof(Box2)));
    for (DevBuf* d : {&d_left, &d_right, &d_cnt, &d_parent, &d_first, &d_height}) PLOC_CUDA(d->alloc((size_t)2 * n * 4));
    PLOC_CUDA(d_total.alloc(256)); PLOC_CUDA(d_bsum.alloc((size_t)(nb_max + 1) * 4));
    Tree T{d_box.as<Box2>(), d_left.as<int32_t>(), d_right.as<int32_t>(), d_cnt.as<int32_t>(), d_parent.as<int32_t>(), d_first.as<int32_t>(), d_height.as<int32_t>()};
    PLOC_CUDA(cudaMemcpy(d_verts.p, verts, (size_t)n * 36, cudaMemcpyHostToDevice));
    ReinsBufs reins;
    if (full_device && pr.optimize > 0 && n >= 8) PLOC_CUDA(reins.alloc(n_nodes));
    cudaEvent_t e0, e1;
    PLOC_CUDA(cudaEventCreate(&e0)); PLOC_CUDA(cudaEventCreate(&e1));
    PLOC_CUDA(cudaEventRecord(e0, 0));
    // 1. bounds, boxes, Morton keys, sort
    const unsigned init_bounds[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    PLOC_CUDA(cudaMemcpyAsync(d_bounds.p, init_bounds, sizeof init_bounds, cudaMemcpyHostToDevice, 0));
    ploc_bounds_kernel<<<ctx->n_sms * 8, PB>>>(d_verts.as<float>(), n, d_bounds.as<unsigned>());
    const unsigned gridn = (unsigned)((n + PB - 1) / PB);
    ploc_prims_kernel<<<gridn, PB>>>(d_verts.as<float>(), n, d_bounds.as<unsigned>(), d_tri_box.as<Box2>(), d_keys.as<uint32_t>(), d_vals.as<int32_t>());
    crt_status st = launch_radix_sort(ctx, d_keys.as<uint32_t>(), d_vals.as<int32_t>(), n, d_keys2.as<uint32_t>(), d_vals2.as<int32_t>(), d_sort.p, sort_bytes, 0);
    if (st != CRT_OK) return st;
    ploc_init_kernel<<<gridn, PB>>>(d_vals2.as<int32_t>(), d_tri_box.as<Box2>(), n, d_cl_id[0].as<int32_t>(), d_cl_box[0].as<Box2>(), T);
    // 2. clustering rounds
    int cur = 0, n_cl = (int)n, rounds = 0; int32_t node_base = (int32_t)n;
    while (n_cl > 1) {
        const unsigned g = (unsigned)((n_cl + PB - 1) / PB);
        ploc_nn_kernel<<<g, PB>>>(d_cl_box[cur].as<Box2>(), n_cl, radius, d_nn.as<int32_t>());
        ploc_mark_kernel<<<g, PB>>>(d_nn.as<int32_t>(), n_cl, d_keep.as<int32_t>());
        exclusive_scan(d_keep.as<int32_t>(), d_pos.as<int32_t>(), n_cl, d_bsum.as<int32_t>(), d_total.as<int32_t>());
        ploc_build_kernel<<<g, PB>>>(d_nn.as<int32_t>(), d_keep.as<int32_t>(), d_pos.as<int32_t>(), d_cl_id[cur].as<int32_t>(), d_cl_box[cur].as<Box2>(), n_cl, node_base,
                                     d_cl_id[1 - cur].as<int32_t>(), d_cl_box[1 - cur].as<Box2>(), T);
        int32_t n_new = 0;
        PLOC_CUDA(cudaMemcpy(&n_new, d_total.p, 4, cudaMemcpyDeviceToHost));
        if (n_new >= n_cl || n_new < 1) return crt_fail(ctx, CRT_ERR_CUDA, "build_bvh(device): clustering made no progress (%d -> %d clusters)", n_cl, n_new);
        node_base += n_cl - n_new; n_cl = n_new; cur = 1 - cur; ++rounds;
    }
    if (node_base != n_nodes) return crt_fail(ctx, CRT_ERR_CUDA, "build_bvh(device): inconsistent tree (%d nodes for %lld triangles)", node_base, (long long)n);
    const int root = n_nodes - 1;
    b->ploc_rounds = rounds;
    // 2d. parallel re-insertion (builder 1; builder 2 runs the host's optimisation on the tree it copies back)
    b->opt_iters = 0;
    if (full_device && pr.optimize > 0 && n >= 8) {
        const crt_status rst = reinsertion_loop(ctx, T, (int)n, n_nodes, pr.optimize, &b->opt_iters, reins);
        if (rst != CRT_OK) return rst;
    }
    unsigned ob[6]; int32_t height = 0;
    PLOC_CUDA(cudaMemcpy(ob, d_bounds.p, sizeof ob, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(&height, d_height.as<int32_t>() + root, 4, cudaMemcpyDeviceToHost));
    float maxabs = 0.f;
    for (int k = 0; k < 6; ++k) {
        const unsigned u = ob[k]; const unsigned bits = u ^ ((u >> 31) ? 0x80000000u : 0xffffffffu);
        float f; std::memcpy(&f, &bits, 4); b->bounds[k] = f; maxabs = std::max(maxabs, std::fabs(f));
    }
    const float pad = maxabs * (1.0f / 131072.0f);          // the same conservative padding as the host builder (D:R10)
    if (full_device) {
        // 4. layouts on the device
        DevBuf d_w, d_slot, d_ref, d_sums, d_qbad, d_gn, d_qn, d_gt, d_sop;
        PLOC_CUDA(d_w.alloc((size_t)n * 4)); PLOC_CUDA(d_slot.alloc((size_t)n * 4)); PLOC_CUDA(d_ref.alloc((size_t)n_nodes * 4));
        PLOC_CUDA(d_sums.alloc(64)); PLOC_CUDA(d_qbad.alloc(16));
        PLOC_CUDA(cudaMemsetAsync(d_w.p, 0, (size_t)n * 4, 0)); PLOC_CUDA(cudaMemsetAsync(d_sums.p, 0, 64, 0)); PLOC_CUDA(cudaMemsetAsync(d_qbad.p, 0, 16, 0));
        const unsigned gn_grid = (unsigned)((n_nodes + PB - 1) / PB);
        int32_t* inner = d_keep.as<int32_t>(); int32_t* inner_before = d_pos.as<int32_t>();
        layout_classify_kernel<<<gn_grid, PB>>>(T, n_nodes, pr.max_leaf, inner, d_w.as<int32_t>());
        exclusive_scan(inner, inner_before, n_nodes, d_bsum.as<int32_t>(), d_total.as<int32_t>());
        int32_t n_inner = 0;
        PLOC_CUDA(cudaMemcpy(&n_inner, d_total.p, 4, cudaMemcpyDeviceToHost));
        exclusive_scan(d_w.as<int32_t>(), d_slot.as<int32_t>(), (int)n, d_bsum.as<int32_t>(), d_total.as<int32_t>());
        if (n_inner < 1) return crt_fail(ctx, CRT_ERR_STATE, "build_bvh(device): the whole scene is one leaf (use the host builder)");
        PLOC_CUDA(d_gn.alloc((size_t)n_inner * sizeof(GpuNode))); PLOC_CUDA(d_qn.alloc((size_t)n_inner * sizeof(QNode)));
        PLOC_CUDA(d_gt.alloc((size_t)n * sizeof(GpuTri))); PLOC_CUDA(d_sop.alloc((size_t)n * 4));
        double glo[3], ghi[3];
        for (int k = 0; k < 3; ++k) { glo[k] = (double)(b->bounds[k] - pad); ghi[k] = (double)(b->bounds[3 + k] + pad); }
        crt_qgrid_for_box(glo, ghi, &b->qgrid);
        layout_leaves_kernel<<<gn_grid, PB>>>(T, n_nodes, pr.max_leaf, inner_before, n_inner, d_slot.as<int32_t>(), d_vals2.as<int32_t>(), d_verts.as<float>(),
                                              d_gt.as<GpuTri>(), d_sop.as<int32_t>(), d_ref.as<int32_t>(), (double)pr.cost_intersect, d_sums.as<double>() + 3);
        layout_nodes_kernel<<<gn_grid, PB>>>(T, n_nodes, pr.max_leaf, d_ref.as<int32_t>(), pad, b->qgrid, d_gn.as<GpuNode>(), d_qn.as<QNode>(),
                                             (double)pr.cost_traversal, d_sums.as<double>(), d_qbad.as<int32_t>());
        PLOC_CUDA(cudaEventRecord(e1, 0));
        PLOC_CUDA(cudaEventSynchronize(e1));
        PLOC_CUDA(cudaGetLastError());
        double sums[4]; int32_t qbad = 0; Box2 rb;
        PLOC_CUDA(cudaMemcpy(sums, d_sums.p, sizeof sums, cudaMemcpyDeviceToHost));
        PLOC_CUDA(cudaMemcpy(&qbad, d_qbad.p, 4, cudaMemcpyDeviceToHost));
        PLOC_CUDA(cudaMemcpy(&rb, d_box.as<Box2>() + root, sizeof rb, cudaMemcpyDeviceToHost));
        const double ra = ((double)rb.hi.x - rb.lo.x) * ((double)rb.hi.y - rb.lo.y) + ((double)rb.hi.y - rb.lo.y) * ((double)rb.hi.z - rb.lo.z) + ((double)rb.hi.z - rb.lo.z) * ((double)rb.hi.x - rb.lo.x);
        b->sah = ra > 0 ? (sums[0] + sums[3]) / ra : 0;
        b->q_violations = qbad; b->q_inflation = sums[1] > 0 ? sums[2] / sums[1] : 1.0;
        b->depth = height;                                   // height of the binary clustering tree: an upper bound of the collapsed tree's depth
        b->n_gpu_nodes = n_inner; b->n_tree_nodes = 2 * (int64_t)n_inner + 1;
        b->device = ctx->device;
        b->device_bytes += (int64_t)n_inner * (sizeof(GpuNode) + sizeof(QNode)) + (int64_t)n * (sizeof(GpuTri) + 4);
        b->d_nodes = static_cast<GpuNode*>(d_gn.release()); b->d_qnodes = static_cast<QNode*>(d_qn.release());
        b->d_tris = static_cast<GpuTri*>(d_gt.release()); b->d_slot_of_prim = static_cast<int32_t*>(d_sop.release());
        float ms = 0.f; PLOC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        cudaEventDestroy(e0); cudaEventDestroy(e1);
        b->device_build_ms = ms;
        b->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        return CRT_OK;
    }
    PLOC_CUDA(cudaEventRecord(e1, 0));
    PLOC_CUDA(cudaEventSynchronize(e1));
    PLOC_CUDA(cudaGetLastError());
    float ms = 0.f; PLOC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    b->device_build_ms = ms;
    // 3. (builder 2) back to the host in the builder-independent form; subtrees of <= max_leaf triangles become leaves
    std::vector<int32_t> left((size_t)n_nodes), right((size_t)n_nodes), cnt((size_t)n_nodes), sorted_tri((size_t)n);
    std::vector<Box2> box((size_t)n_nodes);
    PLOC_CUDA(cudaMemcpy(left.data(), d_left.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(right.data(), d_right.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(cnt.data(), d_cnt.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(box.data(), d_box.p, (size_t)n_nodes * sizeof(Box2), cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(sorted_tri.data(), d_vals2.p, (size_t)n * 4, cudaMemcpyDeviceToHost));
    b->nodes.reserve((size_t)n_nodes); b->prim.reserve((size_t)n);
    struct Item { int32_t src, dst, depth; };
    std::vector<Item> stack; std::vector<int32_t> sub;
    b->nodes.emplace_back(); stack.push_back({root, 0, 1});
    int max_depth = 0; double cost = 0;
    auto half_area = [](const Box2& x) { double dx = (double)x.hi.x - x.lo.x, dy = (double)x.hi.y - x.lo.y, dz = (double)x.hi.z - x.lo.z; return dx * dy + dy * dz + dz * dx; };
    while (!stack.empty()) {
        const Item it = stack.back(); stack.pop_back();
        BuildNode nd;
        const Box2& bx = box[it.src];
        nd.bmin[0] = bx.lo.x; nd.bmin[1] = bx.lo.y; nd.bmin[2] = bx.lo.z; nd.bmax[0] = bx.hi.x; nd.bmax[1] = bx.hi.y; nd.bmax[2] = bx.hi.z;
        max_depth = std::max(max_depth, it.depth);
        if (cnt[it.src] <= pr.max_leaf) {
            nd.left = nd.right = -1; nd.first = (int32_t)b->prim.size(); nd.count = cnt[it.src];
            sub.assign(1, it.src);
            while (!sub.empty()) {          // the triangles of the collapsed subtree, left to right
                const int32_t s = sub.back(); sub.pop_back();
                if (left[s] < 0) b->prim.push_back(sorted_tri[s]); else { sub.push_back(right[s]); sub.push_back(left[s]); }
            }
            cost += half_area(bx) * (double)pr.cost_intersect * nd.count;
        } else {
            const int32_t c = (int32_t)b->nodes.size();
            nd.left = c; nd.right = c + 1; nd.first = 0; nd.count = 0;
            b->nodes.emplace_back(); b->nodes.emplace_back();
            stack.push_back({right[it.src], c + 1, it.depth + 1}); stack.push_back({left[it.src], c, it.depth + 1});
            cost += half_area(bx) * (double)pr.cost_traversal;
        }
        b->nodes[it.dst] = nd;
    }
    b->depth = max_depth;
    const double ra = half_area(box[root]);
    if (pr.optimize > 0) {          // the host builder's insertion-based optimisation on the clustering tree (same leaves); cost recounted on the result
        b->depth = crt_bvh_optimize_tree(b, pr, max_depth);
        cost = 0;
        for (const BuildNode& x : b->nodes) {
            const double dx = (double)x.bmax[0] - x.bmin[0], dy = (double)x.bmax[1] - x.bmin[1], dz = (double)x.bmax[2] - x.bmin[2];
            cost += (dx * dy + dy * dz + dz * dx) * (x.left >= 0 ? (double)pr.cost_traversal : (double)pr.cost_intersect * x.count);
        }
    }
    b->sah = ra > 0 ? cost / ra : 0;
    for (BuildNode& nd : b->nodes)
        for (int k = 0; k < 3; ++k) { nd.bmin[k] -= pad; nd.bmax[k] += pad; }
    b->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return CRT_OK;
}

// The same parallel re-insertion for a HOST-built tree (crt_build_bvh, builder 0 with a context): b->nodes goes to the device in the index convention
// of this file (leaves first, the root last; a leaf of several triangles is one atomic node), is optimised, and comes back as b->nodes with the root
// at 0 and siblings adjacent; leaves keep their triangle ranges.  Boxes may be padded or not (a union of padded boxes is the padded union).
// collapse_max_leaf > 1: the host tree has one reference per leaf; after the optimisation subtrees of at most that many references become leaves (b->prim is
// rewritten in the new leaf order).  Returns the iterations kept in b->opt_iters and the new depth in b->depth.
crt_status crt_bvh_reinsert_device(crt_ctx* ctx, crt_bvh* b, int iterations, int collapse_max_leaf)
{
    b->opt_iters = 0;
    const int n_nodes = (int)b->nodes.size();
    if (iterations <= 0 || n_nodes < 15 || (n_nodes & 1) == 0) return CRT_OK;
    const int n_leaves = (n_nodes + 1) / 2;
    // new indices: leaves 0 .. n_leaves - 1 in order of appearance, inner nodes in REVERSE order of appearance after them (the root, node 0, becomes the last)
    std::vector<int32_t> idx((size_t)n_nodes);
    { int l = 0, in = 0; for (int i = 0; i < n_nodes; ++i) idx[i] = b->nodes[i].left < 0 ? l++ : n_nodes - 1 - in++; if (l != n_leaves) return crt_fail(ctx, CRT_ERR_STATE, "build_bvh: tree is not a full binary tree"); }
    std::vector<Box2> box((size_t)n_nodes); std::vector<int32_t> left((size_t)n_nodes, -1), right((size_t)n_nodes, -1), parent((size_t)n_nodes, -1), cnt((size_t)n_nodes, 0), first((size_t)n_nodes, 0), height((size_t)n_nodes, 1);
    std::vector<int32_t> leaf_of((size_t)n_leaves);          // device leaf -> host node (for the triangle range)
    for (int i = 0; i < n_nodes; ++i) {
        const BuildNode& nd = b->nodes[i]; const int k = idx[i];
        box[k].lo = make_float4(nd.bmin[0], nd.bmin[1], nd.bmin[2], 0.f); box[k].hi = make_float4(nd.bmax[0], nd.bmax[1], nd.bmax[2], 0.f);
        if (nd.left >= 0) { left[k] = idx[nd.left]; right[k] = idx[nd.right]; parent[idx[nd.left]] = k; parent[idx[nd.right]] = k; }
        else { cnt[k] = nd.count; first[k] = k; leaf_of[k] = i; }
    }
    DevBuf d_box, d_left, d_right, d_cnt, d_parent, d_first, d_height, d_arrive;
    PLOC_CUDA(d_box.alloc((size_t)n_nodes * sizeof(Box2)));
    for (DevBuf* d : {&d_left, &d_right, &d_cnt, &d_parent, &d_first, &d_height, &d_arrive}) PLOC_CUDA(d->alloc((size_t)n_nodes * 4));
    PLOC_CUDA(cudaMemcpy(d_box.p, box.data(), (size_t)n_nodes * sizeof(Box2), cudaMemcpyHostToDevice));
    PLOC_CUDA(cudaMemcpy(d_left.p, left.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice)); PLOC_CUDA(cudaMemcpy(d_right.p, right.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice));
    PLOC_CUDA(cudaMemcpy(d_parent.p, parent.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice)); PLOC_CUDA(cudaMemcpy(d_cnt.p, cnt.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice));
    PLOC_CUDA(cudaMemcpy(d_first.p, first.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice)); PLOC_CUDA(cudaMemcpy(d_height.p, height.data(), (size_t)n_nodes * 4, cudaMemcpyHostToDevice));
    Tree T{d_box.as<Box2>(), d_left.as<int32_t>(), d_right.as<int32_t>(), d_cnt.as<int32_t>(), d_parent.as<int32_t>(), d_first.as<int32_t>(), d_height.as<int32_t>()};
    PLOC_CUDA(cudaMemset(d_arrive.p, 0, (size_t)n_nodes * 4));
    reins_refit_kernel<<<(unsigned)((n_leaves + PB - 1) / PB), PB>>>(T, n_leaves, d_arrive.as<int32_t>());          // inner counts and heights in this file's form
    ReinsBufs reins;
    PLOC_CUDA(reins.alloc(n_nodes));
    const crt_status st = reinsertion_loop(ctx, T, n_leaves, n_nodes, iterations, &b->opt_iters, reins);
    if (st != CRT_OK) return st;
    if (b->opt_iters == 0 && collapse_max_leaf <= 1) return CRT_OK;          // nothing kept: the host tree stays as it is
    PLOC_CUDA(cudaMemcpy(box.data(), d_box.p, (size_t)n_nodes * sizeof(Box2), cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(left.data(), d_left.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost)); PLOC_CUDA(cudaMemcpy(right.data(), d_right.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(height.data(), d_height.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(cnt.data(), d_cnt.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    // back to the host form: root at 0, the two children of a node adjacent, depth-first
    std::vector<BuildNode> out((size_t)n_nodes);
    struct Item { int32_t src, dst; };
    std::vector<Item> stack{{n_nodes - 1, 0}};
    int32_t next = 1; int64_t seen = 0;
    std::vector<int32_t> new_prim, sub;
    if (collapse_max_leaf > 1) {
        // the tree was built and optimised with one reference per leaf; subtrees of at most collapse_max_leaf references become leaves now
        new_prim.reserve(b->prim.size());
        int depth = 0; std::vector<std::pair<Item, int>> st2{{{n_nodes - 1, 0}, 1}};
        out.clear(); out.emplace_back();
        while (!st2.empty()) {
            const Item it = st2.back().first; const int d = st2.back().second; st2.pop_back();
            depth = std::max(depth, d);
            BuildNode nd;
            nd.bmin[0] = box[it.src].lo.x; nd.bmin[1] = box[it.src].lo.y; nd.bmin[2] = box[it.src].lo.z; nd.bmax[0] = box[it.src].hi.x; nd.bmax[1] = box[it.src].hi.y; nd.bmax[2] = box[it.src].hi.z;
            if (cnt[it.src] <= collapse_max_leaf) {
                nd.left = nd.right = -1; nd.first = (int32_t)new_prim.size();
                sub.assign(1, it.src);
                while (!sub.empty()) {
                    const int32_t q = sub.back(); sub.pop_back();
                    if (left[q] >= 0) { sub.push_back(right[q]); sub.push_back(left[q]); continue; }
                    const BuildNode& old = b->nodes[leaf_of[q]];
                    for (int j = 0; j < old.count; ++j) {
                        const int32_t pr_id = b->prim[old.first + j];
                        bool dup = false; for (size_t m = (size_t)nd.first; m < new_prim.size(); ++m) dup |= new_prim[m] == pr_id;
                        if (!dup) new_prim.push_back(pr_id);          // two references of one triangle in one leaf: one record is enough
                    }
                }
                nd.count = (int32_t)new_prim.size() - nd.first;
            } else {
                const int32_t c = (int32_t)out.size();
                nd.left = c; nd.right = c + 1; nd.first = 0; nd.count = 0;
                if ((int64_t)out.size() + 2 > n_nodes) return crt_fail(ctx, CRT_ERR_STATE, "build_bvh: re-insertion left an inconsistent tree");
                out.emplace_back(); out.emplace_back();
                st2.push_back({{right[it.src], c + 1}, d + 1}); st2.push_back({{left[it.src], c}, d + 1});
            }
            out[it.dst] = nd;
        }
        b->nodes.swap(out); b->prim.swap(new_prim); b->n_refs = (int64_t)b->prim.size();
        b->depth = depth;
        return CRT_OK;
    }
    while (!stack.empty()) {
        const Item it = stack.back(); stack.pop_back(); ++seen;
        BuildNode nd;
        nd.bmin[0] = box[it.src].lo.x; nd.bmin[1] = box[it.src].lo.y; nd.bmin[2] = box[it.src].lo.z; nd.bmax[0] = box[it.src].hi.x; nd.bmax[1] = box[it.src].hi.y; nd.bmax[2] = box[it.src].hi.z;
        if (left[it.src] >= 0) {
            if (next + 2 > n_nodes) return crt_fail(ctx, CRT_ERR_STATE, "build_bvh: re-insertion left an inconsistent tree");
            nd.left = next; nd.right = next + 1; nd.first = 0; nd.count = 0;
            stack.push_back({right[it.src], next + 1}); stack.push_back({left[it.src], next});
            next += 2;
        } else {
            const BuildNode& old = b->nodes[leaf_of[it.src]];
            nd.left = nd.right = -1; nd.first = old.first; nd.count = old.count;
        }
        out[it.dst] = nd;
    }
    if (seen != n_nodes || next != n_nodes) return crt_fail(ctx, CRT_ERR_STATE, "build_bvh: re-insertion left an inconsistent tree (%lld of %d nodes reachable)", (long long)seen, n_nodes);
    b->nodes.swap(out);
    b->depth = height[n_nodes - 1];
    return CRT_OK;
}
