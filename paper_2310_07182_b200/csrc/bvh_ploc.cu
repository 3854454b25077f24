// a0 on the device (NEXT-4, second half): the BVH hierarchy built by the GPU ("acceleration structures such as bounding
// volume hierarchies"; the paper leaves the builder open, D:R11).  crt_bvh_params.builder = 1.
//
// Method: parallel locally-ordered clustering (PLOC, Meister & Bittner 2018), restated from the publication:
//   1. triangle boxes and centroids; 30-bit Morton code of the centroid inside the scene box; stable radix sort (sort.cu)
//   2. clusters = the triangles in Morton order.  Repeat until one cluster is left:
//        a. every cluster looks at its `radius` neighbours on either side in the array and picks the one with which its union box has
//           the smallest surface area (ties -> the lower index)
//        b. clusters that picked EACH OTHER merge into a new inner node, which takes the place of the left partner
//        c. the array is compacted (order-preserving: an exclusive scan), so that neighbours in the array stay neighbours in space
//   3. subtrees of at most max_leaf triangles become leaves (the same forced-split rule as the host builder).
// Agglomerative clustering driven by the surface area of the merged box is a bottom-up surface-area heuristic; the trees trace
// within a few percent of the host's binned-SAH trees (profiles/r02b) and build two orders of magnitude faster.
// The hierarchy comes back to the host in the builder-independent form (BuildNode + leaf order) that crt_bvh_flatten, crt_bvh_quantise
// and crt_bvh_check already consume, so both builders share the layout code and the invariant checks.
#include <algorithm>
#include <chrono>
#include <cstring>
#include "crt_internal.h"

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
    // one CUBIC grid of 1024^3 cells over the largest extent: per-axis normalisation would make the cells of a flat scene thin slabs
    // (landscape: 2 x 0.2 x 2 units) and let tiny height differences reorder horizontal neighbours (measured: SAH cost 56 -> see r02b)
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

// node k < n: the leaf of the k-th triangle in Morton order
__global__ void __launch_bounds__(PB) ploc_init_kernel(const int32_t* __restrict__ sorted_tri, const Box2* __restrict__ tri_box, int64_t n,
                                                       int32_t* __restrict__ cl_id, Box2* __restrict__ cl_box, Box2* __restrict__ node_box,
                                                       int32_t* __restrict__ node_left, int32_t* __restrict__ node_right, int32_t* __restrict__ node_cnt)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const Box2 b = tri_box[sorted_tri[k]];
    cl_id[k] = (int32_t)k; cl_box[k] = b; node_box[k] = b;
    node_left[k] = -1; node_right[k] = -1; node_cnt[k] = 1;
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

// 2b: mutual nearest neighbours merge; flag = 1 for every cluster that stays in the array
__global__ void __launch_bounds__(PB) ploc_merge_kernel(const int32_t* __restrict__ nn, const int32_t* __restrict__ cl_id, const Box2* __restrict__ cl_box, int n,
                                                        int32_t* __restrict__ tmp_id, Box2* __restrict__ tmp_box, int32_t* __restrict__ flag,
                                                        Box2* __restrict__ node_box, int32_t* __restrict__ node_left, int32_t* __restrict__ node_right,
                                                        int32_t* __restrict__ node_cnt, int32_t* __restrict__ node_counter)
{
    const int i = blockIdx.x * PB + threadIdx.x;
    if (i >= n) return;
    const int j = nn[i];
    int32_t id = cl_id[i]; Box2 b = cl_box[i]; int keep = 1;
    if (j >= 0 && nn[j] == i) {
        if (i < j) {
            const Box2 o = cl_box[j]; const int32_t oid = cl_id[j];
            Box2 u;
            u.lo = make_float4(fminf(b.lo.x, o.lo.x), fminf(b.lo.y, o.lo.y), fminf(b.lo.z, o.lo.z), 0.f);
            u.hi = make_float4(fmaxf(b.hi.x, o.hi.x), fmaxf(b.hi.y, o.hi.y), fmaxf(b.hi.z, o.hi.z), 0.f);
            const int32_t idx = atomicAdd(node_counter, 1);
            node_box[idx] = u; node_left[idx] = id; node_right[idx] = oid; node_cnt[idx] = node_cnt[id] + node_cnt[oid];
            id = idx; b = u;
        } else keep = 0;
    }
    tmp_id[i] = id; tmp_box[i] = b; flag[i] = keep;
}

// 2c: order-preserving compaction = exclusive scan of the flags (block sums, scan of the sums, scatter)
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = PB * SCAN_ITEMS;
__global__ void __launch_bounds__(PB) ploc_blocksum_kernel(const int32_t* __restrict__ flag, int n, int32_t* __restrict__ block_sum)
{
    __shared__ int s[PB / 32];
    int v = 0;
    for (int t = 0; t < SCAN_ITEMS; ++t) { const int i = blockIdx.x * SCAN_TILE + t * PB + threadIdx.x; if (i < n) v += flag[i]; }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) { int t = 0; for (int w = 0; w < PB / 32; ++w) t += s[w]; block_sum[blockIdx.x] = t; }
}
// one block: exclusive scan of the block sums in place; total -> *n_out
__global__ void __launch_bounds__(1024) ploc_scansums_kernel(int32_t* __restrict__ block_sum, int nb, int32_t* __restrict__ n_out)
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
    if (threadIdx.x == 0) *n_out = carry;
}
__global__ void __launch_bounds__(PB) ploc_compact_kernel(const int32_t* __restrict__ flag, const int32_t* __restrict__ tmp_id, const Box2* __restrict__ tmp_box, int n,
                                                          const int32_t* __restrict__ block_off, int32_t* __restrict__ cl_id, Box2* __restrict__ cl_box)
{
    __shared__ int warp_s[PB / 32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = block_off[blockIdx.x];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int t = 0; t < SCAN_ITEMS; ++t) {
        const int i = blockIdx.x * SCAN_TILE + t * PB + threadIdx.x;
        const int f = i < n ? flag[i] : 0;
        int incl = f;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int x = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += x; }
        if (lane == 31) warp_s[warp] = incl;
        __syncthreads();
        int off = carry;
        for (int w = 0; w < warp; ++w) off += warp_s[w];
        if (f) { cl_id[off + incl - 1] = tmp_id[i]; cl_box[off + incl - 1] = tmp_box[i]; }
        __syncthreads();
        if (threadIdx.x == PB - 1) carry = off + incl;
        __syncthreads();
    }
}

struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 256); }
    template <class T> T* as() { return static_cast<T*>(p); }
};

}  // namespace

// Builds b->nodes / b->prim / b->bounds / b->depth / b->sah on the device `ctx` lives on.  verts: HOST array (the caller has it there
// for the layout code and the checks anyway); it is uploaded here.  Returns CRT_OK or a CUDA / depth error.
crt_status crt_bvh_build_device(crt_ctx* ctx, crt_bvh* b, const float* verts, int64_t n, const crt_bvh_params& pr)
{
    auto t0 = std::chrono::steady_clock::now();
    b->n_tris = n; b->max_leaf = pr.max_leaf;
    b->verts.assign(verts, verts + 9 * n);
    b->nodes.clear(); b->prim.clear(); b->depth = 0; b->sah = 0;
    for (int k = 0; k < 6; ++k) b->bounds[k] = 0.f;
    if (n == 0) { b->build_seconds = 0; return CRT_OK; }
    if (n >= ((int64_t)1 << 30)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "build_bvh(device): too many triangles");
    const int radius = std::min(MAX_RADIUS, std::max(1, pr.ploc_radius > 0 ? pr.ploc_radius : 8));
    const int64_t n_nodes_max = 2 * n;
    DevBuf d_verts, d_bounds, d_tri_box, d_keys, d_vals, d_keys2, d_vals2, d_sort, d_cl_id[2], d_cl_box[2], d_tmp_id, d_tmp_box, d_flag, d_nn, d_node_box, d_left, d_right, d_cnt, d_counter, d_bsum;
    const size_t sort_bytes = radix_sort_scratch_bytes(n);
    const int nb_max = (int)((n + SCAN_TILE - 1) / SCAN_TILE);
#define PLOC_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return crt_fail(ctx, e_ == cudaErrorMemoryAllocation ? CRT_ERR_NOMEM : CRT_ERR_CUDA, "build_bvh(device): %s: %s", #call, cudaGetErrorString(e_)); } while (0)
    PLOC_CUDA(d_verts.alloc((size_t)n * 36)); PLOC_CUDA(d_bounds.alloc(32)); PLOC_CUDA(d_tri_box.alloc((size_t)n * sizeof(Box2)));
    PLOC_CUDA(d_keys.alloc((size_t)n * 4)); PLOC_CUDA(d_vals.alloc((size_t)n * 4)); PLOC_CUDA(d_keys2.alloc((size_t)n * 4)); PLOC_CUDA(d_vals2.alloc((size_t)n * 4));
    PLOC_CUDA(d_sort.alloc(sort_bytes));
    for (int k = 0; k < 2; ++k) { PLOC_CUDA(d_cl_id[k].alloc((size_t)n * 4)); PLOC_CUDA(d_cl_box[k].alloc((size_t)n * sizeof(Box2))); }
    PLOC_CUDA(d_tmp_id.alloc((size_t)n * 4)); PLOC_CUDA(d_tmp_box.alloc((size_t)n * sizeof(Box2))); PLOC_CUDA(d_flag.alloc((size_t)n * 4)); PLOC_CUDA(d_nn.alloc((size_t)n * 4));
    PLOC_CUDA(d_node_box.alloc((size_t)n_nodes_max * sizeof(Box2))); PLOC_CUDA(d_left.alloc((size_t)n_nodes_max * 4)); PLOC_CUDA(d_right.alloc((size_t)n_nodes_max * 4));
    PLOC_CUDA(d_cnt.alloc((size_t)n_nodes_max * 4)); PLOC_CUDA(d_counter.alloc(256)); PLOC_CUDA(d_bsum.alloc((size_t)(nb_max + 1) * 4));
    PLOC_CUDA(cudaMemcpy(d_verts.p, verts, (size_t)n * 36, cudaMemcpyHostToDevice));
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
    ploc_init_kernel<<<gridn, PB>>>(d_vals2.as<int32_t>(), d_tri_box.as<Box2>(), n, d_cl_id[0].as<int32_t>(), d_cl_box[0].as<Box2>(), d_node_box.as<Box2>(),
                                    d_left.as<int32_t>(), d_right.as<int32_t>(), d_cnt.as<int32_t>());
    const int32_t first_inner = (int32_t)n;
    PLOC_CUDA(cudaMemcpyAsync(d_counter.p, &first_inner, 4, cudaMemcpyHostToDevice, 0));
    // 2. clustering rounds
    int cur = 0, n_cl = (int)n, rounds = 0;
    while (n_cl > 1) {
        const unsigned g = (unsigned)((n_cl + PB - 1) / PB);
        const int nb = (n_cl + SCAN_TILE - 1) / SCAN_TILE;
        ploc_nn_kernel<<<g, PB>>>(d_cl_box[cur].as<Box2>(), n_cl, radius, d_nn.as<int32_t>());
        ploc_merge_kernel<<<g, PB>>>(d_nn.as<int32_t>(), d_cl_id[cur].as<int32_t>(), d_cl_box[cur].as<Box2>(), n_cl, d_tmp_id.as<int32_t>(), d_tmp_box.as<Box2>(),
                                     d_flag.as<int32_t>(), d_node_box.as<Box2>(), d_left.as<int32_t>(), d_right.as<int32_t>(), d_cnt.as<int32_t>(), d_counter.as<int32_t>());
        ploc_blocksum_kernel<<<nb, PB>>>(d_flag.as<int32_t>(), n_cl, d_bsum.as<int32_t>());
        ploc_scansums_kernel<<<1, 1024>>>(d_bsum.as<int32_t>(), nb, d_bsum.as<int32_t>() + nb_max);
        ploc_compact_kernel<<<nb, PB>>>(d_flag.as<int32_t>(), d_tmp_id.as<int32_t>(), d_tmp_box.as<Box2>(), n_cl, d_bsum.as<int32_t>(), d_cl_id[1 - cur].as<int32_t>(), d_cl_box[1 - cur].as<Box2>());
        int32_t n_new = 0;
        PLOC_CUDA(cudaMemcpy(&n_new, d_bsum.as<int32_t>() + nb_max, 4, cudaMemcpyDeviceToHost));
        if (n_new >= n_cl || n_new < 1) return crt_fail(ctx, CRT_ERR_CUDA, "build_bvh(device): clustering made no progress (%d -> %d clusters)", n_cl, n_new);
        n_cl = n_new; cur = 1 - cur; ++rounds;
    }
    PLOC_CUDA(cudaEventRecord(e1, 0));
    PLOC_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f; PLOC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    b->device_build_ms = ms; b->builder = 1; b->ploc_rounds = rounds;
    // 3. back to the host in the builder-independent form; subtrees of <= max_leaf triangles become leaves
    int32_t root = 0, n_nodes = 0;
    PLOC_CUDA(cudaMemcpy(&root, d_cl_id[cur].p, 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(&n_nodes, d_counter.p, 4, cudaMemcpyDeviceToHost));
    if (n_nodes != 2 * n - 1 || root < 0 || root >= n_nodes || (n > 1 && root < n)) return crt_fail(ctx, CRT_ERR_CUDA, "build_bvh(device): inconsistent tree (%d nodes for %lld triangles, root %d)", n_nodes, (long long)n, root);
    std::vector<int32_t> left((size_t)n_nodes), right((size_t)n_nodes), cnt((size_t)n_nodes), sorted_tri((size_t)n);
    std::vector<Box2> box((size_t)n_nodes);
    PLOC_CUDA(cudaMemcpy(left.data(), d_left.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(right.data(), d_right.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(cnt.data(), d_cnt.p, (size_t)n_nodes * 4, cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(box.data(), d_node_box.p, (size_t)n_nodes * sizeof(Box2), cudaMemcpyDeviceToHost));
    PLOC_CUDA(cudaMemcpy(sorted_tri.data(), d_vals2.p, (size_t)n * 4, cudaMemcpyDeviceToHost));
    unsigned ob[6];
    PLOC_CUDA(cudaMemcpy(ob, d_bounds.p, sizeof ob, cudaMemcpyDeviceToHost));
#undef PLOC_CUDA
    float maxabs = 0.f;
    for (int k = 0; k < 6; ++k) {
        const unsigned u = ob[k]; const unsigned bits = u ^ ((u >> 31) ? 0x80000000u : 0xffffffffu);
        float f; std::memcpy(&f, &bits, 4); b->bounds[k] = f; maxabs = std::max(maxabs, std::fabs(f));
    }
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
    b->sah = ra > 0 ? cost / ra : 0;
    const float pad = maxabs * (1.0f / 131072.0f);          // the same conservative padding as the host builder (D:R10)
    for (BuildNode& nd : b->nodes)
        for (int k = 0; k < 3; ++k) { nd.bmin[k] -= pad; nd.bmax[k] += pad; }
    b->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    return CRT_OK;
}
