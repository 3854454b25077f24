// a5, trace_kernel 5: BVH traversal with a WARP-COOPERATIVE TRIANGLE PHASE (intersection is "the most time-consuming
// segment"; warps lose lanes to divergence).  An alternative to the default kernel of trace.cu, kept with its measurements
// (profiles/r02a: same hit records, 15-25 % SLOWER: the triangle phase shrinks from 174 M to 111 M warp instructions per launch,
// but the warp-uniform node loop stalls lanes that meet a second leaf (19 instead of 20 live lanes), its shared memory takes 60 KB
// of L1 per SM (+6 % time by itself) and the kernel is bound by memory latency, not by the instruction count).
//
// Why: in the per-lane kernel (trace.cu) the triangle phase runs at 6-12 live lanes of 32 and holds a third of the warp
// instructions (profiles/r01f, r02a): a lane tests the 1-3 triangles of ITS leaf while the lanes without a leaf, or with a
// shorter one, idle.  Here the triangles of all leaves a warp has parked become ONE work list in shared memory (positions from
// three ballots, no atomics) and are tested one item per lane, every lane busy: the ray of an item is read from a shared-memory
// mirror of the warp's rays, the result goes to the owner's (t, id) record with a 64-bit atomicMin whose ordering IS the
// closest-hit rule of D:R10 (smaller t, then lower primitive id); the owner refreshes its pruning bound after the phase.
// The node loop is the one of trace.cu (16-bit 32-byte nodes, one LDG.256, PRMT + FFMA per plane, predicated push/pop) minus the
// ray's origin and direction, which only the triangle test needs and which now live in shared memory; the whole loop is
// warp-uniform (rounds of CRT_TQ_VISITS visits, then a vote), so idle lanes can take part in the triangle tests.
//
// Exactness: the triangle test is the same bit-exact sequence (crt_device.cuh); the box test only ever uses a bound >= the best t
// of the ray, so the result is the all-triangles definition whatever the order in which items are tested.
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

constexpr int STACK_SIZE = 64;
constexpr int SENTINEL = 0x7fffffff;
constexpr int TQ_BLOCK = 128;                 // 4 warps
constexpr int TQ_WARPS = TQ_BLOCK / 32;
constexpr int TQ_ITEMS = 96;                  // work list of one leaf phase: 32 lanes x one parked leaf x at most 3 triangles
#ifndef CRT_TQ_VISITS
#define CRT_TQ_VISITS 3
#endif
constexpr int TQ_VISITS = CRT_TQ_VISITS;      // node visits per round (between two votes)
#ifndef CRT_TQ_MINB
#define CRT_TQ_MINB 8
#endif

struct WarpShared {
    float4 ro[32], rd[32];            // each lane's current ray: ox oy oz tmin | dx dy dz tmax
    unsigned long long best[32];      // (ordered(t) << 32) | prim of the nearest hit so far; starts at (ordered(tmax) << 32) | 0xffffffff (prim -1)
    float2 uv[32];                    // barycentrics of that hit
    unsigned items[TQ_ITEMS];         // the work list of one leaf phase: (owner lane << 27) | index into the leaf-ordered triangle array
};

// monotone map float -> unsigned (negative t can only occur with a negative tmin)
CRT_DEV unsigned ordered(float f) { const unsigned b = __float_as_uint(f); return b ^ ((unsigned)((int)b >> 31) | 0x80000000u); }
CRT_DEV float unordered(unsigned u) { return __uint_as_float(u ^ ((u >> 31) ? 0x80000000u : 0xffffffffu)); }

CRT_DEV float safe_rcp(float d)
{
    const float eps = 8.673617379884035e-19f;      // 2^-60 (trace.cu: a zero direction component must not give an infinite reciprocal)
    return dvd(1.0f, fabsf(d) > eps ? d : copysignf(eps, d));
}

// per-ray constants of the 16-bit box test (trace.cu QRay<false>: same arithmetic, same error budget)
struct QRayQ {
    float sx, sy, sz, cx, cy, cz;
    unsigned nx, ny, nz, fx, fy, fz;
    float tmin, best_t;
    CRT_DEV void init(float4 ro, float4 rd, const QGrid& g)
    {
        const float ix = safe_rcp(rd.x), iy = safe_rcp(rd.y), iz = safe_rcp(rd.z);
        sx = ix * g.inv_scale[0]; sy = iy * g.inv_scale[1]; sz = iz * g.inv_scale[2];
        const float px = (ro.x - g.gmin[0]) * g.scale[0], py = (ro.y - g.gmin[1]) * g.scale[1], pz = (ro.z - g.gmin[2]) * g.scale[2];
        cx = __fmaf_rn(-8388608.f, sx, -(px * sx)); cy = __fmaf_rn(-8388608.f, sy, -(py * sy)); cz = __fmaf_rn(-8388608.f, sz, -(pz * sz));
        nx = rd.x >= 0.f ? 0x7610u : 0x7632u; ny = rd.y >= 0.f ? 0x7610u : 0x7632u; nz = rd.z >= 0.f ? 0x7610u : 0x7632u;
        fx = nx ^ 0x0022u; fy = ny ^ 0x0022u; fz = nz ^ 0x0022u;
        tmin = ro.w; best_t = rd.w;
    }
};
CRT_DEV float qplane(unsigned w, unsigned sel, float s, float c)
{
    unsigned f;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(f) : "r"(w), "r"(0x4B000000u), "r"(sel));
    return __fmaf_rn(__uint_as_float(f), s, c);
}
CRT_DEV int visit_qnode(const QNode* __restrict__ nodes, int idx, const QRayQ& q, int*& top)
{
    unsigned w0, w1, w2, w3, w4, w5; int ra, rb;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(ra), "=r"(rb) : "l"(nodes + idx));
    const float tfar = q.best_t * 1.0000005f;
    const float tn0 = fmaxf(fmaxf(qplane(w0, q.nx, q.sx, q.cx), qplane(w1, q.ny, q.sy, q.cy)), fmaxf(qplane(w2, q.nz, q.sz, q.cz), q.tmin));
    const float tf0 = fminf(fminf(qplane(w0, q.fx, q.sx, q.cx), qplane(w1, q.fy, q.sy, q.cy)), fminf(qplane(w2, q.fz, q.sz, q.cz), tfar));
    const float tn1 = fmaxf(fmaxf(qplane(w3, q.nx, q.sx, q.cx), qplane(w4, q.ny, q.sy, q.cy)), fmaxf(qplane(w5, q.nz, q.sz, q.cz), q.tmin));
    const float tf1 = fminf(fminf(qplane(w3, q.fx, q.sx, q.cx), qplane(w4, q.fy, q.sy, q.cy)), fminf(qplane(w5, q.fz, q.sz, q.cz), tfar));
    const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
    const bool second = h1 && (!h0 || tn1 < tn0);
    int next = second ? rb : ra;
    if (h0 && h1) *++top = second ? ra : rb;
    if (!(h0 || h1)) next = *top--;
    return next;
}

// Tests items [base, base + count) of the warp's work list, one per lane (count <= 32).
template <bool COUNT>
CRT_DEV void test_batch(WarpShared& S, unsigned base, unsigned count, unsigned lane, const GpuTri* __restrict__ tris, unsigned& c_tris)
{
    bool hit = false; unsigned long long key = 0; int owner = 0; float u = 0.f, v = 0.f;
    if (lane < count) {
        const unsigned e = S.items[base + lane];
        owner = (int)(e >> 27);
        const char* tp = reinterpret_cast<const char*>(tris + (e & 0x7ffffffu));
        float4 a, b, c;
        asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(tp));
        asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(c.x), "=f"(c.y), "=f"(c.z), "=f"(c.w) : "l"(tp + 32));
        const float4 ro = S.ro[owner], rd = S.rd[owner];
        float t;
        if (COUNT) ++c_tris;
        if (tri_test(mk(a.x, a.y, a.z), mk(b.x, b.y, b.z), mk(c.x, c.y, c.z), mk(ro.x, ro.y, ro.z), mk(rd.x, rd.y, rd.z), ro.w, rd.w, t, u, v)) {
            key = ((unsigned long long)ordered(t) << 32) | (unsigned)__float_as_int(a.w);
            // smaller t wins, then the lower primitive id (D:R10); t < tmax was checked by the test, so any hit beats the initial record
            hit = atomicMin(&S.best[owner], key) > key;
        }
    }
    __syncwarp();
    if (hit && S.best[owner] == key) S.uv[owner] = make_float2(u, v);
}

template <bool COUNT>
__global__ void __launch_bounds__(TQ_BLOCK, CRT_TQ_MINB) trace_queue_kernel(const QNode* __restrict__ qnodes, const QGrid grid, const GpuTri* __restrict__ tris,
                                                                           const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n,
                                                                           unsigned int* __restrict__ counter, int refill_threshold, int leaf_wait,
                                                                           unsigned long long* __restrict__ stats)
{
    __shared__ WarpShared shared[TQ_WARPS];
    WarpShared& S = shared[threadIdx.x >> 5];
    const unsigned lane = threadIdx.x & 31u;
    int stack[STACK_SIZE]; int* top = stack; stack[0] = SENTINEL;
    int node = SENTINEL, leaf = 0;            // leaf: parked leaf reference (< 0) or 0
    int ray_idx = -1;
    bool exhausted = false;                   // uniform across the warp
    QRayQ q; q.best_t = 0.f; q.tmin = 0.f; q.sx = q.sy = q.sz = q.cx = q.cy = q.cz = 0.f; q.nx = q.ny = q.nz = q.fx = q.fy = q.fz = 0u;
    unsigned c_nodes = 0, c_tris = 0, c_rays = 0;

    for (;;) {
        // ---- 1. when few lanes have work left: finished rays retire, idle lanes take the next rays in slot order
        const int n_busy = __popc(__ballot_sync(0xffffffffu, node != SENTINEL || leaf != 0));
        if (n_busy == 0 || (!exhausted && n_busy < refill_threshold)) {
            if (ray_idx >= 0 && node == SENTINEL && leaf == 0) {
                if (!COUNT) {
                    // the record IS the hit record: t = the nearest hit's (or still the ray's tmax), prim = its id (or still -1)
                    const unsigned long long k = S.best[lane];
                    const float2 uv = S.uv[lane];
                    reinterpret_cast<float4*>(hits)[ray_idx] = make_float4(unordered((unsigned)(k >> 32)), uv.x, uv.y, __int_as_float((int)(unsigned)k));
                }
                ray_idx = -1;
            }
            while (!exhausted) {
                const bool want = ray_idx < 0;
                const unsigned m = __ballot_sync(0xffffffffu, want);
                if (m == 0u) break;
                unsigned base = 0;
                const int leader = __ffs(m) - 1;
                if ((int)lane == leader) base = atomicAdd(counter, (unsigned)__popc(m));
                base = __shfl_sync(0xffffffffu, base, leader);
                bool past_end = false;
                if (want) {
                    unsigned lt_mask;
                    asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt_mask));
                    const unsigned i = base + __popc(m & lt_mask);
                    if ((int64_t)i >= n) { past_end = true; }
                    else {
                        const float4* rp = reinterpret_cast<const float4*>(rays + i);
                        const float4 rd = __ldg(rp + 1);
                        if (rd.w < 0.f) {                 // inactive slot: a miss, nothing to traverse
                            if (!COUNT) reinterpret_cast<float4*>(hits)[i] = make_float4(rd.w, 0.f, 0.f, __int_as_float(-1));
                        } else {
                            const float4 ro = __ldg(rp);
                            q.init(ro, rd, grid);
                            S.ro[lane] = ro; S.rd[lane] = rd;
                            S.best[lane] = ((unsigned long long)ordered(rd.w) << 32) | 0xffffffffull; S.uv[lane] = make_float2(0.f, 0.f);
                            ray_idx = (int)i; node = 0; leaf = 0; top = stack;
                            if (COUNT) ++c_rays;
                        }
                    }
                }
                exhausted = __any_sync(0xffffffffu, past_end);
            }
            if (__ballot_sync(0xffffffffu, ray_idx >= 0) == 0u) break;     // every lane idle and the ray list exhausted
            __syncwarp();
        }

        // ---- 2. a round of node visits; the first leaf a lane meets is parked and the descent goes on
#pragma unroll
        for (int rep = 0; rep < TQ_VISITS; ++rep) {
            if ((unsigned)node < (unsigned)SENTINEL) {
                if (COUNT) ++c_nodes;
                node = visit_qnode(qnodes, node, q, top);
                if (node < 0 && leaf == 0) { leaf = node; node = *top--; }
            }
        }

        // ---- 3. leaf phase, once (nearly) every lane that is still descending holds a leaf: the triangles of all parked leaves
        //         become one work list and are tested one per lane
        const unsigned need = __ballot_sync(0xffffffffu, (unsigned)node < (unsigned)SENTINEL && leaf == 0);
        const unsigned b1 = __ballot_sync(0xffffffffu, leaf < 0);
        if (b1 != 0u && __popc(need) <= leaf_wait) {
            const int l = ~leaf;
            const unsigned cnt = leaf < 0 ? (unsigned)(l & 7) + 1u : 0u, item = (lane << 27) | (unsigned)(l >> 3);
            const unsigned b2 = __ballot_sync(0xffffffffu, cnt >= 2u), b3 = __ballot_sync(0xffffffffu, cnt >= 3u);
            unsigned lt_mask;
            asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt_mask));
            const unsigned pos = __popc(b1 & lt_mask) + __popc(b2 & lt_mask) + __popc(b3 & lt_mask);
            const unsigned total = __popc(b1) + __popc(b2) + __popc(b3);
            if (cnt >= 1u) S.items[pos] = item;
            if (cnt >= 2u) S.items[pos + 1] = item + 1u;
            if (cnt >= 3u) S.items[pos + 2] = item + 2u;
            __syncwarp();
            for (unsigned base = 0; base < total; base += 32u) test_batch<COUNT>(S, base, min(32u, total - base), lane, tris, c_tris);
            __syncwarp();
            if (ray_idx >= 0) q.best_t = unordered((unsigned)(S.best[lane] >> 32));
            leaf = 0;
            if (node < 0) { leaf = node; node = *top--; }       // a second leaf met while the first was parked
        }
    }
    if (COUNT) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            c_nodes += __shfl_xor_sync(0xffffffffu, c_nodes, d); c_tris += __shfl_xor_sync(0xffffffffu, c_tris, d); c_rays += __shfl_xor_sync(0xffffffffu, c_rays, d);
        }
        if (lane == 0) { atomicAdd(stats, (unsigned long long)c_nodes); atomicAdd(stats + 1, (unsigned long long)c_tris); atomicAdd(stats + 2, (unsigned long long)c_rays); }
    }
}

}  // namespace

// the queue kernel needs leaves of at most 3 triangles (ring capacity) and triangle indices below 2^27 (item = lane << 27 | index)
bool trace_queue_supported(const crt_bvh* bvh) { return bvh->max_leaf <= 3 && bvh->n_refs < ((int64_t)1 << 27) && bvh->q_inflation <= 2.0 && bvh->q_violations == 0; }

crt_status launch_trace_queue(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st)
{
    int per_sm = ctx->trace_blocks_per_sm;
    if (per_sm <= 0) {
        if (stats) CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_queue_kernel<true>, TQ_BLOCK, 0));
        else CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_queue_kernel<false>, TQ_BLOCK, 0));
        if (per_sm < 1) per_sm = 1;
    }
    CRT_CUDA(ctx, cudaMemsetAsync(ctx->d_counter, 0, sizeof(unsigned int), st));
    int64_t want = (n + TQ_BLOCK - 1) / TQ_BLOCK, grid = (int64_t)ctx->n_sms * per_sm;
    if (grid > want) grid = want;
    if (stats) trace_queue_kernel<true><<<(unsigned)grid, TQ_BLOCK, 0, st>>>(bvh->d_qnodes, bvh->qgrid, bvh->d_tris, rays, hits, n, ctx->d_counter, ctx->trace_refill_threshold, ctx->trace_leaf_wait, stats);
    else trace_queue_kernel<false><<<(unsigned)grid, TQ_BLOCK, 0, st>>>(bvh->d_qnodes, bvh->qgrid, bvh->d_tris, rays, hits, n, ctx->d_counter, ctx->trace_refill_threshold, ctx->trace_leaf_wait, nullptr);
    CRT_CHECK_LAUNCH(ctx, "trace_queue");
    return CRT_OK;
}
