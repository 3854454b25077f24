// a5, trace_kernel 8: GROUP-COHERENT traversal -- the sixteen rays of a half-warp walk ONE shared stack (rays of a warp
// that "access the same BVH node" cost one fetch; the paper's kernel shares the sample through shared memory; the method makes
// the K rays of a group leave neighbouring points in one local direction, and with K = 16 a group IS a half-warp in slot order).
// An alternative to the default per-lane kernel of trace.cu, kept with its measurements (profiles/r02h).
//
// One half-warp = one packet of 16 consecutive ray slots:
//   - the packet has ONE current node and ONE stack (shared memory, 8 bytes per entry: node reference + the mask of lanes whose own ray
//     entered that node's box), so a node is fetched once per packet (16 lanes, one address: a broadcast 256-bit load) and there is no
//     per-lane stack traffic and no per-lane leaf bookkeeping;
//   - every lane of the node's mask tests the two child boxes against ITS ray (the 16-bit box test of trace.cu: PRMT decode, six FFMA2);
//     two ballots give the children's lane masks; a child is entered if ANY lane hit it, the one more lanes would enter first goes first,
//     the other is pushed with its mask; a lane outside a node's mask carries a dead predicate through that subtree;
//   - at a leaf every lane of the mask tests the leaf's triangles (uniform addresses again), so there is no parked-leaf vote;
//   - the two half-warps of a warp run in lockstep through a while-while loop (node phase until both hold a leaf or are done, then the
//     leaf phase), so the warp never executes the two packets' code one after the other;
//   - persistent: a packet that is done takes the next 16 slots from the global counter.
// Exactness: the box test is the conservative one of trace.cu and only ever uses a bound >= the lane's best t; the triangle test is the
// bit-exact sequence of crt_device.cuh with the (t, id) rule of D:R10: the hit records are those of the per-lane kernel, whatever the
// order in which the packet visits the leaves.
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

constexpr int SENTINEL = 0x7fffffff;
constexpr int TG_BLOCK = 128;
constexpr int TG_STACK = 64;          // entries per packet: at most one push per level of the tree (the per-lane kernels' bound)
#ifndef CRT_TG_MINB
#define CRT_TG_MINB 8
#endif

CRT_DEV float safe_rcp(float d)
{
    const float eps = 8.673617379884035e-19f;      // 2^-60 (trace.cu: a zero direction component must not give an infinite reciprocal)
    return dvd(1.0f, fabsf(d) > eps ? d : copysignf(eps, d));
}

struct F2 { unsigned long long v; };
CRT_DEV F2 pack2(float lo, float hi) { F2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
CRT_DEV void unpack2(F2 a, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
CRT_DEV F2 fma2(F2 a, F2 b, F2 c) { F2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
CRT_DEV float qbits(unsigned w, unsigned sel)
{
    unsigned f;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(f) : "r"(w), "r"(0x4B000000u), "r"(sel));
    return __uint_as_float(f);
}

// one lane's ray: the triangle test's origin and direction, the constants of the 16-bit box test (trace.cu QRay<false> / QRay2: same
// arithmetic and error budget: origins within 16 scene extents of the scene), the best hit so far
struct GRay {
    V3 o, d;
    F2 sxy, szz, cxy, czz;
    unsigned nx, ny, nz, fx, fy, fz;
    float tmin, best_t; int best_prim;
    CRT_DEV void init(float4 ro, float4 rd, const QGrid& g)
    {
        o = mk(ro.x, ro.y, ro.z); d = mk(rd.x, rd.y, rd.z);
        const float ix = safe_rcp(rd.x), iy = safe_rcp(rd.y), iz = safe_rcp(rd.z);
        const float sx = ix * g.inv_scale[0], sy = iy * g.inv_scale[1], sz = iz * g.inv_scale[2];
        const float px = (ro.x - g.gmin[0]) * g.scale[0], py = (ro.y - g.gmin[1]) * g.scale[1], pz = (ro.z - g.gmin[2]) * g.scale[2];
        const float cx = __fmaf_rn(-8388608.f, sx, -(px * sx)), cy = __fmaf_rn(-8388608.f, sy, -(py * sy)), cz = __fmaf_rn(-8388608.f, sz, -(pz * sz));
        sxy = pack2(sx, sy); szz = pack2(sz, sz); cxy = pack2(cx, cy); czz = pack2(cz, cz);
        nx = rd.x >= 0.f ? 0x7610u : 0x7632u; ny = rd.y >= 0.f ? 0x7610u : 0x7632u; nz = rd.z >= 0.f ? 0x7610u : 0x7632u;
        fx = nx ^ 0x0022u; fy = ny ^ 0x0022u; fz = nz ^ 0x0022u;
        tmin = ro.w; best_t = rd.w; best_prim = -1;
    }
};

// Both child boxes of node idx against this lane's ray (visit_qnode2 of trace.cu): entry distances and hit flags
CRT_DEV void box_pair(const QNode* __restrict__ nodes, int idx, const GRay& q, float& tn0, float& tn1, bool& h0, bool& h1, int& ra, int& rb)
{
    unsigned w0, w1, w2, w3, w4, w5;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(ra), "=r"(rb) : "l"(nodes + idx));
    const float tfar = q.best_t * 1.0000005f;
    float n0x, n0y, f0x, f0y, n1x, n1y, f1x, f1y, n0z, n1z, f0z, f1z;
    unpack2(fma2(pack2(qbits(w0, q.nx), qbits(w1, q.ny)), q.sxy, q.cxy), n0x, n0y);
    unpack2(fma2(pack2(qbits(w0, q.fx), qbits(w1, q.fy)), q.sxy, q.cxy), f0x, f0y);
    unpack2(fma2(pack2(qbits(w3, q.nx), qbits(w4, q.ny)), q.sxy, q.cxy), n1x, n1y);
    unpack2(fma2(pack2(qbits(w3, q.fx), qbits(w4, q.fy)), q.sxy, q.cxy), f1x, f1y);
    unpack2(fma2(pack2(qbits(w2, q.nz), qbits(w5, q.nz)), q.szz, q.czz), n0z, n1z);
    unpack2(fma2(pack2(qbits(w2, q.fz), qbits(w5, q.fz)), q.szz, q.czz), f0z, f1z);
    tn0 = fmaxf(fmaxf(n0x, n0y), fmaxf(n0z, q.tmin));
    const float tf0 = fminf(fminf(f0x, f0y), fminf(f0z, tfar));
    tn1 = fmaxf(fmaxf(n1x, n1y), fmaxf(n1z, q.tmin));
    const float tf1 = fminf(fminf(f1x, f1y), fminf(f1z, tfar));
    h0 = tn0 <= tf0; h1 = tn1 <= tf1;
}

CRT_DEV void store_miss(crt_hit* hits, int64_t i, float tmax)
{
    reinterpret_cast<float4*>(hits)[i] = make_float4(tmax, 0.f, 0.f, __int_as_float(-1));
}

// COUNT: work counters instead of hit records.  stats: [0] lane-level node visits (lanes of the node's mask), [1] lane-level triangle
// tests, [2] active rays, [3] PACKET node visits (one per packet and node: what the warp issues instructions for).
// G: rays per packet, 16 (a half-warp) or 32 (the whole warp).
// The node phase is written without a branch on the packet's state: with G = 16 the warp's two packets execute ONE instruction stream, a
// packet that already holds a leaf (or is done) runs dead visits of node 0 with an empty mask until the other one has a leaf too; all votes
// are full-warp ballots cut to the packet's lanes.  The stack's entry 0 is (SENTINEL, 0), so a pop needs no empty check.
template <bool COUNT, int G>
__global__ void __launch_bounds__(TG_BLOCK, CRT_TG_MINB) trace_group_kernel(const QNode* __restrict__ qnodes, const QGrid grid, const GpuTri* __restrict__ tris,
                                                                            const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n,
                                                                            unsigned int* __restrict__ counter, unsigned long long* __restrict__ stats)
{
    __shared__ uint2 s_stack[TG_BLOCK / G][TG_STACK];
    const unsigned lane = threadIdx.x & 31u, hbase = G == 16 ? (lane & 16u) : 0u, gmask = G == 16 ? (0xffffu << hbase) : 0xffffffffu, lbit = 1u << lane;
    uint2* const stk = s_stack[threadIdx.x / G];
    if (lane == hbase) stk[0] = make_uint2((unsigned)SENTINEL, 0u);
    __syncwarp();
    // packet state, replicated in the registers of its lanes
    int node = SENTINEL; unsigned am = 0u;      // am: lanes (warp bit positions) whose ray is inside the current node's box
    uint2* top = stk;                            // the top entry
    bool exhausted = false;
    int ray_idx = -1;
    GRay q;
    unsigned c_lane_nodes = 0, c_tris = 0, c_rays = 0, c_packet_nodes = 0;

    for (;;) {
        // ---- a packet that is done retires its rays and takes the next G slots (one atomic per packet)
        if (node == SENTINEL && !exhausted) {
            for (;;) {
                if (!COUNT && ray_idx >= 0 && q.best_prim < 0) store_miss(hits, ray_idx, q.best_t);
                ray_idx = -1;
                unsigned base = 0;
                if (lane == hbase) base = atomicAdd(counter, (unsigned)G);
                base = __shfl_sync(gmask, base, hbase);
                if ((int64_t)base >= n) { exhausted = true; break; }
                const int64_t i = (int64_t)base + (lane - hbase);
                bool alive = false;
                if (i < n) {
                    const float4* rp = reinterpret_cast<const float4*>(rays + i);
                    const float4 rd = __ldg(rp + 1);
                    if (rd.w < 0.f) { if (!COUNT) store_miss(hits, i, rd.w); }      // inactive slot: a miss, nothing to traverse
                    else { q.init(__ldg(rp), rd, grid); ray_idx = (int)i; alive = true; if (COUNT) ++c_rays; }
                }
                am = __ballot_sync(gmask, alive) & gmask;
                if (am) { node = 0; top = stk; break; }
            }
        }
        if (__all_sync(0xffffffffu, node == SENTINEL)) break;        // every packet done and the ray list exhausted

        for (;;) {
            // ---- node phase: until each packet of the warp holds a leaf or is done
            while (__any_sync(0xffffffffu, (unsigned)node < (unsigned)SENTINEL)) {
                const bool live = (unsigned)node < (unsigned)SENTINEL;           // uniform in the packet
                float tn0, tn1; bool h0, h1; int ra, rb;
                box_pair(qnodes, live ? node : 0, q, tn0, tn1, h0, h1, ra, rb);
                const bool in = live && (am & lbit) != 0u;
                h0 = h0 && in; h1 = h1 && in;
                if (COUNT) { c_lane_nodes += in ? 1u : 0u; if (live && lane == hbase) ++c_packet_nodes; }
                const unsigned m0 = __ballot_sync(0xffffffffu, h0) & gmask, m1 = __ballot_sync(0xffffffffu, h1) & gmask;
                const unsigned p1 = __ballot_sync(0xffffffffu, h1 && (!h0 || tn1 < tn0)) & gmask;      // lanes that would enter child 1 first
                const unsigned any = m0 | m1;
                const bool second = (p1 & (any & (0u - any))) != 0u;             // the order the packet's first hitting lane wants
                if (live) {
                    if (m0 && m1) *++top = second ? make_uint2((unsigned)ra, m0) : make_uint2((unsigned)rb, m1);     // every lane writes the same entry
                    node = second ? rb : ra; am = second ? m1 : m0;
                    if (!any) { const uint2 e = *top--; node = (int)e.x; am = e.y; }
                }
            }
            // ---- leaf phase: the lanes of the mask test the leaf's triangles (D:R10: lower primitive id wins at equal t)
            if (node < 0) {
                const int leaf = ~node, first = leaf >> 3, cnt = (leaf & 7) + 1;
                const bool in = (am & lbit) != 0u;
                for (int j = 0; j < cnt; ++j) {
                    const char* tp = reinterpret_cast<const char*>(tris + first + j);
                    float a0, a1, a2, a3, b0, b1, b2, b3; float4 c;
                    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                                 : "=f"(a0), "=f"(a1), "=f"(a2), "=f"(a3), "=f"(b0), "=f"(b1), "=f"(b2), "=f"(b3) : "l"(tp));
                    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(c.x), "=f"(c.y), "=f"(c.z), "=f"(c.w) : "l"(tp + 32));
                    float t, u, v;
                    if (in) {
                        if (COUNT) ++c_tris;
                        if (tri_test(mk(a0, a1, a2), mk(b0, b1, b2), mk(c.x, c.y, c.z), q.o, q.d, q.tmin, __int_as_float(0x7f800000), t, u, v)) {
                            const int prim = __float_as_int(a3);
                            if (t < q.best_t || (t == q.best_t && q.best_prim >= 0 && prim < q.best_prim)) {
                                q.best_t = t; q.best_prim = prim;
                                if (!COUNT) reinterpret_cast<float4*>(hits)[ray_idx] = make_float4(t, u, v, __int_as_float(prim));
                            }
                        }
                    }
                }
                const uint2 e = *top--; node = (int)e.x; am = e.y;
            }
            // a packet is done: refill it; or leave, if nothing is left (a packet that is done for good just waits for the other one)
            if (__any_sync(0xffffffffu, node == SENTINEL && !exhausted) || __all_sync(0xffffffffu, node == SENTINEL)) break;
        }
    }
    if (COUNT) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            c_lane_nodes += __shfl_xor_sync(0xffffffffu, c_lane_nodes, d); c_tris += __shfl_xor_sync(0xffffffffu, c_tris, d);
            c_rays += __shfl_xor_sync(0xffffffffu, c_rays, d); c_packet_nodes += __shfl_xor_sync(0xffffffffu, c_packet_nodes, d);
        }
        if (lane == 0) {
            atomicAdd(stats, (unsigned long long)c_lane_nodes); atomicAdd(stats + 1, (unsigned long long)c_tris);
            atomicAdd(stats + 2, (unsigned long long)c_rays); atomicAdd(stats + 3, (unsigned long long)c_packet_nodes);
        }
    }
}

template <bool COUNT, int G>
crt_status launch_group(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st, unsigned int* counter)
{
    int per_sm = ctx->trace_blocks_per_sm;
    if (per_sm <= 0) {
        CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_group_kernel<COUNT, G>, TG_BLOCK, 0));
        if (per_sm < 1) per_sm = 1;
    }
    if (!counter) counter = ctx->d_counter;
    CRT_CUDA(ctx, cudaMemsetAsync(counter, 0, sizeof(unsigned int), st));
    int64_t want = (n + TG_BLOCK - 1) / TG_BLOCK, grid = (int64_t)ctx->n_sms * per_sm;
    if (grid > want) grid = want;
    trace_group_kernel<COUNT, G><<<(unsigned)grid, TG_BLOCK, 0, st>>>(bvh->d_qnodes, bvh->qgrid, bvh->d_tris, rays, hits, n, counter, stats);
    CRT_CHECK_LAUNCH(ctx, "trace_group");
    return CRT_OK;
}

}  // namespace

// the 16-bit layout with its own check clean (as the default kernel requires)
bool trace_group_supported(const crt_bvh* bvh) { return bvh->q_inflation <= 2.0 && bvh->q_violations == 0 && bvh->d_qnodes != nullptr; }

crt_status launch_trace_group(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st, unsigned int* counter, int group)
{
    if (n == 0) return CRT_OK;
    if (group == 32) return stats ? launch_group<true, 32>(ctx, bvh, rays, n, hits, stats, st, counter) : launch_group<false, 32>(ctx, bvh, rays, n, hits, stats, st, counter);
    return stats ? launch_group<true, 16>(ctx, bvh, rays, n, hits, stats, st, counter) : launch_group<false, 16>(ctx, bvh, rays, n, hits, stats, st, counter);
}
