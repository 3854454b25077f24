// a1 + a5: primary-ray generation and BVH traversal kernels ("Each thread searches the acceleration
// structure to find the leaf nodes that the ray passes through"; this is "the most time-consuming segment").
//
// B200 design:
//  - stack-based traversal of a binary BVH.  Default layout (trace_kernel 3): 32-byte nodes holding both children's boxes as
//    16-bit planes on a scene grid, fetched with ONE 256-bit load (ld.global.nc.v8 -> LDG.E.ENL2.256) on the read-only path and
//    decoded by one PRMT per plane that also selects the near or far plane by the ray's direction sign (struct QRay below); the
//    twelve plane distances of a visit are six packed FFMA2 (fma.rn.f32x2, new on sm_100: one issue slot for two fused multiply-adds);
//    the fp32 form (64-byte nodes, two 256-bit loads) is trace_kernel 0 / 1; leaf triangles are 64-byte records (v0|id, e1, e2);
//  - with the 16-bit nodes the kernel is issue- and latency-bound, not bandwidth-bound (profiles/r01f): what matters is how many
//    lanes of a warp do useful work and how many warps are resident (8 blocks of 128 threads per SM at 64 registers for camera rays, 9 at 56 for secondary rays).
//    trace_dyn_kernel is a persistent-warp kernel: the grid fills the 148 SMs once; a lane whose ray has terminated takes
//    the next ray from a global counter (one atomicAdd per warp, ballot + popc give each idle lane its index) as soon as
//    fewer than `refill_threshold` lanes of its warp are still traversing, so rays enter a warp in slot order -- the order
//    the generator made coherent (group-major) -- and divergent stragglers do not idle 31 lanes;
//  - inner-node and leaf phases are separated (while-while) and a lane that reaches a leaf postpones it and keeps
//    descending until (nearly) every converged lane has one, so the triangle tests of a warp run together; the vote that decides
//    it is taken every CRT_VISITS_PER_VOTE visits, push and pop are predicated, the stack is addressed through a pointer;
//  - inactive slots (dead paths, out-of-image slots) are skipped at fetch time and cost one 16-byte load;
//  - no tensor cores: traversal is not a dense contraction.
// Exactness: the triangle test is the bit-exact fp32 formula of crt_device.cuh; box tests are conservative (boxes padded at
// build time by 2^-17 of the largest coordinate, 16-bit planes rounded outward plus one grid step, far side inflated, subtree
// skipped only if its entry distance is strictly beyond the best t), so the result equals the all-triangles definition with ties -> lowest primitive id (D:R10), whatever
// the order in which leaves are visited.
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

constexpr int STACK_SIZE = 64;
constexpr int SENTINEL = 0x7fffffff;
constexpr int TRACE_BLOCK = 128;
// resident blocks per SM the persistent kernel is compiled for: fp32 nodes 9 (<= 56 registers), 16-bit nodes 8 (<= 64
// registers; measured 1.5-3 % faster than 9 with this layout, profiles/r01f)
#define CRT_TRACE_MINB(QN) ((QN) ? 8 : 9)      // QN: 0 fp32 nodes; 1 16-bit nodes (default); 2 16-bit nodes with the any-origin box test; 3 as 1 with the
                                               // tolerance-only triangle test (trace_exact = 0); 4 as 1 with the top of the tree staged in shared memory (experiment); 5 the 4-wide form of the 16-bit nodes
constexpr int TREELET_NODES = 512;             // QN 4: nodes 0 .. 511 (the top levels: crt_bvh_flatten numbers them breadth-first) = 16 KB of shared memory per block
#ifndef CRT_VISITS_PER_VOTE
#define CRT_VISITS_PER_VOTE 6   // inner-node visits between two leaf-wait votes of a warp (3 until the trees of profiles/r02k / r02o: re-measured there, 5-8 are 1.5-2.7 % faster than 3)
#endif

CRT_DEV unsigned long long globaltimer_ns() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

struct ChildRegs { float min_x, max_x, min_y, max_y, min_z, max_z; int ref; };

// one 32-byte child record through the non-coherent path (LDG.E.ENL2.256.CONSTANT)
CRT_DEV ChildRegs load_child(const char* p)
{
    ChildRegs c; float a6, a7;
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(c.min_x), "=f"(c.max_x), "=f"(c.min_y), "=f"(c.max_y), "=f"(c.min_z), "=f"(c.max_z), "=f"(a6), "=f"(a7) : "l"(p));
    c.ref = __float_as_int(a6);
    return c;
}
struct NodeRegs { ChildRegs a, b; };
CRT_DEV NodeRegs load_node(const GpuNode* __restrict__ nodes, int idx)
{
    const char* p = reinterpret_cast<const char*>(nodes + idx);
    NodeRegs n; n.a = load_child(p); n.b = load_child(p + 32);
    return n;
}

// a ray record is read once: it must not take an L1 line from the nodes (the kernel lives on the L1: profiles/r02a)
CRT_DEV float4 ld_stream(const float4* p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

struct Hit { float t; int prim; };     // u, v go straight to the hit record when a nearer hit is found (two registers fewer)

// 1/d for the box test only.  A direction component of (nearly) zero is replaced by +-2^-60: with an infinite reciprocal the
// two plane distances of an axis can come out as -inf and NaN, and min/max then keep the -inf for BOTH the entry and the
// exit distance, which rejects boxes the ray is inside of.  With a huge finite reciprocal the distances are huge finite
// numbers of the right signs; their cancellation error is an ulp of the origin, far inside the boxes' padding.
CRT_DEV float safe_rcp(float d)
{
    const float eps = 8.673617379884035e-19f;      // 2^-60
    return dvd(1.0f, fabsf(d) > eps ? d : copysignf(eps, d));
}

// Per-ray traversal state.  The slab test is t = b * (1/d) - o * (1/d) as one FMA per plane: its rounding error is a few
// ulps of |o/d|, which the build-time padding of the boxes (>= 128 of those ulps for origins inside the padded scene box,
// DESIGN.md section 5) and the inflated far side absorb; it only ever decides which subtrees are visited.
struct RayState {
    V3 o, d;
    float idx, idy, idz, ox, oy, oz;     // 1/d and -o/d
    float tmin;                           // best.t starts at the ray's tmax, so "t < tmax" is "t < best.t" until a hit exists
    Hit best;
    // prune bound: best t so far, inflated (recomputed per visit: one FMUL instead of a register)
    CRT_DEV float tfar() const { return best.t * 1.0000005f; }
    CRT_DEV void init(float4 ro, float4 rd)
    {
        o = mk(ro.x, ro.y, ro.z); d = mk(rd.x, rd.y, rd.z);
        idx = safe_rcp(d.x); idy = safe_rcp(d.y); idz = safe_rcp(d.z);
        ox = -o.x * idx; oy = -o.y * idy; oz = -o.z * idz;
        tmin = ro.w;
        best.t = rd.w; best.prim = -1;
    }
};

// Tests both children of `n`; returns the next node reference (nearer child, other child pushed) or pops the stack.
CRT_DEV int visit_node(const NodeRegs& n, const RayState& r, int*& top)
{
    // every distance is finite (safe_rcp); a NaN could only come from non-finite ray data, and fminf/fmaxf drop NaN operands
    const float ax0 = __fmaf_rn(n.a.min_x, r.idx, r.ox), ax1 = __fmaf_rn(n.a.max_x, r.idx, r.ox);
    const float ay0 = __fmaf_rn(n.a.min_y, r.idy, r.oy), ay1 = __fmaf_rn(n.a.max_y, r.idy, r.oy);
    const float az0 = __fmaf_rn(n.a.min_z, r.idz, r.oz), az1 = __fmaf_rn(n.a.max_z, r.idz, r.oz);
    const float bx0 = __fmaf_rn(n.b.min_x, r.idx, r.ox), bx1 = __fmaf_rn(n.b.max_x, r.idx, r.ox);
    const float by0 = __fmaf_rn(n.b.min_y, r.idy, r.oy), by1 = __fmaf_rn(n.b.max_y, r.idy, r.oy);
    const float bz0 = __fmaf_rn(n.b.min_z, r.idz, r.oz), bz1 = __fmaf_rn(n.b.max_z, r.idz, r.oz);
    const float tfar = r.tfar();
    const float tn0 = fmaxf(fmaxf(fminf(ax0, ax1), fminf(ay0, ay1)), fmaxf(fminf(az0, az1), r.tmin));
    const float tf0 = fminf(fminf(fmaxf(ax0, ax1), fmaxf(ay0, ay1)), fminf(fmaxf(az0, az1), tfar));
    const float tn1 = fmaxf(fmaxf(fminf(bx0, bx1), fminf(by0, by1)), fmaxf(fminf(bz0, bz1), r.tmin));
    const float tf1 = fminf(fminf(fmaxf(bx0, bx1), fmaxf(by0, by1)), fminf(fmaxf(bz0, bz1), tfar));
    const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
    if (h0 && h1) {
        const bool swap = tn1 < tn0;
        *++top = swap ? n.a.ref : n.b.ref;
        return swap ? n.b.ref : n.a.ref;
    }
    if (h0) return n.a.ref;
    if (h1) return n.b.ref;
    return *top--;
}

// ---- 16-bit nodes (QNode, 32 bytes, ONE 256-bit load; crt_internal.h, bvh_build.cpp: crt_bvh_quantise) -----------------
// Per-ray constants of the box test in grid units.  A plane q (16 bits) becomes the float 2^23 + q with one PRMT (the two
// plane bytes under the exponent byte of 0x4B000000) and its distance is one FMA: t = (2^23 + q) * s + c, c = -(o' + 2^23) * s
// (o' = ray origin in grid units).
// The PRMT selector picks the min or the max plane by the sign of the ray direction, so near and far distances come out
// directly and no per-axis min/max is needed: 12 PRMT + 12 FFMA + 8 FMNMX per node against 12 FFMA + 20 FMNMX for fp32 nodes.
template <bool SAFE>
struct QRay {
    float sx, sy, sz;                     // 1 / (d * scale): distance per grid step
    float cx, cy, cz;                     // -(o' + 2^23) * s (SAFE: rounded down and moved outward, for near planes)
    float fcx, fcy, fcz;                  // SAFE only: the same rounded up and moved outward, for far planes
    unsigned nx, ny, nz, fx, fy, fz;      // PRMT selectors of the near / far plane
    // Error budget of t = (2^23 + q) * s + c against the exact (q - o') * s, in grid steps of position: c is rounded to an ulp
    // of 2^23 * s, i.e. at most HALF a step; o' (two roundings), s (three), the product o' * s and the final FMA add at most
    // 6 * 2^-24 * |o'| + 2^-7 step.  The stored planes are moved ONE step outward (crt_bvh_quantise), so the test is
    // conservative while 0.5 + 6 * 2^-24 * |o'| <= 1, i.e. |o'| <= 1.4 M steps; the stated contract (include/crt.h) is ray
    // origins within 16 scene extents of the scene (0.9 step; tests/test_abi.py re-enacts this arithmetic).  The fp32-node
    // kernel's own limit is about 128 extents.  Rounding c in opposite directions for near and far planes with a per-ray margin
    // lifts the limit but was measured 3-4 % slower (six constant registers instead of three defeat the operand reuse of the
    // FFMA pairs; profiles/r01f).
    CRT_DEV void init(const RayState& r, const QGrid& g)
    {
        sx = r.idx * g.inv_scale[0]; sy = r.idy * g.inv_scale[1]; sz = r.idz * g.inv_scale[2];
        const float px = (r.o.x - g.gmin[0]) * g.scale[0], py = (r.o.y - g.gmin[1]) * g.scale[1], pz = (r.o.z - g.gmin[2]) * g.scale[2];
        if (SAFE) {
            // trace_kernel 4: conservative for ANY ray origin.  c is rounded down for near planes and up for far planes after being
            // moved outward by m = (|o'| + 65536) * 2^-19 steps per axis, which exceeds the relative errors of o', s and the FMA
            // (6 * 2^-24 (|o'| + 65536)); costs three more registers and 3-4 % of the speed (profiles/r01f).
            const float k = 1.9073486328125e-6f;        // 2^-19
            const float mx = __fmul_ru(__fmul_ru(__fadd_ru(fabsf(px), 65536.f), k), fabsf(sx));
            const float my = __fmul_ru(__fmul_ru(__fadd_ru(fabsf(py), 65536.f), k), fabsf(sy));
            const float mz = __fmul_ru(__fmul_ru(__fadd_ru(fabsf(pz), 65536.f), k), fabsf(sz));
            cx = __fmaf_rd(-8388608.f, sx, __fmaf_rd(-px, sx, -mx)); fcx = __fmaf_ru(-8388608.f, sx, __fmaf_ru(-px, sx, mx));
            cy = __fmaf_rd(-8388608.f, sy, __fmaf_rd(-py, sy, -my)); fcy = __fmaf_ru(-8388608.f, sy, __fmaf_ru(-py, sy, my));
            cz = __fmaf_rd(-8388608.f, sz, __fmaf_rd(-pz, sz, -mz)); fcz = __fmaf_ru(-8388608.f, sz, __fmaf_ru(-pz, sz, mz));
        } else {
            cx = __fmaf_rn(-8388608.f, sx, -(px * sx)); cy = __fmaf_rn(-8388608.f, sy, -(py * sy)); cz = __fmaf_rn(-8388608.f, sz, -(pz * sz));
        }
        nx = r.d.x >= 0.f ? 0x7610u : 0x7632u; ny = r.d.y >= 0.f ? 0x7610u : 0x7632u; nz = r.d.z >= 0.f ? 0x7610u : 0x7632u;
        fx = nx ^ 0x0022u; fy = ny ^ 0x0022u; fz = nz ^ 0x0022u;
    }
};
CRT_DEV float qplane(unsigned w, unsigned sel, float s, float c)
{
    unsigned f;      // prmt directly: __byte_perm would mask the selector with 0x7777 at every use
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(f) : "r"(w), "r"(0x4B000000u), "r"(sel));
    return __fmaf_rn(__uint_as_float(f), s, c);
}
// a direction component of zero: s is huge but finite (safe_rcp), both distances of that axis are huge with the right signs
template <bool SAFE>
CRT_DEV int visit_qnode(const QNode* __restrict__ nodes, int idx, const RayState& r, const QRay<SAFE>& q, int*& top)
{
    unsigned w0, w1, w2, w3, w4, w5; int ra, rb;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(ra), "=r"(rb) : "l"(nodes + idx));
    const float tfar = r.tfar();
    const float tn0 = fmaxf(fmaxf(qplane(w0, q.nx, q.sx, q.cx), qplane(w1, q.ny, q.sy, q.cy)), fmaxf(qplane(w2, q.nz, q.sz, q.cz), r.tmin));
    const float tf0 = fminf(fminf(qplane(w0, q.fx, q.sx, SAFE ? q.fcx : q.cx), qplane(w1, q.fy, q.sy, SAFE ? q.fcy : q.cy)), fminf(qplane(w2, q.fz, q.sz, SAFE ? q.fcz : q.cz), tfar));
    const float tn1 = fmaxf(fmaxf(qplane(w3, q.nx, q.sx, q.cx), qplane(w4, q.ny, q.sy, q.cy)), fmaxf(qplane(w5, q.nz, q.sz, q.cz), r.tmin));
    const float tf1 = fminf(fminf(qplane(w3, q.fx, q.sx, SAFE ? q.fcx : q.cx), qplane(w4, q.fy, q.sy, SAFE ? q.fcy : q.cy)), fminf(qplane(w5, q.fz, q.sz, SAFE ? q.fcz : q.cz), tfar));
    // next node without a three-way branch: the nearer hit child (the farther one pushed), else the top of the stack
    const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
    const bool second = h1 && (!h0 || tn1 < tn0);          // child 1 is the one to enter
    int next = second ? rb : ra;
    if (h0 && h1) *++top = second ? ra : rb;     // (an L1 prefetch of the pushed node was measured 5 % slower)
    if (!(h0 || h1)) next = *top--;
    return next;
}

// The same visit with the twelve plane distances computed by SIX packed FFMA2 (fma.rn.f32x2, new on sm_100): the kernel is bound
// by instruction issue, and a packed instruction is one issue slot for two fused multiply-adds.  Each half of a packed operation is
// the same IEEE fma as the scalar one, so the distances, and hence the visit order, are bit-identical to visit_qnode<false>.
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
struct QRay2 {
    F2 sxy, szz, cxy, czz;                // (sx, sy), (sz, sz), (cx, cy), (cz, cz)
    unsigned nx, ny, nz, fx, fy, fz;
    template <bool SAFE> CRT_DEV void init(const QRay<SAFE>& q)
    {
        sxy = pack2(q.sx, q.sy); szz = pack2(q.sz, q.sz); cxy = pack2(q.cx, q.cy); czz = pack2(q.cz, q.cz);
        nx = q.nx; ny = q.ny; nz = q.nz; fx = q.fx; fy = q.fy; fz = q.fz;
    }
};
template <bool TREELET>
CRT_DEV int visit_qnode2(const QNode* __restrict__ nodes, const uint4* s_treelet, int idx, const RayState& r, const QRay2& q, int*& top)
{
    unsigned w0, w1, w2, w3, w4, w5; int ra, rb;
    if (TREELET && idx < TREELET_NODES) {
        const uint4 a = s_treelet[2 * idx], b = s_treelet[2 * idx + 1];
        w0 = a.x; w1 = a.y; w2 = a.z; w3 = a.w; w4 = b.x; w5 = b.y; ra = (int)b.z; rb = (int)b.w;
    } else
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(ra), "=r"(rb) : "l"(nodes + idx));
    const float tfar = r.tfar();
    float n0x, n0y, f0x, f0y, n1x, n1y, f1x, f1y, n0z, n1z, f0z, f1z;
    unpack2(fma2(pack2(qbits(w0, q.nx), qbits(w1, q.ny)), q.sxy, q.cxy), n0x, n0y);
    unpack2(fma2(pack2(qbits(w0, q.fx), qbits(w1, q.fy)), q.sxy, q.cxy), f0x, f0y);
    unpack2(fma2(pack2(qbits(w3, q.nx), qbits(w4, q.ny)), q.sxy, q.cxy), n1x, n1y);
    unpack2(fma2(pack2(qbits(w3, q.fx), qbits(w4, q.fy)), q.sxy, q.cxy), f1x, f1y);
    unpack2(fma2(pack2(qbits(w2, q.nz), qbits(w5, q.nz)), q.szz, q.czz), n0z, n1z);
    unpack2(fma2(pack2(qbits(w2, q.fz), qbits(w5, q.fz)), q.szz, q.czz), f0z, f1z);
    const float tn0 = fmaxf(fmaxf(n0x, n0y), fmaxf(n0z, r.tmin));
    const float tf0 = fminf(fminf(f0x, f0y), fminf(f0z, tfar));
    const float tn1 = fmaxf(fmaxf(n1x, n1y), fmaxf(n1z, r.tmin));
    const float tf1 = fminf(fminf(f1x, f1y), fminf(f1z, tfar));
    const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
    const bool second = h1 && (!h0 || tn1 < tn0);
    int next = second ? rb : ra;
    if (h0 && h1) *++top = second ? ra : rb;
    if (!(h0 || h1)) next = *top--;
    return next;
}

// ---- 4-wide visit (QN 5, trace_kernel 7): node idx = records 2 idx and 2 idx + 1 of the 4-wide array (crt_bvh_collapse4), fetched with two INDEPENDENT
// 256-bit loads; four box tests by twelve FFMA2.  Order: inside a pair the nearer hit child first; the pair whose nearest hit is nearer first; the other
// hit children are pushed so that they pop in that order (an approximate front-to-back order: the result does not depend on it, D:R10).
CRT_DEV void q4_pair(const QNode* __restrict__ rec, const RayState& r, const QRay2& q, float tfar, float& tn_a, float& tn_b, bool& ha, bool& hb, int& ra, int& rb)
{
    unsigned w0, w1, w2, w3, w4, w5;
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(ra), "=r"(rb) : "l"(rec));
    float n0x, n0y, f0x, f0y, n1x, n1y, f1x, f1y, n0z, n1z, f0z, f1z;
    unpack2(fma2(pack2(qbits(w0, q.nx), qbits(w1, q.ny)), q.sxy, q.cxy), n0x, n0y);
    unpack2(fma2(pack2(qbits(w0, q.fx), qbits(w1, q.fy)), q.sxy, q.cxy), f0x, f0y);
    unpack2(fma2(pack2(qbits(w3, q.nx), qbits(w4, q.ny)), q.sxy, q.cxy), n1x, n1y);
    unpack2(fma2(pack2(qbits(w3, q.fx), qbits(w4, q.fy)), q.sxy, q.cxy), f1x, f1y);
    unpack2(fma2(pack2(qbits(w2, q.nz), qbits(w5, q.nz)), q.szz, q.czz), n0z, n1z);
    unpack2(fma2(pack2(qbits(w2, q.fz), qbits(w5, q.fz)), q.szz, q.czz), f0z, f1z);
    tn_a = fmaxf(fmaxf(n0x, n0y), fmaxf(n0z, r.tmin));
    const float tf_a = fminf(fminf(f0x, f0y), fminf(f0z, tfar));
    tn_b = fmaxf(fmaxf(n1x, n1y), fmaxf(n1z, r.tmin));
    const float tf_b = fminf(fminf(f1x, f1y), fminf(f1z, tfar));
    ha = tn_a <= tf_a; hb = tn_b <= tf_b;
}
CRT_DEV int visit_q4node(const QNode* __restrict__ q4, int idx, const RayState& r, const QRay2& q, int*& top)
{
    const float tfar = r.tfar();
    float ta0, ta1, tb0, tb1; bool ha0, ha1, hb0, hb1; int ra0, ra1, rb0, rb1;
    q4_pair(q4 + 2 * idx, r, q, tfar, ta0, ta1, ha0, ha1, ra0, ra1);
    q4_pair(q4 + 2 * idx + 1, r, q, tfar, tb0, tb1, hb0, hb1, rb0, rb1);
    // inside each pair: near / far child
    const bool sa = ha1 && (!ha0 || ta1 < ta0), sb = hb1 && (!hb0 || tb1 < tb0);
    const int an = sa ? ra1 : ra0, af = sa ? ra0 : ra1, bn = sb ? rb1 : rb0, bf = sb ? rb0 : rb1;
    const bool a_any = ha0 || ha1, a_both = ha0 && ha1, b_any = hb0 || hb1, b_both = hb0 && hb1;
    const float ta = sa ? ta1 : ta0, tb = sb ? tb1 : tb0;          // entry distance of each pair's near child (meaningful when the pair has a hit)
    const bool b_first = b_any && (!a_any || tb < ta);
    const int c1 = b_first ? bn : an, c2 = b_first ? bf : af, c3 = b_first ? an : bn, c4 = b_first ? af : bf;
    const bool f1 = a_any || b_any, f2 = b_first ? b_both : a_both, f3 = b_first ? a_any : b_any, f4 = b_first ? a_both : b_both;
    if (f4) *++top = c4;
    if (f3) *++top = c3;
    if (f2) *++top = c2;
    int next = c1;
    if (!f1) next = *top--;
    return next;
}

// Tests the triangles of a leaf reference (D:R10 tie-break: lower primitive id wins at equal t).
// SPLIT (tail splitting, see trace_dyn_kernel): a lane that works on a subtree of ANOTHER lane's ray (ray_idx <= -2) keeps u, v in aux[0..1]
template <bool COUNT, bool FAST = false, bool SPLIT = false>
CRT_DEV void visit_leaf(const GpuTri* __restrict__ tris, int ref, RayState& r, unsigned& n_tris, crt_hit* __restrict__ hits, int ray_idx, int* aux = nullptr)
{
    const int leaf = ~ref;
    const int first = leaf >> 3, cnt = (leaf & 7) + 1;
    for (int j = 0; j < cnt; ++j) {
        // 64-byte record = two 256-bit loads: v0 | prim | e1 | 0, e2 | 0 | pad
        const char* tp = reinterpret_cast<const char*>(tris + first + j);
        const ChildRegs q0 = load_child(tp); float4 c;
        asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(c.x), "=f"(c.y), "=f"(c.z), "=f"(c.w) : "l"(tp + 32));
        const float4 a = make_float4(q0.min_x, q0.max_x, q0.min_y, q0.max_y), b = make_float4(q0.min_z, q0.max_z, __int_as_float(q0.ref), 0.f);
        float t, u, v;
        if (COUNT) ++n_tris;
        if (FAST ? tri_test_fast(mk(a.x, a.y, a.z), mk(b.x, b.y, b.z), mk(c.x, c.y, c.z), r.o, r.d, r.tmin, __int_as_float(0x7f800000), t, u, v)
                 : tri_test(mk(a.x, a.y, a.z), mk(b.x, b.y, b.z), mk(c.x, c.y, c.z), r.o, r.d, r.tmin, __int_as_float(0x7f800000), t, u, v)) {
            // t < tmax and the (t, id) rule in one: best.t is the ray's tmax until a hit exists, the best t afterwards
            const int prim = __float_as_int(a.w);
            if (t < r.best.t || (t == r.best.t && r.best.prim >= 0 && prim < r.best.prim)) {
                r.best.t = t; r.best.prim = prim;
                if (!COUNT) {
                    if (!SPLIT || ray_idx >= 0) reinterpret_cast<float4*>(hits)[ray_idx] = make_float4(t, u, v, __int_as_float(prim));
                    else { aux[0] = __float_as_int(u); aux[1] = __float_as_int(v); }
                }
            }
        }
    }
}

// record of a ray that hit nothing: t = the ray's tmax, prim = -1
CRT_DEV void store_miss(crt_hit* hits, int64_t i, float tmax)
{
    reinterpret_cast<float4*>(hits)[i] = make_float4(tmax, 0.f, 0.f, __int_as_float(-1));
}

// variant 0: one thread per ray, plain while-while loop (kept as the simple cross-check of the persistent kernel)
__global__ void __launch_bounds__(TRACE_BLOCK) trace_flat_kernel(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris,
                                                                 const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4* rp = reinterpret_cast<const float4*>(rays + i);
    const float4 ro = __ldg(rp), rd = __ldg(rp + 1);
    RayState r; r.init(ro, rd);
    if (rd.w >= 0.f) {
        int stack[STACK_SIZE]; int* top = stack; stack[0] = SENTINEL;      // top: pointer to the top entry (no index-to-address LEA per push/pop)
        int node = 0; unsigned dummy = 0;
        while (node != SENTINEL) {
            while ((unsigned)node < (unsigned)SENTINEL) node = visit_node(load_node(nodes, node), r, top);
            while (node < 0) { visit_leaf<false>(tris, node, r, dummy, hits, (int)i); node = *top--; }
        }
    }
    if (r.best.prim < 0) store_miss(hits, i, rd.w);
}

// variant 1 (default): persistent warps, per-lane dynamic ray fetch, postponed leaves.  COUNT adds work counters.
// 9 blocks/SM (<= 56 registers, 36 warps): measured faster than 8 blocks at 64 registers and 10 blocks at 48 (profiles/).
// SPLIT (trace_tail_split, default on): once the ray list is exhausted, the tail of the launch is a few long rays, each a serial chain of
// dependent node fetches on one lane while the other lanes of its warp idle (measured: the last 1 % of the warps end 45 us after the 99th
// percentile, 0.3 us per visit; profiles/r02i).  In that phase an idle lane takes over the BOTTOM entry of a busy lane's stack (the
// earliest pushed = largest postponed subtree) together with a copy of its ray and traverses it concurrently.  The closest hit with the
// (t, id) rule of D:R10 does not depend on who finds it or in which order: a helper keeps its candidate in registers (u, v in local
// memory) and, when its subtree is done, writes it to the ray's record if it beats what the record holds (the record is initialised when
// the ray first gives work away; all lanes of a ray are in ONE warp and deliveries happen at a warp-wide point of the loop, so there is no
// concurrent writer); the lanes still working on that ray adopt the delivered t as their pruning bound.
// TIMELINE (crt_trace_timeline): the same traversal with four marks per warp written to `stats` at the end: [0] start, [1] the moment the warp
// first saw the ray list exhausted, [2] end (globaltimer, ns), [3] the largest number of node visits one of its lanes made after [1].
// MINB: resident blocks per SM the instantiation is compiled for.  The default kernel exists twice: 8 blocks (64 registers) for camera rays and 9 blocks (56
// registers, 16 bytes of spill outside the node loop) for secondary rays, whose divergent gathers gain more from the ninth block's warps than they lose to its
// share of the L1 (interior secondary rays -1.2 to -2.5 %; camera rays +2 % if they took it too: profiles/r02a).
template <bool COUNT, int QN, bool SPLIT, bool TIMELINE = false, int MINB = CRT_TRACE_MINB(QN)>
__global__ void __launch_bounds__(TRACE_BLOCK, MINB) trace_dyn_kernel(const GpuNode* __restrict__ nodes, const QNode* __restrict__ qnodes, const QGrid grid, const GpuTri* __restrict__ tris,
                                                                const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n,
                                                                unsigned int* __restrict__ counter, int refill_threshold, int leaf_wait,
                                                                unsigned long long* __restrict__ stats, int n_qnodes)
{
    const unsigned lane = threadIdx.x & 31u;
    extern __shared__ uint4 s_treelet[];
    if (QN == 4) {       // experiment (north_star: "a node-prefetch stage in shared memory"): the top of the tree, once per block
        for (int i = threadIdx.x; i < 2 * TREELET_NODES; i += blockDim.x) s_treelet[i] = i < 2 * n_qnodes ? reinterpret_cast<const uint4*>(qnodes)[i] : make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();
    }
    int stack[STACK_SIZE + 4]; int* top = stack; stack[0] = SENTINEL;      // top: pointer to the top entry (no index-to-address LEA per push/pop)
    int* const aux = stack + STACK_SIZE;      // SPLIT: [0], [1] = u, v of a helper's candidate; [2] = bot: stack[bot] is this lane's sentinel (entries below were given away); [3] = the hit id a helper started from
    if (SPLIT) aux[2] = 0;
    int node = SENTINEL, leaf = 0;      // leaf: postponed leaf reference (< 0) or 0 = none
    int ray_idx = -1;                   // SPLIT: <= -2 = helper of ray -2 - ray_idx
    bool exhausted = false, tail = false;
    RayState r; QRay<QN == 2> q; QRay2 q2;
    unsigned c_nodes = 0, c_tris = 0, c_rays = 0;
    unsigned long long tl_start = 0, tl_exhausted = 0; unsigned tl_visits = 0;
    if (TIMELINE) tl_start = globaltimer_ns();

    for (;;) {
        __syncwarp();
        // ---- retire finished rays; idle lanes take the next rays in slot order (warp-wide: one atomic per round)
        if (node == SENTINEL && ray_idx >= 0) { if (!COUNT && r.best.prim < 0) store_miss(hits, ray_idx, r.best.t); ray_idx = -1; }      // (a helper, ray_idx <= -2, is retired by its delivery below)
        if (SPLIT && tail) {      // helpers whose subtree is done deliver their candidate
            unsigned fin = __ballot_sync(0xffffffffu, node == SENTINEL && ray_idx <= -2);
            while (fin) {
                const int h = __ffs(fin) - 1; fin &= fin - 1u;
                const float ht = __shfl_sync(0xffffffffu, r.best.t, h);
                const int hp = __shfl_sync(0xffffffffu, r.best.prim, h), hid = -2 - __shfl_sync(0xffffffffu, ray_idx, h);
                if ((int)lane == h) {
                    if (hp >= 0 && hp != aux[3]) {      // its own find (aux[3]: the id it started from or adopted; the subtrees of a ray's lanes are disjoint)
                        float4* rec = reinterpret_cast<float4*>(hits) + hid;
                        float rt; int rp;
                        asm volatile("ld.volatile.global.f32 %0, [%1];" : "=f"(rt) : "l"(rec));
                        asm volatile("ld.volatile.global.s32 %0, [%1+12];" : "=r"(rp) : "l"(rec));
                        if (ht < rt || (ht == rt && rp >= 0 && hp < rp)) *rec = make_float4(ht, __int_as_float(aux[0]), __int_as_float(aux[1]), __int_as_float(hp));
                    }
                    ray_idx = -1;
                } else if (node != SENTINEL && (ray_idx >= 0 ? ray_idx : -2 - ray_idx) == hid && hp >= 0 &&
                           (ht < r.best.t || (ht == r.best.t && r.best.prim >= 0 && hp < r.best.prim))) { r.best.t = ht; r.best.prim = hp; if (ray_idx <= -2) aux[3] = hp; }
                __syncwarp();
            }
        }
        for (;;) {
            const bool want = (node == SENTINEL) && !exhausted;
            const unsigned m = __ballot_sync(0xffffffffu, want);
            if (m == 0u) break;
            unsigned base = 0;
            const int leader = __ffs(m) - 1;
            if ((int)lane == leader) base = atomicAdd(counter, (unsigned)__popc(m));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (want) {
                unsigned lt_mask;                                      // read where it is used: not a register held across the traversal loops
                asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt_mask));
                const unsigned i = base + __popc(m & lt_mask);        // n < 2^31 (checked by crt_trace); the counter cannot wrap
                if ((int64_t)i >= n) { exhausted = true; }
                else {
                    const float4* rp = reinterpret_cast<const float4*>(rays + i);
                    const float4 rd = ld_stream(rp + 1);
                    if (rd.w < 0.f) {                 // inactive slot: a miss, nothing to traverse
                        if (!COUNT) store_miss(hits, i, rd.w);
                    } else {
                        r.init(ld_stream(rp), rd);
                        if (QN) q.init(r, grid);
                        if (QN == 1 || QN >= 3) q2.init(q);
                        ray_idx = (int)i; node = 0; leaf = 0; top = stack;
                        if (SPLIT) aux[2] = 0;
                        if (COUNT) ++c_rays;
                    }
                }
            }
        }
        if (__ballot_sync(0xffffffffu, node != SENTINEL) == 0u) break;     // every lane idle and the ray list is exhausted
        if (TIMELINE && tl_exhausted == 0 && __any_sync(0xffffffffu, exhausted)) tl_exhausted = globaltimer_ns();
        if (__any_sync(0xffffffffu, exhausted)) { tail = true; refill_threshold = SPLIT ? 32 : 0; }      // nothing left to fetch: run the stragglers to the end (SPLIT: come back here whenever a lane falls idle)
        if (SPLIT && tail) {
            unsigned lt_mask; asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(lt_mask));
            // (2) the k-th idle lane takes the bottom stack entry of the k-th lane that has one
            const unsigned idle = __ballot_sync(0xffffffffu, node == SENTINEL);
            const unsigned donors = __ballot_sync(0xffffffffu, node != SENTINEL && (int)(((unsigned)__cvta_generic_to_local(top) - (unsigned)__cvta_generic_to_local(stack)) >> 2) > aux[2]);      // (local-window offsets: a generic pointer difference makes the compiler carry a 64-bit copy of top through the node loop)
            const int n_pairs = min(__popc(idle), __popc(donors));
            if (n_pairs > 0) {
                const bool take = (idle >> lane & 1u) && __popc(idle & lt_mask) < n_pairs, give = (donors >> lane & 1u) && __popc(donors & lt_mask) < n_pairs;
                int e = 0;
                if (give) {
                    if (ray_idx >= 0 && r.best.prim < 0) store_miss(hits, ray_idx, r.best.t);      // the record a helper will compare with
                    const int bot = aux[2];
                    e = stack[bot + 1]; stack[bot + 1] = SENTINEL; aux[2] = bot + 1;
                }
                const int src = take ? (int)__fns(donors, 0u, __popc(idle & lt_mask) + 1) : (int)lane;
                const float4 ro = make_float4(__shfl_sync(0xffffffffu, r.o.x, src), __shfl_sync(0xffffffffu, r.o.y, src), __shfl_sync(0xffffffffu, r.o.z, src), __shfl_sync(0xffffffffu, r.tmin, src));
                const float4 rd = make_float4(__shfl_sync(0xffffffffu, r.d.x, src), __shfl_sync(0xffffffffu, r.d.y, src), __shfl_sync(0xffffffffu, r.d.z, src), __shfl_sync(0xffffffffu, r.best.t, src));
                const int bp = __shfl_sync(0xffffffffu, r.best.prim, src), didx = __shfl_sync(0xffffffffu, ray_idx, src);
                e = __shfl_sync(0xffffffffu, e, src);
                if (take) {
                    r.init(ro, rd); r.best.prim = bp;
                    if (QN) q.init(r, grid);
                    if (QN == 1 || QN >= 3) q2.init(q);
                    ray_idx = didx >= 0 ? -2 - didx : didx;
                    top = stack; aux[2] = 0; aux[3] = bp; leaf = 0; node = e;
                    if (e < 0) { leaf = e; node = SENTINEL; }      // a leaf reference: goes straight to the triangle phase
                }
            }
        }

        // ---- traverse until this lane's ray ends or too few lanes of the warp are still busy
        // (a warp-uniform formulation of these loops, every exit a full-mask vote, was measured 3-10 % slower: profiles/r01f)
        while (node != SENTINEL || (SPLIT && leaf < 0)) {
            // inner nodes; the first leaf a lane meets is postponed so that the warp's leaves are processed together
            // (several visits per vote: the vote and its warp synchronisation cost 7 issue slots)
            while ((unsigned)node < (unsigned)SENTINEL) {
#pragma unroll
                for (int rep = 0; rep < CRT_VISITS_PER_VOTE; ++rep) {
                    if (rep > 0 && (unsigned)node >= (unsigned)SENTINEL) break;
                    if (COUNT) ++c_nodes;
                    if (TIMELINE && tl_exhausted) ++tl_visits;
                    node = QN == 5 ? visit_q4node(qnodes, node, r, q2, top) : QN == 4 ? visit_qnode2<true>(qnodes, s_treelet, node, r, q2, top) : ((QN == 1 || QN == 3) ? visit_qnode2<false>(qnodes, nullptr, node, r, q2, top) : (QN ? visit_qnode(qnodes, node, r, q, top) : visit_node(load_node(nodes, node), r, top)));
                    if (node < 0 && leaf == 0) { leaf = node; node = *top--; }
                }
                if (__popc(__ballot_sync(__activemask(), leaf == 0)) <= leaf_wait) break;   // (nearly) every converged lane holds a leaf
            }
            // leaves: the postponed one, then any further leaf references that come off the stack
            while (leaf < 0) {
                visit_leaf<COUNT, QN == 3, SPLIT>(tris, leaf, r, c_tris, hits, ray_idx, aux);
                leaf = 0;
                if (node < 0) { leaf = node; node = *top--; }
            }
            if (__popc(__activemask()) < refill_threshold) break;
        }
    }
    if (TIMELINE) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) tl_visits = max(tl_visits, __shfl_xor_sync(0xffffffffu, tl_visits, d));
        if (lane == 0) {
            unsigned long long* o = stats + 4 * ((size_t)blockIdx.x * (TRACE_BLOCK / 32) + (threadIdx.x >> 5));
            o[0] = tl_start; o[1] = tl_exhausted; o[2] = globaltimer_ns(); o[3] = tl_visits;
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

struct CamDev { float eye[3], U[3], V[3], W[3]; };

// a1: camera ray of each slot's path (D:R6); the rays are then traversed by the same kernel as secondary rays
__global__ void __launch_bounds__(256) primary_rays_kernel(CamDev cam, DevLayout L, int64_t slot0, int64_t n_slots, crt_ray* __restrict__ rays, int32_t* __restrict__ r2p)
{
    int64_t i = slot0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // [slot0, n_slots): the whole frame, or one band of whole tiles
    if (i >= n_slots) return;
    int32_t pixel, sample, p;
    if (L.reuse && L.lattice == 2) {
        // LCG-sequence rule (D:R21): the slot -> pixel inverse is a discrete logarithm, so the thread is mapped FORWARD: it takes pixel number
        // n of its tile and writes the ray to the slot of the n-th term (a permutation inside the tile's block of M slots)
        const uint32_t nn = (uint32_t)(i & (L.M - 1));
        const int64_t blk = i >> L.log2M;
        const int32_t tile = (int32_t)(blk % L.n_tiles);
        sample = (int32_t)(blk / L.n_tiles);
        const uint4 r = philox((uint32_t)tile, (uint32_t)sample, 0u, PURPOSE_TILE, L.seed, L.frame);
        const uint32_t Mm = (uint32_t)(L.M - 1);
        const uint32_t m = lcg_sequence_term(((r.x & Mm) & ~3u) | 1u, (r.y & Mm) | 1u, r.z & Mm, nn, (uint32_t)L.M);
        const int32_t x = (tile % L.tiles_x) * L.W + (int32_t)(nn & (uint32_t)(L.W - 1)), y = (tile / L.tiles_x) * L.H + (int32_t)(nn >> L.log2W);
        i = (blk << L.log2M) + m;
        if (x >= L.w || y >= L.h) { pixel = -1; p = -1; }
        else { pixel = y * L.w + x; p = (int32_t)(((int64_t)sample * L.h + y) * L.w + x); }
    } else p = slot_to_path(L, i, pixel, sample);
    r2p[i] = p;
    float4* rp = reinterpret_cast<float4*>(rays + i);
    if (p < 0) { rp[0] = make_float4(0.f, 0.f, 0.f, 0.f); rp[1] = make_float4(0.f, 0.f, 0.f, -1.f); return; }
    const int32_t x = pixel % L.w, y = pixel / L.w;
    const uint4 r = philox((uint32_t)pixel, (uint32_t)sample, 0u, PURPOSE_CAMERA, L.seed, L.frame);
    const float jx = u01(r.x), jy = u01(r.y);
    const float fx = dvd(add((float)x, jx), (float)L.w), fy = dvd(add((float)y, jy), (float)L.h);
    const float sx = sub(mul(2.0f, fx), 1.0f), sy = sub(1.0f, mul(2.0f, fy));
    float dx = add(add(cam.W[0], mul(sx, cam.U[0])), mul(sy, cam.V[0]));
    float dy = add(add(cam.W[1], mul(sx, cam.U[1])), mul(sy, cam.V[1]));
    float dz = add(add(cam.W[2], mul(sx, cam.U[2])), mul(sy, cam.V[2]));
    const float len = sqr(add(add(mul(dx, dx), mul(dy, dy)), mul(dz, dz)));
    dx = dvd(dx, len); dy = dvd(dy, len); dz = dvd(dz, len);
    rp[0] = make_float4(cam.eye[0], cam.eye[1], cam.eye[2], 0.f);
    rp[1] = make_float4(dx, dy, dz, 1e30f);
}

template <bool COUNT, int QN, bool SPLIT = false, bool TIMELINE = false, int MINB = CRT_TRACE_MINB(QN)>
crt_status launch_dyn(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st, unsigned int* counter = nullptr, int64_t max_warps = 0, int32_t* n_warps = nullptr)
{
    int per_sm = ctx->trace_blocks_per_sm;
    if (per_sm <= 0) {
        CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_dyn_kernel<COUNT, QN, SPLIT, TIMELINE, MINB>, TRACE_BLOCK, QN == 4 ? (size_t)TREELET_NODES * 32 : (size_t)0));
        if (per_sm < 1) per_sm = 1;
    }
    if (!counter) counter = ctx->d_counter;
    CRT_CUDA(ctx, cudaMemsetAsync(counter, 0, sizeof(unsigned int), st));
    int64_t want = (n + TRACE_BLOCK - 1) / TRACE_BLOCK, grid = (int64_t)ctx->n_sms * per_sm;
    if (grid > want) grid = want;
    if (TIMELINE) {
        if (grid * (TRACE_BLOCK / 32) > max_warps) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_timeline: marks buffer holds %lld warps, the launch has %lld", (long long)max_warps, (long long)(grid * (TRACE_BLOCK / 32)));
        *n_warps = (int32_t)(grid * (TRACE_BLOCK / 32));
    }
    trace_dyn_kernel<COUNT, QN, SPLIT, TIMELINE, MINB><<<(unsigned)grid, TRACE_BLOCK, QN == 4 ? (size_t)TREELET_NODES * 32 : (size_t)0, st>>>(bvh->d_nodes, QN == 5 ? bvh->d_q4nodes : bvh->d_qnodes, bvh->qgrid, bvh->d_tris, rays, hits, n, counter, ctx->trace_refill_threshold, ctx->trace_leaf_wait, stats, (int)bvh->n_gpu_nodes);
    CRT_CHECK_LAUNCH(ctx, "trace_dyn");
    return CRT_OK;
}

}  // namespace

crt::DevLayout make_dev_layout(const Layout& L, const crt_frame& f)
{
    crt::DevLayout D;
    D.w = L.w; D.h = L.h; D.spp = L.spp; D.reuse = (L.mode == CRT_MODE_DIRECT_REUSE || L.mode == CRT_MODE_WORLD_REUSE);
    D.W = L.W; D.H = L.H; D.M = L.M; D.K = L.K; D.tiles_x = L.tiles_x; D.n_tiles = L.n_tiles;
    D.log2W = L.log2W; D.log2M = L.log2M; D.log2K = L.log2K; D.lattice = L.lattice; D.gw = L.gw; D.sx = L.sx; D.sy = L.sy; D.seed = (uint32_t)f.seed; D.frame = (uint32_t)f.frame;
    return D;
}

// far_origins: the caller knows the ray origins may lie beyond the default box test's contract (16 scene extents from the scene;
// crt_trace_primary checks the camera eye): the any-origin box test (trace_kernel 4's) is used instead
crt_status launch_trace(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, cudaStream_t st, bool far_origins, unsigned int* counter, bool camera_rays)
{
    if (n == 0) return CRT_OK;
    if (ctx->trace_kernel == 2 && bvh->d_wnodes && bvh->wide_violations == 0) return launch_trace_wide(ctx, bvh, rays, n, hits, st);
    if (ctx->trace_kernel == 0) {
        trace_flat_kernel<<<(unsigned)((n + TRACE_BLOCK - 1) / TRACE_BLOCK), TRACE_BLOCK, 0, st>>>(bvh->d_nodes, bvh->d_tris, rays, hits, n);
        CRT_CHECK_LAUNCH(ctx, "trace_flat");
        return CRT_OK;
    }
    // 16-bit nodes unless the grid is too coarse for this scene's detail (decoded boxes more than twice the fp32 boxes' area) or
    // the layout failed its own check (a plane clamped or less than one step outside its box: crt_bvh_check bit 16)
    const bool q_ok = bvh->q_inflation <= 2.0 && bvh->q_violations == 0;
    if (ctx->trace_kernel == 5 && !far_origins && trace_queue_supported(bvh)) return launch_trace_queue(ctx, bvh, rays, n, hits, nullptr, st);
    if (ctx->trace_kernel >= 8 && !far_origins && trace_group_supported(bvh)) return launch_trace_group(ctx, bvh, rays, n, hits, nullptr, st, counter, ctx->trace_kernel == 9 ? 32 : 16);
    if (ctx->trace_kernel == 6 && !far_origins && q_ok) return launch_dyn<false, 4>(ctx, bvh, rays, n, hits, nullptr, st, counter);
    if (ctx->trace_kernel == 7 && !far_origins && q_ok && crt_bvh_ensure_q4(bvh)) return launch_dyn<false, 5>(ctx, bvh, rays, n, hits, nullptr, st, counter);
    if (ctx->trace_kernel == 3 && !ctx->trace_exact && !far_origins && q_ok) return launch_dyn<false, 3>(ctx, bvh, rays, n, hits, nullptr, st, counter);
    if ((ctx->trace_kernel == 4 || (ctx->trace_kernel >= 3 && far_origins)) && q_ok) return launch_dyn<false, 2>(ctx, bvh, rays, n, hits, nullptr, st, counter);
    if (ctx->trace_kernel >= 3 && q_ok) return ctx->trace_tail_split ? launch_dyn<false, 1, true>(ctx, bvh, rays, n, hits, nullptr, st, counter)
                                                               : (camera_rays ? launch_dyn<false, 1>(ctx, bvh, rays, n, hits, nullptr, st, counter) : launch_dyn<false, 1, false, false, 9>(ctx, bvh, rays, n, hits, nullptr, st, counter));
    return launch_dyn<false, 0>(ctx, bvh, rays, n, hits, nullptr, st, counter);
}

// crt_trace_timeline: the default kernel (16-bit nodes) with per-warp time marks
crt_status launch_trace_timeline(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, uint64_t* marks, int64_t max_warps, int32_t* n_warps, cudaStream_t st)
{
    *n_warps = 0;
    if (n == 0) return CRT_OK;
    if (!(bvh->q_inflation <= 2.0 && bvh->q_violations == 0)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "trace_timeline: needs the 16-bit node layout");
    return ctx->trace_tail_split ? launch_dyn<false, 1, true, true>(ctx, bvh, rays, n, hits, reinterpret_cast<unsigned long long*>(marks), st, nullptr, max_warps, n_warps)
                                 : launch_dyn<false, 1, false, true>(ctx, bvh, rays, n, hits, reinterpret_cast<unsigned long long*>(marks), st, nullptr, max_warps, n_warps);
}

// counting build of the default kernel (crt_trace_stats): same traversal, no hit records written
crt_status launch_trace_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, int64_t* counters, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    if (ctx->trace_kernel == 2 && bvh->d_wnodes && bvh->wide_violations == 0) return launch_trace_wide_stats(ctx, bvh, rays, n, counters, st);
    const bool q_ok = bvh->q_inflation <= 2.0 && bvh->q_violations == 0;
    if (ctx->trace_kernel == 5 && trace_queue_supported(bvh)) return launch_trace_queue(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
    if (ctx->trace_kernel >= 8 && trace_group_supported(bvh)) return launch_trace_group(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st, nullptr, ctx->trace_kernel == 9 ? 32 : 16);
    if (ctx->trace_kernel == 7 && q_ok && crt_bvh_ensure_q4(bvh)) return launch_dyn<true, 5>(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
    if (ctx->trace_kernel == 4 && q_ok) return launch_dyn<true, 2>(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
    if (ctx->trace_kernel >= 3 && q_ok) return launch_dyn<true, 1>(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
    return launch_dyn<true, 0>(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
}

crt_status launch_primary(crt_ctx* ctx, const crt_bvh* bvh, const crt_camera& cam, const crt_frame& f, const Layout& L,
                          crt_ray* rays, crt_hit* hits, int32_t* r2p, cudaStream_t st, const Band* band)
{
    if (L.n_slots == 0) return CRT_OK;
    const int64_t slot0 = band ? band->slot0 : 0, count = band ? band->count : L.n_slots;
    if (count == 0) return CRT_OK;
    CamDev c;
    for (int k = 0; k < 3; ++k) { c.eye[k] = cam.eye[k]; c.U[k] = cam.U[k]; c.V[k] = cam.V[k]; c.W[k] = cam.W[k]; }
    primary_rays_kernel<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(c, make_dev_layout(L, f), slot0, slot0 + count, rays, r2p);
    CRT_CHECK_LAUNCH(ctx, "primary_rays");
    // the default box test is conservative for origins within 16 scene extents of the scene box (include/crt.h); a camera farther
    // away takes the any-origin test
    bool far_eye = false;
    for (int k = 0; k < 3; ++k) {
        const float ext = bvh->bounds[3 + k] - bvh->bounds[k];
        float maxext = ext; for (int j = 0; j < 3; ++j) maxext = fmaxf(maxext, bvh->bounds[3 + j] - bvh->bounds[j]);
        const float reach = 15.0f * fmaxf(ext, maxext * (1.0f / 4096.0f));
        if (cam.eye[k] < bvh->bounds[k] - reach || cam.eye[k] > bvh->bounds[3 + k] + reach) far_eye = true;
    }
    return launch_trace(ctx, bvh, rays + slot0, count, hits + slot0, st, far_eye, band ? band->counter : nullptr, true);
}
