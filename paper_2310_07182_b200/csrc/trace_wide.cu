// a5 (alternative kernel, trace_kernel = 2): traversal of the 8-wide compressed BVH (layout: bvh_wide.cpp).
// intersection is "the most time-consuming segment" and divergent rays "lead to cache misses".
//
// Why it exists (profiles/r01a): the binary-BVH kernel is bound by the L1 data pipe, so this kernel fetches EIGHT child boxes
// per node visit with four 256-bit loads (ld.global.nc.v8: LDG.E.ENL2.256); leaves are single triangles whose box is one of
// those eight (most triangles are rejected without touching their 64-byte record), and planes are bf16 offsets decoded on
// the FMA pipe (a shift by IMAD for low halves, nothing for high halves) because the ALU pipe is the next limiter.
// What was measured (profiles/r01b): it halves the dependent fetches (23 node visits against 54) but tests 1.7x as many boxes
// at the same 16 bytes per box, so it ties with the binary kernel on the interior scene and loses on coherent rays and on the
// landscape; the binary kernel (trace.cu) therefore stays the default and this one is kept, parity-tested, for comparison.
//  - persistent warps, per-lane dynamic ray fetch in slot order (the order the generator made coherent), as in trace.cu;
//  - hit children are kept as bit groups (no per-child stack entries, no distance sort): inner hits are visited in the
//    order of descending (slot XOR octinv) via a 2 KB shared-memory table; the stack holds one 8-byte group per level;
//  - triangle tests of a warp are batched: a lane keeps its pending triangle group and the warp switches to the triangle
//    phase when enough lanes hold one (or nobody can go on with nodes);
//  - exactness: boxes are conservative (outward-rounded planes over boxes padded at build time, prune bound inflated),
//    the triangle test is the bit-exact formula, ties resolve to the lowest primitive id (D:R10).
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

constexpr int WIDE_BLOCK = 128;
constexpr int WIDE_STACK = 40;

struct Hit { float t, u, v; int prim; };

CRT_DEV void ld256(const void* p, uint32_t (&r)[8])
{
    asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
}
CRT_DEV void store_hit(crt_hit* hits, int64_t i, const Hit& h)
{
    reinterpret_cast<float4*>(hits)[i] = make_float4(h.t, h.u, h.v, __int_as_float(h.prim));
}
// 1/d with |d| clamped away from zero so that every slab distance stays finite (a ray parallel to a slab then sees both
// planes at the same huge distance of the correct sign)
CRT_DEV float safe_rcp(float d)
{
    const float eps = 8.27e-25f;                    // 2^-80
    return dvd(1.0f, fabsf(d) > eps ? d : copysignf(eps, d));
}

struct WRay {
    float ox, oy, oz, dx, dy, dz;
    float idx, idy, idz, nox, noy, noz;      // 1/d and -o/d
    float tmin, tmax, tfar;                   // tfar: best t so far, inflated (prune bound)
    uint32_t octinv;
    Hit best;
    CRT_DEV void init(float4 ro, float4 rd)
    {
        ox = ro.x; oy = ro.y; oz = ro.z; dx = rd.x; dy = rd.y; dz = rd.z;
        idx = safe_rcp(dx); idy = safe_rcp(dy); idz = safe_rcp(dz);
        nox = -ox * idx; noy = -oy * idy; noz = -oz * idz;
        tmin = ro.w; tmax = rd.w; tfar = rd.w;
        octinv = (idx < 0.f ? 0u : 4u) | (idy < 0.f ? 0u : 2u) | (idz < 0.f ? 0u : 1u);
        best.t = rd.w; best.u = 0.f; best.v = 0.f; best.prim = -1;
    }
};

// Near/far plane words of one axis, chosen by the direction sign.  w[0..3] = LO planes, w[4..7] = HI planes.
CRT_DEV void pick_planes(const uint32_t (&w)[8], bool neg, uint32_t (&wn)[4], uint32_t (&wf)[4])
{
#pragma unroll
    for (int k = 0; k < 4; ++k) { wn[k] = neg ? w[4 + k] : w[k]; wf[k] = neg ? w[k] : w[4 + k]; }
}
// bf16 plane of child j out of its word: the low half needs a shift (IMAD on the FMA pipe), the high half is used as is
// (its low 16 bits only enlarge the value; the builder rounds for that)
template <int J> CRT_DEV float plane(const uint32_t (&w)[4]) { return __uint_as_float((J & 1) ? w[J >> 1] : (w[J >> 1] << 16)); }

template <int J>
CRT_DEV uint32_t test_child(const uint32_t (&nx)[4], const uint32_t (&fx)[4], const uint32_t (&ny)[4], const uint32_t (&fy)[4],
                            const uint32_t (&nz)[4], const uint32_t (&fz)[4], float Sx, float Ox, float Sy, float Oy, float Sz, float Oz,
                            float tmin, float tfar)
{
    const float tnx = __fmaf_rn(plane<J>(nx), Sx, Ox), tny = __fmaf_rn(plane<J>(ny), Sy, Oy), tnz = __fmaf_rn(plane<J>(nz), Sz, Oz);
    const float tfx = __fmaf_rn(plane<J>(fx), Sx, Ox), tfy = __fmaf_rn(plane<J>(fy), Sy, Oy), tfz = __fmaf_rn(plane<J>(fz), Sz, Oz);
    const float N = fmaxf(fmaxf(tnx, tny), fmaxf(tnz, tmin));        // FMNMX + FMNMX3
    const float F = fminf(fminf(tfx, tfy), fminf(tfz, tfar));
    return N <= F ? (1u << J) : 0u;
}

// Tests the eight children of node `idx`; returns the slot mask of children whose (conservative) box the ray enters
// before the prune bound.  hdr receives sector 0 of the node.
CRT_DEV uint32_t visit_wnode(const WNode* __restrict__ nodes, uint32_t idx, const WRay& r, uint32_t (&hdr)[8])
{
    const char* p = reinterpret_cast<const char*>(nodes + idx);
    uint32_t ax[8], ay[8], az[8];
    ld256(p, hdr); ld256(p + 32, ax); ld256(p + 64, ay); ld256(p + 96, az);
    const float Sx = __uint_as_float(hdr[3]) * r.idx, Sy = __uint_as_float(hdr[4] & 0xffff0000u) * r.idy, Sz = __uint_as_float(hdr[4] << 16) * r.idz;   // exact: E is a power of two
    const float Ox = __fmaf_rn(__uint_as_float(hdr[0]), r.idx, r.nox), Oy = __fmaf_rn(__uint_as_float(hdr[1]), r.idy, r.noy), Oz = __fmaf_rn(__uint_as_float(hdr[2]), r.idz, r.noz);
    uint32_t nx[4], fx[4], ny[4], fy[4], nz[4], fz[4];
    pick_planes(ax, r.idx < 0.f, nx, fx); pick_planes(ay, r.idy < 0.f, ny, fy); pick_planes(az, r.idz < 0.f, nz, fz);
#define CRT_CHILD(J) test_child<J>(nx, fx, ny, fy, nz, fz, Sx, Ox, Sy, Oy, Sz, Oz, r.tmin, r.tfar)
    return (CRT_CHILD(0) | CRT_CHILD(1)) | (CRT_CHILD(2) | CRT_CHILD(3)) | ((CRT_CHILD(4) | CRT_CHILD(5)) | (CRT_CHILD(6) | CRT_CHILD(7)));
#undef CRT_CHILD
}

// D:R10: bit-exact Moeller-Trumbore; ties -> lowest primitive id
CRT_DEV void test_triangle(const GpuTri* __restrict__ tris, uint32_t ti, WRay& r)
{
    uint32_t a[8], b[8];
    const char* p = reinterpret_cast<const char*>(tris + ti);
    ld256(p, a); ld256(p + 32, b);
    float t, u, v;
    if (tri_test(mk(__uint_as_float(a[0]), __uint_as_float(a[1]), __uint_as_float(a[2])), mk(__uint_as_float(a[4]), __uint_as_float(a[5]), __uint_as_float(a[6])),
                 mk(__uint_as_float(b[0]), __uint_as_float(b[1]), __uint_as_float(b[2])), mk(r.ox, r.oy, r.oz), mk(r.dx, r.dy, r.dz), r.tmin, r.tmax, t, u, v)) {
        const int prim = (int)a[3];
        if (r.best.prim < 0 || t < r.best.t || (t == r.best.t && prim < r.best.prim)) {
            r.best.t = t; r.best.u = u; r.best.v = v; r.best.prim = prim;
            r.tfar = t * 1.0000005f;
        }
    }
}

template <bool COUNT>
__global__ void __launch_bounds__(WIDE_BLOCK, 6) trace_wide_kernel(const WNode* __restrict__ nodes, const GpuTri* __restrict__ tris,
                                                                   const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n,
                                                                   unsigned int* __restrict__ counter, int refill_threshold, int tri_wait,
                                                                   unsigned long long* __restrict__ stats)
{
    // priority table: bit s of a slot mask moves to bit (s XOR octinv)
    __shared__ uint8_t prio_lut[8 * 256];
    for (int i = threadIdx.x; i < 8 * 256; i += blockDim.x) {
        const int o = i >> 8, m = i & 255; int q = 0;
#pragma unroll
        for (int s = 0; s < 8; ++s) if ((m >> s) & 1) q |= 1 << (s ^ o);
        prio_lut[i] = (uint8_t)q;
    }
    __syncthreads();

    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    uint2 stack[WIDE_STACK]; int sp = 0;
    uint2 ng = make_uint2(0u, 0u), tg = make_uint2(0u, 0u);     // node group: x = child base, y = prio hits << 24 | imask;  triangle group: x = tri base, y = lmask << 8 | hits
    int ray_idx = -1;
    bool busy = false, exhausted = false;
    WRay r;
    unsigned c_nodes = 0, c_tris = 0, c_rays = 0;

    for (;;) {
        __syncwarp();
        // ---- retire finished rays; idle lanes take the next rays in slot order (one atomic per warp and round)
        if (!busy && ray_idx >= 0) { if (!COUNT) store_hit(hits, ray_idx, r.best); ray_idx = -1; }
        for (;;) {
            const bool want = !busy && !exhausted;
            const unsigned m = __ballot_sync(0xffffffffu, want);
            if (m == 0u) break;
            unsigned base = 0;
            const int leader = __ffs(m) - 1;
            if ((int)lane == leader) base = atomicAdd(counter, (unsigned)__popc(m));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (want) {
                const unsigned i = base + __popc(m & lt_mask);
                if ((int64_t)i >= n) exhausted = true;
                else {
                    const float4* rp = reinterpret_cast<const float4*>(rays + i);
                    const float4 rd = __ldg(rp + 1);
                    if (rd.w < 0.f) {                 // inactive slot: a miss, nothing to traverse
                        if (!COUNT) { Hit h; h.t = rd.w; h.u = 0.f; h.v = 0.f; h.prim = -1; store_hit(hits, i, h); }
                    } else {
                        r.init(__ldg(rp), rd);
                        ray_idx = (int)i; busy = true; sp = 0;
                        ng = make_uint2(0u, 0x80000000u); tg = make_uint2(0u, 0u);      // pseudo group whose only child is the root
                        if (COUNT) ++c_rays;
                    }
                }
            }
        }
        if (__ballot_sync(0xffffffffu, busy) == 0u) break;
        if (__any_sync(0xffffffffu, exhausted)) refill_threshold = 0;

        while (busy) {
            // ---- node phase: one node visit for every lane that has an inner hit left and no pending triangles
            const bool do_node = (ng.y >> 24) != 0u && (tg.y & 0xffu) == 0u;
            if (do_node) {
                const int bit = 31 - __clz(ng.y);
                ng.y &= ~(1u << bit);
                const uint32_t slot = (uint32_t)(bit - 24) ^ r.octinv;
                const uint32_t idx = ng.x + __popc(ng.y & 0xffu & ((1u << slot) - 1u));
                if ((ng.y >> 24) != 0u) stack[sp++] = ng;
                uint32_t hdr[8];
                const uint32_t mask = visit_wnode(nodes, idx, r, hdr);
                if (COUNT) ++c_nodes;
                const uint32_t imask = hdr[7] & 0xffu, lmask = (hdr[7] >> 8) & 0xffu;
                ng = make_uint2(hdr[5], ((uint32_t)prio_lut[(r.octinv << 8) | (mask & imask)] << 24) | imask);
                tg = make_uint2(hdr[6], (lmask << 8) | (mask & lmask));
            }
            // ---- triangle phase, entered together: when enough lanes hold triangles or nobody can continue with nodes
            const unsigned act = __activemask();
            const bool has_tri = (tg.y & 0xffu) != 0u;
            const unsigned tri_lanes = __ballot_sync(act, has_tri);
            const unsigned node_lanes = __ballot_sync(act, !has_tri && (ng.y >> 24) != 0u);
            if (__popc(tri_lanes) >= tri_wait || node_lanes == 0u) {
                while ((tg.y & 0xffu) != 0u) {
                    const uint32_t slot = (uint32_t)__ffs((int)(tg.y & 0xffu)) - 1u;
                    tg.y &= ~(1u << slot);
                    const uint32_t ti = tg.x + __popc((tg.y >> 8) & ((1u << slot) - 1u));
                    if (COUNT) ++c_tris;
                    test_triangle(tris, ti, r);
                }
            }
            // ---- next group
            if ((ng.y >> 24) == 0u && (tg.y & 0xffu) == 0u) {
                if (sp == 0) busy = false;
                else ng = stack[--sp];
            }
            if (__popc(__activemask()) < refill_threshold) break;
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

template <bool COUNT>
static crt_status launch_wide_t(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st)
{
    int per_sm = ctx->trace_blocks_per_sm;
    if (per_sm <= 0) {
        CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_wide_kernel<COUNT>, WIDE_BLOCK, 0));
        if (per_sm < 1) per_sm = 1;
    }
    CRT_CUDA(ctx, cudaMemsetAsync(ctx->d_counter, 0, sizeof(unsigned int), st));
    int64_t want = (n + WIDE_BLOCK - 1) / WIDE_BLOCK, grid = (int64_t)ctx->n_sms * per_sm;
    if (grid > want) grid = want;
    trace_wide_kernel<COUNT><<<(unsigned)grid, WIDE_BLOCK, 0, st>>>(bvh->d_wnodes, bvh->d_tris, rays, hits, n, ctx->d_counter, ctx->trace_refill_threshold,
                                                                    ctx->trace_tri_wait, stats);
    CRT_CHECK_LAUNCH(ctx, "trace_wide");
    return CRT_OK;
}

crt_status launch_trace_wide(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, cudaStream_t st)
{
    return launch_wide_t<false>(ctx, bvh, rays, n, hits, nullptr, st);
}
crt_status launch_trace_wide_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, int64_t* counters, cudaStream_t st)
{
    return launch_wide_t<true>(ctx, bvh, rays, n, nullptr, reinterpret_cast<unsigned long long*>(counters), st);
}
