// a1 + a5: primary-ray generation and BVH traversal kernels ("Each thread searches the acceleration
// structure to find the leaf nodes that the ray passes through"; this is "the most time-consuming segment").
//
// B200 design:
//  - one thread per ray, stack-based while-while traversal of a binary BVH whose 64-byte nodes hold both children's
//    boxes, fetched as two 256-bit loads (ld.global.nc.L2::256B.v8.f32 -> LDG.E.256) on the read-only path;
//  - leaf triangles are three float4 (v0|id, e1, e2) read with ld.global.nc.v4;
//  - persistent warps: the grid is sized to fill the 148 SMs once; each warp takes the next 32 consecutive rays
//    from a global counter when all of its lanes have finished (warp vote), so a slow warp never idles a whole block and
//    rays stay in slot order inside a warp -- the order the generator made coherent (group-major);
//  - no tensor cores: traversal is not a dense contraction.
// Exactness: the triangle test is the bit-exact fp32 formula of crt_device.cuh; box tests are conservative
// (padded boxes, far side inflated, subtree skipped only if its entry distance is strictly beyond the best t), so
// the result equals the all-triangles definition with ties -> lowest primitive id (D:R10).
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

constexpr int STACK_SIZE = 64;
constexpr int SENTINEL = 0x7fffffff;

struct NodeRegs { float4 xy0, xy1, z01; int ref0, ref1; };

CRT_DEV NodeRegs load_node(const GpuNode* __restrict__ nodes, int idx)
{
    // two 32-byte loads through the non-coherent path
    const float* p = reinterpret_cast<const float*>(nodes + idx);
    NodeRegs n; float a0, a1, a2, a3, a4, a5, a6, a7;
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a0), "=f"(a1), "=f"(a2), "=f"(a3), "=f"(a4), "=f"(a5), "=f"(a6), "=f"(a7) : "l"(p));
    n.xy0 = make_float4(a0, a1, a2, a3); n.xy1 = make_float4(a4, a5, a6, a7);
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a0), "=f"(a1), "=f"(a2), "=f"(a3), "=f"(a4), "=f"(a5), "=f"(a6), "=f"(a7) : "l"(p + 8));
    n.z01 = make_float4(a0, a1, a2, a3); n.ref0 = __float_as_int(a4); n.ref1 = __float_as_int(a5);
    return n;
}

struct Hit { float t, u, v; int prim; };

// nearest hit of one ray; `stack` is this thread's private stack.  COUNT: also count node visits / triangle tests.
template <bool COUNT = false>
CRT_DEV Hit traverse(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris, V3 o, V3 d, float tmin, float tmax,
                     unsigned* n_nodes = nullptr, unsigned* n_tris = nullptr)
{
    Hit best; best.t = tmax; best.u = 0.f; best.v = 0.f; best.prim = -1;
    const float idx = dvd(1.0f, d.x), idy = dvd(1.0f, d.y), idz = dvd(1.0f, d.z);
    int stack[STACK_SIZE];
    int sp = 0;
    stack[0] = SENTINEL;
    int node = 0;
    float tbest = tmax;
    while (node != SENTINEL) {
        // ---- inner nodes
        while (node >= 0 && node != SENTINEL) {
            const NodeRegs n = load_node(nodes, node);
            if (COUNT) ++*n_nodes;
            // slab test, (b - o) * (1/d): error stays relative to the result (no cancellation against o/d)
            float ax0 = (n.xy0.x - o.x) * idx, ax1 = (n.xy0.y - o.x) * idx;
            float ay0 = (n.xy0.z - o.y) * idy, ay1 = (n.xy0.w - o.y) * idy;
            float az0 = (n.z01.x - o.z) * idz, az1 = (n.z01.y - o.z) * idz;
            float bx0 = (n.xy1.x - o.x) * idx, bx1 = (n.xy1.y - o.x) * idx;
            float by0 = (n.xy1.z - o.y) * idy, by1 = (n.xy1.w - o.y) * idy;
            float bz0 = (n.z01.z - o.z) * idz, bz1 = (n.z01.w - o.z) * idz;
            float tn0 = fmaxf(fmaxf(fminf(ax0, ax1), fminf(ay0, ay1)), fmaxf(fminf(az0, az1), tmin));
            float tf0 = fminf(fminf(fmaxf(ax0, ax1), fmaxf(ay0, ay1)), fminf(fmaxf(az0, az1), tbest)) * 1.0000005f;
            float tn1 = fmaxf(fmaxf(fminf(bx0, bx1), fminf(by0, by1)), fmaxf(fminf(bz0, bz1), tmin));
            float tf1 = fminf(fminf(fmaxf(bx0, bx1), fmaxf(by0, by1)), fminf(fmaxf(bz0, bz1), tbest)) * 1.0000005f;
            const bool h0 = tn0 <= tf0, h1 = tn1 <= tf1;
            if (h0 && h1) {
                const bool swap = tn1 < tn0;
                const int nearc = swap ? n.ref1 : n.ref0, farc = swap ? n.ref0 : n.ref1;
                stack[++sp] = farc;
                node = nearc;
            } else if (h0 || h1) {
                node = h0 ? n.ref0 : n.ref1;
            } else {
                node = stack[sp--];
            }
        }
        // ---- leaves
        while (node < 0) {
            const int leaf = ~node;
            const int first = leaf >> 3, cnt = (leaf & 7) + 1;
            for (int j = 0; j < cnt; ++j) {
                const float4* tp = reinterpret_cast<const float4*>(tris + first + j);
                const float4 a = __ldg(tp), b = __ldg(tp + 1), c = __ldg(tp + 2);
                float t, u, v;
                if (COUNT) ++*n_tris;
                if (tri_test(mk(a.x, a.y, a.z), mk(b.x, b.y, b.z), mk(c.x, c.y, c.z), o, d, tmin, tmax, t, u, v)) {
                    const int prim = __float_as_int(a.w);
                    if (best.prim < 0 || t < best.t || (t == best.t && prim < best.prim)) {
                        best.t = t; best.u = u; best.v = v; best.prim = prim; tbest = t;
                    }
                }
            }
            node = stack[sp--];
        }
    }
    return best;
}

CRT_DEV void store_hit(crt_hit* hits, int64_t i, const Hit& h)
{
    reinterpret_cast<float4*>(hits)[i] = make_float4(h.t, h.u, h.v, __int_as_float(h.prim));
}

CRT_DEV void trace_one(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris, const crt_ray* __restrict__ rays,
                       crt_hit* __restrict__ hits, int64_t i)
{
    const float4* rp = reinterpret_cast<const float4*>(rays + i);
    const float4 ro = __ldg(rp), rd = __ldg(rp + 1);
    Hit h; h.t = rd.w; h.u = 0.f; h.v = 0.f; h.prim = -1;
    if (rd.w >= 0.f) h = traverse(nodes, tris, mk(ro.x, ro.y, ro.z), mk(rd.x, rd.y, rd.z), ro.w, rd.w);
    store_hit(hits, i, h);
}

// variant 0: one thread per ray
__global__ void __launch_bounds__(128) trace_flat_kernel(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris,
                                                         const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) trace_one(nodes, tris, rays, hits, i);
}

// variant 1: persistent warps, each fetching the next 32 consecutive rays when the whole warp is done
__global__ void __launch_bounds__(128) trace_persistent_kernel(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris,
                                                               const crt_ray* __restrict__ rays, crt_hit* __restrict__ hits, int64_t n,
                                                               unsigned int* __restrict__ counter)
{
    const int lane = threadIdx.x & 31;
    for (;;) {
        unsigned int base = 0;
        if (lane == 0) base = atomicAdd(counter, 32u);
        base = __shfl_sync(0xffffffffu, base, 0);
        if ((int64_t)base >= n) break;
        const int64_t i = (int64_t)base + lane;
        if (i < n) trace_one(nodes, tris, rays, hits, i);
        __syncwarp();
    }
}

// counting build of the traversal (crt_trace_stats): same code path, results discarded
__global__ void __launch_bounds__(128) trace_stats_kernel(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris,
                                                          const crt_ray* __restrict__ rays, int64_t n, unsigned long long* __restrict__ counters)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned nn = 0, nt = 0, act = 0;
    if (i < n) {
        const float4* rp = reinterpret_cast<const float4*>(rays + i);
        const float4 ro = __ldg(rp), rd = __ldg(rp + 1);
        if (rd.w >= 0.f) { act = 1; traverse<true>(nodes, tris, mk(ro.x, ro.y, ro.z), mk(rd.x, rd.y, rd.z), ro.w, rd.w, &nn, &nt); }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        nn += __shfl_xor_sync(0xffffffffu, nn, d); nt += __shfl_xor_sync(0xffffffffu, nt, d); act += __shfl_xor_sync(0xffffffffu, act, d);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(counters, (unsigned long long)nn); atomicAdd(counters + 1, (unsigned long long)nt); atomicAdd(counters + 2, (unsigned long long)act); }
}

}  // namespace

namespace {

struct CamDev { float eye[3], U[3], V[3], W[3]; };

// a1: camera ray of the slot's path, then the same traversal (D:R6)
__global__ void __launch_bounds__(128) primary_kernel(const GpuNode* __restrict__ nodes, const GpuTri* __restrict__ tris, CamDev cam,
                                                      DevLayout L, int64_t n_slots, crt_ray* __restrict__ rays, crt_hit* __restrict__ hits,
                                                      int32_t* __restrict__ r2p)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_slots) return;
    int32_t pixel, sample;
    const int32_t p = slot_to_path(L, i, pixel, sample);
    r2p[i] = p;
    float4* rp = reinterpret_cast<float4*>(rays + i);
    if (p < 0) {
        rp[0] = make_float4(0.f, 0.f, 0.f, 0.f); rp[1] = make_float4(0.f, 0.f, 0.f, -1.f);
        Hit h; h.t = -1.f; h.u = 0.f; h.v = 0.f; h.prim = -1; store_hit(hits, i, h);
        return;
    }
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
    const Hit h = traverse(nodes, tris, mk(cam.eye[0], cam.eye[1], cam.eye[2]), mk(dx, dy, dz), 0.f, 1e30f);
    store_hit(hits, i, h);
}

}  // namespace

crt::DevLayout make_dev_layout(const Layout& L, const crt_frame& f)
{
    crt::DevLayout D;
    D.w = L.w; D.h = L.h; D.spp = L.spp; D.reuse = (L.mode == CRT_MODE_DIRECT_REUSE);
    D.W = L.W; D.H = L.H; D.M = L.M; D.K = L.K; D.tiles_x = L.tiles_x; D.n_tiles = L.n_tiles;
    D.log2W = L.log2W; D.log2M = L.log2M; D.log2K = L.log2K; D.seed = (uint32_t)f.seed; D.frame = (uint32_t)f.frame;
    return D;
}

crt_status launch_trace(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    if (ctx->trace_kernel == 0) {
        const int block = 128;
        trace_flat_kernel<<<(unsigned)((n + block - 1) / block), block, 0, st>>>(bvh->d_nodes, bvh->d_tris, rays, hits, n);
    } else {
        int per_sm = ctx->trace_blocks_per_sm;
        if (per_sm <= 0) {
            CRT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trace_persistent_kernel, 128, 0));
            if (per_sm < 1) per_sm = 1;
        }
        CRT_CUDA(ctx, cudaMemsetAsync(ctx->d_counter, 0, sizeof(unsigned int), st));
        int64_t want = (n + 127) / 128, grid = (int64_t)ctx->n_sms * per_sm;
        if (grid > want) grid = want;
        trace_persistent_kernel<<<(unsigned)grid, 128, 0, st>>>(bvh->d_nodes, bvh->d_tris, rays, hits, n, ctx->d_counter);
    }
    CRT_CHECK_LAUNCH(ctx, "trace");
    return CRT_OK;
}

crt_status launch_trace_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, int64_t* counters, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    trace_stats_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(bvh->d_nodes, bvh->d_tris, rays, n, reinterpret_cast<unsigned long long*>(counters));
    CRT_CHECK_LAUNCH(ctx, "trace_stats");
    return CRT_OK;
}

crt_status launch_primary(crt_ctx* ctx, const crt_bvh* bvh, const crt_camera& cam, const crt_frame& f, const Layout& L,
                          crt_ray* rays, crt_hit* hits, int32_t* r2p, cudaStream_t st)
{
    if (L.n_slots == 0) return CRT_OK;
    CamDev c;
    for (int k = 0; k < 3; ++k) { c.eye[k] = cam.eye[k]; c.U[k] = cam.U[k]; c.V[k] = cam.V[k]; c.W[k] = cam.W[k]; }
    const int block = 128;
    primary_kernel<<<(unsigned)((L.n_slots + block - 1) / block), block, 0, st>>>(bvh->d_nodes, bvh->d_tris, c, make_dev_layout(L, f), L.n_slots,
                                                                                  rays, hits, r2p);
    CRT_CHECK_LAUNCH(ctx, "primary");
    return CRT_OK;
}
