// a6: shading of the segment just traced and image accumulation ("shading the ray hits"; P:L113, L166
// accumulation over iterations; DESIGN.md D:R14: emission on hit, environment on a miss, no next-event
// estimation, no Russian roulette).  Also crt_paths_init and the roofline microbenchmarks.
#include "crt_device.cuh"
#include "crt_internal.h"

using namespace crt;

namespace {

struct Env6 { float a[3], b[3]; };

// PIXEL_ORDER (grouped orders, last segment): thread j takes in-tile pixel number j mod M of its tile and finds its slot through the forward map
// of the partition, so that a warp's image updates fall on consecutive pixels of a tile row instead of the tile's shuffled pixels (12-byte
// read-modify-writes scattered over the tile); the 32-byte records it then gathers inside the tile's block are whole sectors either way.
template <bool PIXEL_ORDER>
__global__ void __launch_bounds__(256) shade_kernel(const int32_t* __restrict__ mat_id, int32_t n_tris, const crt_material* __restrict__ mats, Env6 env, int32_t wh,
                                                    float inv_spp, int is_last, const crt_ray* __restrict__ rays, const crt_hit* __restrict__ hits,
                                                    const int32_t* __restrict__ r2p, int64_t n, crt_path_state* __restrict__ paths,
                                                    float* __restrict__ accum, int atomic_accum, int by_slot, DevLayout L, int64_t slot0)
{
    int64_t i = slot0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // [slot0, n): the whole frame, or one band of whole tiles
    if (i >= n) return;
    if (PIXEL_ORDER) {
        const int64_t blk = i >> L.log2M;
        i = (blk << L.log2M) + pixel_to_slot_in_tile(L, (int32_t)(blk % L.n_tiles), (int32_t)(blk / L.n_tiles), (uint32_t)(i & (L.M - 1)));
    }
    const int32_t p = r2p[i];
    if (p < 0) return;
    // path state by path id (the public layout) or, inside crt_render_frame with a grouped order, by SLOT: the slot order is fixed
    // for the frame, and the shuffled pixel order of a tile would otherwise scatter these 32-byte records
    float4* pp = reinterpret_cast<float4*>(paths + (by_slot ? i : (int64_t)p));
    float4 p0 = pp[0], p1 = pp[1];
    uint32_t flags = __float_as_uint(p0.w);
    const float4 rd = __ldg(reinterpret_cast<const float4*>(rays + i) + 1);
    if ((flags & 1u) && rd.w >= 0.f) {
        const int prim = __float_as_int(__ldg(reinterpret_cast<const float4*>(hits + i)).w);
        float Le[3]; bool ends = false;
        if (prim < 0) {
            const float w = mul(0.5f, add(rd.y, 1.0f));
#pragma unroll
            for (int k = 0; k < 3; ++k) Le[k] = add(env.a[k], mul(sub(env.b[k], env.a[k]), w));
            ends = true;
        } else if (prim < n_tris) {        // (a primitive id beyond this BVH -- a stale hit buffer -- is ignored rather than dereferenced)
            const float4* mp = reinterpret_cast<const float4*>(mats + __ldg(mat_id + prim));
            const float4 m1 = __ldg(mp + 1);
            if (__float_as_int(m1.w) == CRT_MAT_EMISSIVE) { Le[0] = m1.x; Le[1] = m1.y; Le[2] = m1.z; ends = true; }
        }
        if (ends) {
            p1.x = add(p1.x, mul(p0.x, Le[0])); p1.y = add(p1.y, mul(p0.y, Le[1])); p1.z = add(p1.z, mul(p0.z, Le[2]));
            flags &= ~1u; p0.w = __uint_as_float(flags);
            pp[0] = p0; pp[1] = p1;
        }
    }
    if (is_last) {
        const int32_t pix = p % wh;
        float* a = accum + 3 * (int64_t)pix;
        if (atomic_accum) {      // several samples of one pixel may arrive concurrently
            atomicAdd(a, mul(p1.x, inv_spp)); atomicAdd(a + 1, mul(p1.y, inv_spp)); atomicAdd(a + 2, mul(p1.z, inv_spp));
        } else {
            a[0] = add(a[0], mul(p1.x, inv_spp)); a[1] = add(a[1], mul(p1.y, inv_spp)); a[2] = add(a[2], mul(p1.z, inv_spp));
        }
    }
}

__global__ void paths_init_kernel(crt_path_state* paths, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4* pp = reinterpret_cast<float4*>(paths + i);
    pp[0] = make_float4(1.f, 1.f, 1.f, __uint_as_float(1u));
    pp[1] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// FP32 peak: 8 independent FFMA chains per thread
__global__ void __launch_bounds__(256) ffma_kernel(float* out, int iters)
{
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    const float b = 0.999f, c = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = __fmaf_rn(a0, b, c); a1 = __fmaf_rn(a1, b, c); a2 = __fmaf_rn(a2, b, c); a3 = __fmaf_rn(a3, b, c);
            a4 = __fmaf_rn(a4, b, c); a5 = __fmaf_rn(a5, b, c); a6 = __fmaf_rn(a6, b, c); a7 = __fmaf_rn(a7, b, c);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}
__global__ void __launch_bounds__(256) copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, int64_t n)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace

crt::DevLayout make_dev_layout(const Layout& L, const crt_frame& f);

crt_status launch_shade(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats& mats, const crt_frame& f, int is_last,
                        const crt_ray* rays, const crt_hit* hits, const int32_t* r2p, int64_t n, crt_path_state* paths, float* accum, cudaStream_t st, bool paths_by_slot,
                        const Layout* pixel_order, const Band* band)
{
    if (n == 0) return CRT_OK;
    const int64_t slot0 = band ? band->slot0 : 0, count = band ? band->count : n, end = slot0 + count;
    if (count == 0) return CRT_OK;
    Env6 e;
    for (int k = 0; k < 3; ++k) { e.a[k] = mats.env[k]; e.b[k] = mats.env[3 + k]; }
    if (pixel_order && is_last && n == pixel_order->n_slots && ctx->shade_pixel_order)
        shade_kernel<true><<<(unsigned)((count + 255) / 256), 256, 0, st>>>(bvh->d_mat_id, (int32_t)bvh->n_tris, mats.materials, e, f.w * f.h, 1.0f / (float)f.spp, is_last, rays, hits, r2p, end,
                                                                        paths, accum, f.spp > 1, paths_by_slot ? 1 : 0, make_dev_layout(*pixel_order, f), slot0);
    else
        shade_kernel<false><<<(unsigned)((count + 255) / 256), 256, 0, st>>>(bvh->d_mat_id, (int32_t)bvh->n_tris, mats.materials, e, f.w * f.h, 1.0f / (float)f.spp, is_last, rays, hits, r2p, end,
                                                                         paths, accum, f.spp > 1, paths_by_slot ? 1 : 0, crt::DevLayout(), slot0);
    CRT_CHECK_LAUNCH(ctx, "shade");
    return CRT_OK;
}

crt_status launch_paths_init(crt_ctx* ctx, crt_path_state* paths, int64_t n, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    paths_init_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(paths, n);
    CRT_CHECK_LAUNCH(ctx, "paths_init");
    return CRT_OK;
}

crt_status measure_peaks(crt_ctx* ctx, double* tflops, double* gbs)
{
    cudaEvent_t e0, e1;
    CRT_CUDA(ctx, cudaEventCreate(&e0)); CRT_CUDA(ctx, cudaEventCreate(&e1));
    const int blocks = ctx->n_sms * 8, iters = 4096;
    float* out = nullptr;
    CRT_CUDA(ctx, cudaMalloc(&out, (size_t)blocks * 256 * 4));
    double best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        CRT_CUDA(ctx, cudaEventRecord(e0));
        ffma_kernel<<<blocks, 256>>>(out, iters);
        CRT_CUDA(ctx, cudaEventRecord(e1));
        CRT_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0; CRT_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        double fl = 2.0 * 64.0 * iters * (double)blocks * 256.0;
        if (rep > 0) best = fl / (ms * 1e-3) / 1e12 > best ? fl / (ms * 1e-3) / 1e12 : best;
    }
    cudaFree(out);
    *tflops = best;
    const int64_t n16 = (int64_t)64 << 20;     // 1 GiB each way
    float4 *a = nullptr, *b = nullptr;
    CRT_CUDA(ctx, cudaMalloc(&a, (size_t)n16 * 16)); CRT_CUDA(ctx, cudaMalloc(&b, (size_t)n16 * 16));
    CRT_CUDA(ctx, cudaMemset(a, 1, (size_t)n16 * 16));
    best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        CRT_CUDA(ctx, cudaEventRecord(e0));
        copy_kernel<<<ctx->n_sms * 16, 256>>>(a, b, n16);
        CRT_CUDA(ctx, cudaEventRecord(e1));
        CRT_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0; CRT_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        double g = 2.0 * (double)n16 * 16.0 / (ms * 1e-3) / 1e9;
        if (rep > 0 && g > best) best = g;
    }
    cudaFree(a); cudaFree(b); cudaEventDestroy(e0); cudaEventDestroy(e1);
    *gbs = best;
    return CRT_OK;
}
