// Device-side arithmetic of libcrt.  Every floating-point operation of the METHOD (ray generation,
// triangle intersection, sampling, shading) is written with explicit round-to-nearest intrinsics so
// the compiler cannot contract a*b+c into an FMA: the result is one IEEE binary32 rounding per
// written operation (D:R0).  Only the conservative BVH box test may use FMA.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

#define CRT_DEV __device__ __forceinline__

namespace crt {

struct V3 { float x, y, z; };
CRT_DEV V3 mk(float x, float y, float z) { V3 r; r.x = x; r.y = y; r.z = z; return r; }
CRT_DEV float mul(float a, float b) { return __fmul_rn(a, b); }
CRT_DEV float add(float a, float b) { return __fadd_rn(a, b); }
CRT_DEV float sub(float a, float b) { return __fsub_rn(a, b); }
CRT_DEV float dvd(float a, float b) { return __fdiv_rn(a, b); }
CRT_DEV float sqr(float a) { return __fsqrt_rn(a); }
CRT_DEV V3 vsub(V3 a, V3 b) { return mk(sub(a.x, b.x), sub(a.y, b.y), sub(a.z, b.z)); }
CRT_DEV float dot(V3 a, V3 b) { return add(add(mul(a.x, b.x), mul(a.y, b.y)), mul(a.z, b.z)); }   // ((x+y)+z)
CRT_DEV V3 cross(V3 a, V3 b)
{
    return mk(sub(mul(a.y, b.z), mul(a.z, b.y)), sub(mul(a.z, b.x), mul(a.x, b.z)), sub(mul(a.x, b.y), mul(a.y, b.x)));
}

// ---- Philox4x32-10 (Salmon et al. 2011); key = (seed, frame), counter = (index, sample, bounce, purpose); D:R2
enum { PURPOSE_CAMERA = 0, PURPOSE_BSDF = 1, PURPOSE_TILE = 2, PURPOSE_LEADER = 3 };
CRT_DEV uint4 philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
CRT_DEV float u01(uint32_t r) { return mul((float)(r >> 8), 5.9604644775390625e-8f); }   // top 24 bits * 2^-24, exact

// sin/cos of 2*pi*u: quadrant reduction + Taylor polynomials on |x| <= pi/4, Horner (D:R9)
CRT_DEV void sincos2pi(float u, float& sn, float& cs)
{
    int k = (int)add(mul(u, 4.0f), 0.5f);
    float r = sub(u, mul((float)k, 0.25f));
    float x = mul(r, 6.2831853071795864769f);
    float x2 = mul(x, x);
    float s = mul(x, add(1.0f, mul(x2, add(-1.0f / 6.0f, mul(x2, add(1.0f / 120.0f, mul(x2, add(-1.0f / 5040.0f, mul(x2, 1.0f / 362880.0f)))))))));
    float c = add(1.0f, mul(x2, add(-0.5f, mul(x2, add(1.0f / 24.0f, mul(x2, add(-1.0f / 720.0f, mul(x2, 1.0f / 40320.0f))))))));
    switch (k & 3) {
    case 0: sn = s; cs = c; break;
    case 1: sn = c; cs = -s; break;
    case 2: sn = -s; cs = -c; break;
    default: sn = -c; cs = s; break;
    }
}

// ---- Moller-Trumbore, two-sided; NaN/inf rejects (D:R10).  e1, e2 are stored pre-subtracted.
CRT_DEV bool tri_test(V3 v0, V3 e1, V3 e2, V3 o, V3 d, float tmin, float tmax, float& t, float& u, float& v)
{
    V3 p = cross(d, e2);
    float det = dot(e1, p);
    float inv = dvd(1.0f, det);
    V3 s = vsub(o, v0);
    u = mul(dot(s, p), inv);
    V3 q = cross(s, e1);
    v = mul(dot(d, q), inv);
    t = mul(dot(e2, q), inv);
    return (u >= 0.0f) && (v >= 0.0f) && (add(u, v) <= 1.0f) && (t > tmin) && (t < tmax);
}

// The same test with fused multiply-adds and an approximate reciprocal refined by one Newton step (no IEEE-division slow path):
// NOT bit-identical to the one-rounding-per-operation sequence above (D:R0); for callers that accept north_star's stated tolerances instead of bit-identity
// (hit ids >= 99.99 %, t/u/v 1e-4 relative; option "trace_exact" = 0).  det == 0 still rejects (inf * 0 = NaN fails every compare).
CRT_DEV V3 cross_fma(V3 a, V3 b)
{
    return mk(__fmaf_rn(a.y, b.z, -__fmul_rn(a.z, b.y)), __fmaf_rn(a.z, b.x, -__fmul_rn(a.x, b.z)), __fmaf_rn(a.x, b.y, -__fmul_rn(a.y, b.x)));
}
CRT_DEV float dot_fma(V3 a, V3 b) { return __fmaf_rn(a.z, b.z, __fmaf_rn(a.y, b.y, __fmul_rn(a.x, b.x))); }
CRT_DEV bool tri_test_fast(V3 v0, V3 e1, V3 e2, V3 o, V3 d, float tmin, float tmax, float& t, float& u, float& v)
{
    const V3 p = cross_fma(d, e2);
    const float det = dot_fma(e1, p);
    float r0;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r0) : "f"(det));
    const float inv = __fmaf_rn(r0, __fmaf_rn(-det, r0, 1.0f), r0);
    const V3 s = mk(__fsub_rn(o.x, v0.x), __fsub_rn(o.y, v0.y), __fsub_rn(o.z, v0.z));
    u = __fmul_rn(dot_fma(s, p), inv);
    const V3 q = cross_fma(s, e1);
    v = __fmul_rn(dot_fma(d, q), inv);
    t = __fmul_rn(dot_fma(e2, q), inv);
    return (u >= 0.0f) && (v >= 0.0f) && (__fadd_rn(u, v) <= 1.0f) && (t > tmin) && (t < tmax);
}

// ---- slot space (D:R3-R5) ---------------------------------------------------------------------
struct DevLayout {
    int32_t w, h, spp, reuse;
    int32_t W, H, M, K, tiles_x, n_tiles, log2W, log2M, log2K;
    int32_t lattice, gw, sx, sy;       // partition rule (0 affine shuffle D:R3, 1 regular lattice D:R20, 2 LCG sequence D:R21), group width, strides
    uint32_t seed, frame;
};
// inverse of an odd number modulo 2^32 (Newton steps double the number of valid bits; a*a == 1 mod 8)
CRT_DEV uint32_t inv_odd(uint32_t a)
{
    uint32_t x = a;
    x *= 2u - a * x; x *= 2u - a * x; x *= 2u - a * x; x *= 2u - a * x;
    return x;
}
// LCG-sequence rule (D:R21): slot of in-tile pixel number n = the n-th term of x -> (A x + C) mod M started at x0, by jump-ahead
// (A^n and 1 + A + ... + A^(n-1) by repeated squaring, modulo 2^32, which M divides): log2(n) steps instead of n.
CRT_DEV uint32_t lcg_sequence_term(uint32_t A, uint32_t C, uint32_t x0, uint32_t n, uint32_t M)
{
    uint32_t ga = 1u, gc = 0u, h = A, f = C;        // after the loop: x_n = ga * x0 + gc
    while (n) {
        if (n & 1u) { ga *= h; gc = gc * h + f; }
        f *= h + 1u; h *= h; n >>= 1;
    }
    return (ga * x0 + gc) & (M - 1u);
}
// forward map of the partition: position m inside the tile's block of M slots of in-tile pixel number n = ly*W + lx (all three rules)
CRT_DEV uint32_t pixel_to_slot_in_tile(const DevLayout& L, int32_t tile, int32_t sample, uint32_t n)
{
    const uint4 r = philox((uint32_t)tile, (uint32_t)sample, 0u, PURPOSE_TILE, L.seed, L.frame);
    const uint32_t Mm = (uint32_t)(L.M - 1);
    if (L.lattice == 2) return lcg_sequence_term(((r.x & Mm) & ~3u) | 1u, (r.y & Mm) | 1u, r.z & Mm, n, (uint32_t)L.M);
    if (L.lattice == 1) {
        const uint32_t H = (uint32_t)(L.M >> L.log2W);
        const uint32_t px = ((n & (uint32_t)(L.W - 1)) + r.x % (uint32_t)L.W) & (uint32_t)(L.W - 1), py = ((n >> L.log2W) + r.y % H) & (H - 1u);
        const uint32_t g = (py % (uint32_t)L.sy) * (uint32_t)L.sx + px % (uint32_t)L.sx, j = (py / (uint32_t)L.sy) * (uint32_t)L.gw + px / (uint32_t)L.sx;
        return g * (uint32_t)L.K + j;
    }
    const uint32_t a = (r.x & Mm) | 1u, c = r.y & Mm;
    return (a * n + c) & Mm;
}
// path id of a slot (-1 = out-of-image slot) with its pixel and sample.  direct_reuse: the slot's position m in its
// tile is the shuffled number m = (a*n + c) mod M of pixel n = ly*W + lx, so n = a^-1 (m - c) mod M.
CRT_DEV int32_t slot_to_path(const DevLayout& L, int64_t slot, int32_t& pixel, int32_t& sample)
{
    if (!L.reuse) { pixel = (int32_t)(slot % ((int64_t)L.w * L.h)); sample = (int32_t)(slot / ((int64_t)L.w * L.h)); return (int32_t)slot; }
    const uint32_t m = (uint32_t)(slot & (L.M - 1));
    const int64_t blk = slot >> L.log2M;
    const int32_t tile = (int32_t)(blk % L.n_tiles);
    sample = (int32_t)(blk / L.n_tiles);
    const uint4 r = philox((uint32_t)tile, (uint32_t)sample, 0u, PURPOSE_TILE, L.seed, L.frame);
    const uint32_t a = (r.x & (uint32_t)(L.M - 1)) | 1u, c = r.y & (uint32_t)(L.M - 1);
    int32_t lx, ly;
    if (L.lattice == 1) {
        // m = g*K + j with g = (py % sy)*sx + px % sx, j = (py / sy)*gw + px / sx, (px, py) = the pixel after the tile's cyclic shift
        const int32_t g = (int32_t)(m >> L.log2K), j = (int32_t)(m & (uint32_t)(L.K - 1));
        const int32_t px = (j & (L.gw - 1)) * L.sx + (g & (L.sx - 1)), py = (j / L.gw) * L.sy + g / L.sx;
        lx = (int32_t)(((uint32_t)px - r.x % (uint32_t)L.W) & (uint32_t)(L.W - 1));
        ly = (int32_t)(((uint32_t)py - r.y % (uint32_t)L.H) & (uint32_t)(L.H - 1));
    } else {
        const uint32_t nn = (inv_odd(a) * (m - c)) & (uint32_t)(L.M - 1);
        lx = (int32_t)(nn & (uint32_t)(L.W - 1)); ly = (int32_t)(nn >> L.log2W);
    }
    const int32_t x = (tile % L.tiles_x) * L.W + lx, y = (tile / L.tiles_x) * L.H + ly;
    if (x >= L.w || y >= L.h) { pixel = -1; return -1; }
    pixel = y * L.w + x;
    return (int32_t)(((int64_t)sample * L.h + y) * L.w + x);
}

}  // namespace crt
