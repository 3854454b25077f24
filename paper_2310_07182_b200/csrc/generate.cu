// a2-a4: secondary-ray generation (sections 3.2 "Tangent Space Direction Reusing" and 3.3 "Interleaved
// Grouping"; P:L103-105 group strategies; "shares directions between threads using shared memory").
//
// One thread per output slot.  In direct_reuse mode a group is K consecutive slots of one block, so the group's
// material census, its leader and (hybrid groups) the glossy members' directions are exchanged through shared
// memory; the shuffled pixel number m IS the slot, so the rays come out group-major with no sort (D:R5).
// All arithmetic is the bit-exact fp32 sequence of crt_device.cuh (D:R0).
#include "crt_device.cuh"
#include "crt_internal.h"

crt::DevLayout make_dev_layout(const Layout& L, const crt_frame& f);

using namespace crt;

namespace {

struct Frame3 { V3 tx, ty, ng; };
CRT_DEV V3 to_local(const Frame3& f, V3 w) { return mk(dot(w, f.tx), dot(w, f.ty), dot(w, f.ng)); }
CRT_DEV V3 to_world(const Frame3& f, V3 l)
{
    return mk(add(add(mul(f.tx.x, l.x), mul(f.ty.x, l.y)), mul(f.ng.x, l.z)),
              add(add(mul(f.tx.y, l.x), mul(f.ty.y, l.y)), mul(f.ng.y, l.z)),
              add(add(mul(f.tx.z, l.x), mul(f.ty.z, l.y)), mul(f.ng.z, l.z)));
}

// cosine-weighted hemisphere sample (weight = albedo)
CRT_DEV V3 sample_cosine(float u1, float u2)
{
    float r = sqr(u1), sn, cs; sincos2pi(u2, sn, cs);
    return mk(mul(r, cs), mul(r, sn), sqr(sub(1.0f, u1)));
}
CRT_DEV float smith_g1(V3 w, float al)
{
    float tan2 = dvd(add(mul(w.x, w.x), mul(w.y, w.y)), mul(w.z, w.z));
    return dvd(2.0f, add(1.0f, sqr(add(1.0f, mul(mul(al, al), tan2)))));
}
// GGX with visible-normal sampling (Heitz 2018); weight = F_schlick(F0 = albedo) * G1(wi)
CRT_DEV bool sample_ggx(V3 wo, float al, const float* albedo, float u1, float u2, V3& wi, float* weight)
{
    V3 vh = mk(mul(al, wo.x), mul(al, wo.y), wo.z);
    float vl = sqr(dot(vh, vh)); vh = mk(dvd(vh.x, vl), dvd(vh.y, vl), dvd(vh.z, vl));
    float lensq = add(mul(vh.x, vh.x), mul(vh.y, vh.y));
    V3 T1 = mk(1.0f, 0.0f, 0.0f);
    if (lensq > 0.0f) { float il = sqr(lensq); T1 = mk(dvd(-vh.y, il), dvd(vh.x, il), 0.0f); }
    V3 T2 = cross(vh, T1);
    float r = sqr(u1), sn, cs; sincos2pi(u2, sn, cs);
    float t1 = mul(r, cs), t2 = mul(r, sn);
    float sh = mul(0.5f, add(1.0f, vh.z));
    t2 = add(mul(sub(1.0f, sh), sqr(fmaxf(0.0f, sub(1.0f, mul(t1, t1))))), mul(sh, t2));
    float t3 = sqr(fmaxf(0.0f, sub(sub(1.0f, mul(t1, t1)), mul(t2, t2))));
    V3 nh = mk(add(add(mul(t1, T1.x), mul(t2, T2.x)), mul(t3, vh.x)), add(add(mul(t1, T1.y), mul(t2, T2.y)), mul(t3, vh.y)),
               add(add(mul(t1, T1.z), mul(t2, T2.z)), mul(t3, vh.z)));
    V3 h = mk(mul(al, nh.x), mul(al, nh.y), fmaxf(0.0f, nh.z));
    float hl = sqr(dot(h, h)); h = mk(dvd(h.x, hl), dvd(h.y, hl), dvd(h.z, hl));
    float woh = dot(wo, h);
    float two = mul(2.0f, woh);
    wi = mk(sub(mul(two, h.x), wo.x), sub(mul(two, h.y), wo.y), sub(mul(two, h.z), wo.z));
    if (!(wi.z > 0.0f)) return false;
    float g1 = smith_g1(wi, al);
    float c1 = sub(1.0f, woh); if (c1 < 0.0f) c1 = 0.0f;
    float c2 = mul(c1, c1), c5 = mul(mul(c2, c2), c1);
#pragma unroll
    for (int k = 0; k < 3; ++k) weight[k] = mul(add(albedo[k], mul(sub(1.0f, albedo[k]), c5)), g1);
    return true;
}

// GGX weight of a GIVEN exit direction (world-space reuse: "calculating the probability based on the direction and their
// respective materials"): F * G1(wi) with h = normalize(wo + wi)
CRT_DEV bool ggx_weight(V3 wo, V3 wi, float al, const float* albedo, float* weight)
{
    V3 h = mk(add(wo.x, wi.x), add(wo.y, wi.y), add(wo.z, wi.z));
    float hl = sqr(dot(h, h));
    if (!(hl > 0.0f)) return false;
    h = mk(dvd(h.x, hl), dvd(h.y, hl), dvd(h.z, hl));
    float woh = dot(wo, h);
    float g1 = smith_g1(wi, al);
    float c1 = sub(1.0f, woh); if (c1 < 0.0f) c1 = 0.0f;
    float c2 = mul(c1, c1), c5 = mul(mul(c2, c2), c1);
#pragma unroll
    for (int k = 0; k < 3; ++k) weight[k] = mul(add(albedo[k], mul(sub(1.0f, albedo[k]), c5)), g1);
    return true;
}

// 30-bit interleaved origin+direction code (P:L43 [AK10]; D:R12)
CRT_DEV uint32_t quant5(float x)
{
    float fl = floorf(x);
    int q = (fl < 0.0f) ? 0 : ((fl > 31.0f) ? 31 : (int)fl);
    if (x != x) q = 0;
    return (uint32_t)q;
}
CRT_DEV uint32_t spread5(uint32_t v)   // bit l of v -> bit 6*l
{
    return (v & 1u) | ((v & 2u) << 5) | ((v & 4u) << 10) | ((v & 8u) << 15) | ((v & 16u) << 20);
}
struct Bounds6 { float lo[3], scale[3]; float len; };   // scale = 32 / extent; len = 0.25 * largest extent (TwoPoint)
CRT_DEV uint32_t morton_code(const Bounds6& B, float ox, float oy, float oz, float dx, float dy, float dz)
{
    uint32_t qx = quant5(mul(sub(ox, B.lo[0]), B.scale[0])), qy = quant5(mul(sub(oy, B.lo[1]), B.scale[1])), qz = quant5(mul(sub(oz, B.lo[2]), B.scale[2]));
    uint32_t px = quant5(mul(add(dx, 1.0f), 16.0f)), py = quant5(mul(add(dy, 1.0f), 16.0f)), pz = quant5(mul(add(dz, 1.0f), 16.0f));
    return (spread5(qx) << 5) | (spread5(qy) << 4) | (spread5(qz) << 3) | (spread5(px) << 2) | (spread5(py) << 1) | spread5(pz);
}

// The other sort keys of the paper's comparison (D:R19): 1 Origin (10 bits per origin axis), 2 Reis (origin Morton
// code above direction Morton code), 3 Costa (direction above origin), 4 TwoPoint (origin and fixed-length end point interleaved).
CRT_DEV uint32_t quant10(float x)
{
    float fl = floorf(x);
    int q = (fl < 0.0f) ? 0 : ((fl > 1023.0f) ? 1023 : (int)fl);
    if (x != x) q = 0;
    return (uint32_t)q;
}
CRT_DEV uint32_t spread3(uint32_t v)   // bit l of v -> bit 3*l (10 bits)
{
    v = (v | (v << 16)) & 0x030000FFu; v = (v | (v << 8)) & 0x0300F00Fu; v = (v | (v << 4)) & 0x030C30C3u; v = (v | (v << 2)) & 0x09249249u;
    return v;
}
CRT_DEV uint32_t morton3(uint32_t x, uint32_t y, uint32_t z) { return (spread3(x) << 2) | (spread3(y) << 1) | spread3(z); }
CRT_DEV uint32_t ray_code(int code, const Bounds6& B, float ox, float oy, float oz, float dx, float dy, float dz)
{
    if (code == 0) return morton_code(B, ox, oy, oz, dx, dy, dz);
    const float rx = sub(ox, B.lo[0]), ry = sub(oy, B.lo[1]), rz = sub(oz, B.lo[2]);
    if (code == 1)      // 1024 / extent == 32 * (32 / extent) exactly
        return morton3(quant10(mul(rx, mul(B.scale[0], 32.0f))), quant10(mul(ry, mul(B.scale[1], 32.0f))), quant10(mul(rz, mul(B.scale[2], 32.0f))));
    const uint32_t qx = quant5(mul(rx, B.scale[0])), qy = quant5(mul(ry, B.scale[1])), qz = quant5(mul(rz, B.scale[2]));
    if (code == 4) {
        const float ex = add(ox, mul(B.len, dx)), ey = add(oy, mul(B.len, dy)), ez = add(oz, mul(B.len, dz));
        const uint32_t px = quant5(mul(sub(ex, B.lo[0]), B.scale[0])), py = quant5(mul(sub(ey, B.lo[1]), B.scale[1])), pz = quant5(mul(sub(ez, B.lo[2]), B.scale[2]));
        return (spread5(qx) << 5) | (spread5(qy) << 4) | (spread5(qz) << 3) | (spread5(px) << 2) | (spread5(py) << 1) | spread5(pz);
    }
    const uint32_t mo = morton3(qx, qy, qz);
    const uint32_t md = morton3(quant5(mul(add(dx, 1.0f), 16.0f)), quant5(mul(add(dy, 1.0f), 16.0f)), quant5(mul(add(dz, 1.0f), 16.0f)));
    return code == 2 ? ((mo << 15) | md) : ((md << 15) | mo);
}

struct GenArgs {
    const GpuTri* tris; const int32_t* slot_of_prim; const int32_t* mat_id; const crt_material* mats;
    const crt_ray* prev_rays; const crt_hit* prev_hits; const int32_t* prev_r2p; crt_path_state* paths;
    crt_ray* rays_out; int32_t* r2p_out; int32_t* gid_out; int32_t* src_out; uint8_t* cls_out; uint32_t* n_active;
    uint32_t* keys_out;      // morton mode: key per path (rays_out etc. are then the by-path temporaries)
    Bounds6 bounds;
    int32_t fresh;            // first bounce of a fused frame: the path state is not read (throughput 1, radiance 0, alive) and is written in full
    int32_t by_slot;          // path state indexed by slot instead of by path id (crt_render_frame, grouped orders)
    int64_t n_slots; int32_t bounce; int32_t morton;   // morton: 0 = no key, else 1 + sort code
    int64_t slot0;           // first slot of this launch (0, or the start of a band of whole tiles); n_slots = one past its last slot
    int32_t n_tris;          // hit records naming a primitive >= n_tris (a stale buffer from another BVH) are treated as dead, not dereferenced
    int32_t world;           // direct_reuse in WORLD space (mode 3; D:R18)
    int32_t fuse_shade;      // crt_render_frame: shade the previous segment here (same arithmetic as shade_kernel) instead of in its own pass
    float env[6];
};

enum { F_DEAD = 0, F_DIFF = 1, F_GLOSS = 2 };

// REUSE = true: groups of K consecutive slots share directions.  false: every path on its own (K = 1).
template <bool REUSE>
__global__ void __launch_bounds__(1024) generate_kernel(GenArgs A, DevLayout L)
{
    extern __shared__ float smem[];
    // shared: per thread  flag (int), path (int), wi.xyz (float3) -- only used when REUSE
    int* s_flag = reinterpret_cast<int*>(smem);
    int* s_path = s_flag + blockDim.x;
    float* s_wi = reinterpret_cast<float*>(s_path + blockDim.x);

    const int64_t i = A.slot0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // previous-segment slot
    const bool in_range = i < A.n_slots;
    int32_t pixel = -1, sample = 0, p = -1;
    if (in_range) {
        // the previous segment's ray_to_path is the slot -> path map in every mode (under a grouped order it equals slot_to_path(), which
        // costs a Philox call per thread; reading 4 coalesced bytes instead takes 1-3 % off this issue-bound kernel)
        p = A.prev_r2p[i];
        if (p >= 0) { pixel = p % (L.w * L.h); sample = p / (L.w * L.h); }
    }
    // ---- 1. shading point of a live path (D:R7)
    bool live = false;
    int mtype = 0; float albedo[3] = {0.f, 0.f, 0.f}, rough = 1.f;
    Frame3 fr; V3 hp = mk(0.f, 0.f, 0.f), wo = mk(0.f, 0.f, 1.f);
    fr.tx = fr.ty = fr.ng = mk(0.f, 0.f, 0.f);
    crt_path_state ps; ps.flags = 0u;
    if (p >= 0) {
        const float4* pp = reinterpret_cast<const float4*>(A.paths + (A.by_slot ? i : (int64_t)p));
        const float4 p0 = A.fresh ? make_float4(1.f, 1.f, 1.f, __uint_as_float(1u)) : pp[0];
        ps.tr = p0.x; ps.tg = p0.y; ps.tb = p0.z; ps.flags = __float_as_uint(p0.w);
        const float4 rd = __ldg(reinterpret_cast<const float4*>(A.prev_rays + i) + 1);
        const float4 hv = __ldg(reinterpret_cast<const float4*>(A.prev_hits + i));
        const int prim = __float_as_int(hv.w);
        if (A.fuse_shade && (ps.flags & 1u) && rd.w >= 0.f) {
            // a6 fused (D:R14): a miss collects the environment, an emissive hit its emission; either ends the path
            float Le[3]; bool ends = false;
            if (prim < 0) {
                const float w = mul(0.5f, add(rd.y, 1.0f));
#pragma unroll
                for (int k = 0; k < 3; ++k) Le[k] = add(A.env[k], mul(sub(A.env[3 + k], A.env[k]), w));
                ends = true;
            } else if (prim < A.n_tris) {
                const float4 m1 = __ldg(reinterpret_cast<const float4*>(A.mats + __ldg(A.mat_id + prim)) + 1);
                if (__float_as_int(m1.w) == CRT_MAT_EMISSIVE) { Le[0] = m1.x; Le[1] = m1.y; Le[2] = m1.z; ends = true; }
            }
            if (ends) {
                float4* pw = reinterpret_cast<float4*>(A.paths + (A.by_slot ? i : (int64_t)p));
                float4 p1 = A.fresh ? make_float4(0.f, 0.f, 0.f, 0.f) : pw[1];
                p1.x = add(p1.x, mul(ps.tr, Le[0])); p1.y = add(p1.y, mul(ps.tg, Le[1])); p1.z = add(p1.z, mul(ps.tb, Le[2]));
                ps.flags &= ~1u;
                pw[0] = make_float4(ps.tr, ps.tg, ps.tb, __uint_as_float(ps.flags)); pw[1] = p1;
            }
        }
        if ((ps.flags & 1u) && rd.w >= 0.f && (unsigned)prim < (unsigned)A.n_tris) {
            const float4* tp = reinterpret_cast<const float4*>(A.tris + __ldg(A.slot_of_prim + prim));
            const float4 a = __ldg(tp), b = __ldg(tp + 1), c = __ldg(tp + 2);
            const V3 v0 = mk(a.x, a.y, a.z), e1 = mk(b.x, b.y, b.z), e2 = mk(c.x, c.y, c.z), d = mk(rd.x, rd.y, rd.z);
            V3 n = cross(e1, e2);
            const float len = sqr(dot(n, n));
            V3 ng = mk(dvd(n.x, len), dvd(n.y, len), dvd(n.z, len));
            const float cosi = dot(ng, d);
            if (cosi > 0.0f) { ng = mk(-ng.x, -ng.y, -ng.z); live = true; }
            else if (cosi < 0.0f) live = true;
            if (live) {
                const float sign = ng.z >= 0.0f ? 1.0f : -1.0f;
                const float aa = dvd(-1.0f, add(sign, ng.z));
                const float bb = mul(mul(ng.x, ng.y), aa);
                fr.tx = mk(add(1.0f, mul(mul(mul(sign, ng.x), ng.x), aa)), mul(sign, bb), mul(-sign, ng.x));
                fr.ty = mk(bb, add(sign, mul(mul(ng.y, ng.y), aa)), -ng.y);
                fr.ng = ng;
                hp = mk(add(add(v0.x, mul(hv.y, e1.x)), mul(hv.z, e2.x)), add(add(v0.y, mul(hv.y, e1.y)), mul(hv.z, e2.y)),
                        add(add(v0.z, mul(hv.y, e1.z)), mul(hv.z, e2.z)));
                wo = to_local(fr, mk(-d.x, -d.y, -d.z));
                const float4* mp = reinterpret_cast<const float4*>(A.mats + __ldg(A.mat_id + prim));
                const float4 m0 = __ldg(mp), m1 = __ldg(mp + 1);
                albedo[0] = m0.x; albedo[1] = m0.y; albedo[2] = m0.z; rough = m0.w; mtype = __float_as_int(m1.w);
            }
        }
    }
    const int flag = !live ? F_DEAD : (mtype == CRT_MAT_DIFFUSE ? F_DIFF : F_GLOSS);

    // ---- 2. glossy / specular members sample from their own stream, untouched
    bool has_dir = false; V3 wi = mk(0.f, 0.f, 0.f); float weight[3] = {0.f, 0.f, 0.f}; int32_t src = -1;
    if (flag == F_GLOSS) {
        const uint4 r = philox((uint32_t)pixel, (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_BSDF, L.seed, L.frame);
        if (mtype == CRT_MAT_SPECULAR) {
            wi = mk(-wo.x, -wo.y, wo.z); has_dir = true;
            weight[0] = albedo[0]; weight[1] = albedo[1]; weight[2] = albedo[2];
        } else {
            has_dir = sample_ggx(wo, rough, albedo, u01(r.x), u01(r.y), wi, weight);
        }
        src = p;
    }
    V3 wdir = mk(0.f, 0.f, 0.f); bool has_wdir = false;
    if (REUSE && A.world && flag == F_DIFF) {          // world-space reuse: every live member first takes its own sample
        const uint4 r = philox((uint32_t)pixel, (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_BSDF, L.seed, L.frame);
        wi = sample_cosine(u01(r.x), u01(r.y));
        has_dir = true; src = p; weight[0] = albedo[0]; weight[1] = albedo[1]; weight[2] = albedo[2];
    }

    int cls = CRT_CLASS_EMPTY;
    int64_t group = i;
    if (REUSE) {
        // ---- 3. census of the group through shared memory
        const int K = L.K, tid = threadIdx.x, gbase = tid & ~(K - 1);
        group = i >> L.log2K;
        s_flag[tid] = flag | (((A.world || flag == F_GLOSS) && has_dir) ? 4 : 0);
        s_path[tid] = p;
        if (A.world) { const V3 w = has_dir ? to_world(fr, wi) : wi; s_wi[3 * tid] = w.x; s_wi[3 * tid + 1] = w.y; s_wi[3 * tid + 2] = w.z; }
        else { s_wi[3 * tid] = wi.x; s_wi[3 * tid + 1] = wi.y; s_wi[3 * tid + 2] = wi.z; }
        __syncthreads();
        bool any_diff = false, any_gloss = false, any_valid = false;
        // groups of up to 32 slots lie inside one warp: the census and the leader search are three ballots and a find-first-set instead of
        // loops over the members' flags in shared memory (same integers; the kernel is issue-bound)
        const bool in_warp = K <= 32;
        unsigned m_diff = 0u, m_live = 0u, gmask = 0u; int gshift = 0;
        if (in_warp) {
            const int myf = flag | (((A.world || flag == F_GLOSS) && has_dir) ? 4 : 0);
            const unsigned bd = __ballot_sync(0xffffffffu, (myf & 3) == F_DIFF), bg = __ballot_sync(0xffffffffu, (myf & 3) == F_GLOSS), bv = __ballot_sync(0xffffffffu, (myf & 4) != 0);
            gshift = (int)(threadIdx.x & 31u) & ~(K - 1);
            gmask = (K == 32 ? 0xffffffffu : ((1u << K) - 1u)) << gshift;
            m_diff = bd & gmask; m_live = (bd | bg) & gmask;
            any_diff = m_diff != 0u; any_gloss = (bg & gmask) != 0u; any_valid = (bv & gmask) != 0u;
        } else
        for (int j = 0; j < K; ++j) { const int f = s_flag[gbase + j]; any_diff |= (f & 3) == F_DIFF; any_gloss |= (f & 3) == F_GLOSS; any_valid |= (f & 4) != 0; }
        cls = (!any_diff && !any_gloss) ? CRT_CLASS_EMPTY : (!any_gloss ? CRT_CLASS_DIFFUSE : (!any_diff ? CRT_CLASS_GLOSSY : CRT_CLASS_HYBRID));
        // first set member of `mask` (bits gshift .. gshift + K - 1) in cyclic order from member j0: index into the block, or -1
        auto first_from = [&](unsigned mask, int j0) -> int {
            const unsigned g = (mask >> gshift) & (K == 32 ? 0xffffffffu : ((1u << K) - 1u));
            if (g == 0u) return -1;
            const unsigned hi = g >> j0;                                   // members j0 .. K-1
            const int j = hi ? j0 + (__ffs(hi) - 1) : (__ffs(g) - 1);      // else wrap to members 0 .. j0-1
            return gbase + j;
        };
        if (A.world) {
            // one randomly selected live pixel's world direction for the whole group; mirrors keep their reflection
            const uint4 rl = philox((uint32_t)group, (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_LEADER, L.seed, L.frame);
            const int j0 = (int)(rl.x & (uint32_t)(K - 1));
            int lj = -1;
            if (in_warp) lj = first_from(m_live, j0);
            else for (int t = 0; t < K; ++t) { const int j = (j0 + t) & (K - 1); if ((s_flag[gbase + j] & 3) != F_DEAD) { lj = gbase + j; break; } }
            if (flag != F_DEAD && lj >= 0 && lj != tid && (s_flag[lj] & 4) && mtype != CRT_MAT_SPECULAR) {
                wdir = mk(s_wi[3 * lj], s_wi[3 * lj + 1], s_wi[3 * lj + 2]);
                wi = to_local(fr, wdir);
                src = s_path[lj];
                if (!(wi.z > 0.0f)) has_dir = false;                 // the shared direction is below this member's horizon (Fig. 1)
                else if (flag == F_DIFF) { has_dir = true; has_wdir = true; weight[0] = albedo[0]; weight[1] = albedo[1]; weight[2] = albedo[2]; }
                else { has_dir = ggx_weight(wo, wi, rough, albedo, weight); has_wdir = has_dir; }
            }
        } else if (flag == F_DIFF) {
            if (cls == CRT_CLASS_HYBRID && any_valid) {
                // hybrid: mean tangent-space exit direction of the glossy/specular members, summed in slot order
                V3 sum = mk(0.f, 0.f, 0.f);
                for (int j = 0; j < K; ++j)
                    if (s_flag[gbase + j] & 4) sum = mk(add(sum.x, s_wi[3 * (gbase + j)]), add(sum.y, s_wi[3 * (gbase + j) + 1]), add(sum.z, s_wi[3 * (gbase + j) + 2]));
                const float len = sqr(dot(sum, sum));
                wi = mk(dvd(sum.x, len), dvd(sum.y, len), dvd(sum.z, len));
                src = (int32_t)(-2 - group);
            } else {
                // diffuse group: one randomly selected member samples, the others reuse its tangent-space direction
                const uint4 rl = philox((uint32_t)group, (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_LEADER, L.seed, L.frame);
                const int j0 = (int)(rl.x & (uint32_t)(K - 1));
                int leader = -1;
                if (in_warp) leader = s_path[first_from(m_diff, j0)];         // this member is diffuse, so the mask is not empty
                else for (int t = 0; t < K; ++t) { const int j = (j0 + t) & (K - 1); if ((s_flag[gbase + j] & 3) == F_DIFF) { leader = s_path[gbase + j]; break; } }
                const uint4 r = philox((uint32_t)(leader % (L.w * L.h)), (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_BSDF, L.seed, L.frame);
                wi = sample_cosine(u01(r.x), u01(r.y));
                src = leader;
            }
            has_dir = true; weight[0] = albedo[0]; weight[1] = albedo[1]; weight[2] = albedo[2];
        }
        if (in_range && (tid & (K - 1)) == 0) A.cls_out[group] = (uint8_t)cls;
    } else {
        if (flag == F_DIFF) {
            const uint4 r = philox((uint32_t)pixel, (uint32_t)sample, (uint32_t)A.bounce, PURPOSE_BSDF, L.seed, L.frame);
            wi = sample_cosine(u01(r.x), u01(r.y));
            has_dir = true; src = p; weight[0] = albedo[0]; weight[1] = albedo[1]; weight[2] = albedo[2];
        }
        cls = flag == F_DEAD ? CRT_CLASS_EMPTY : (flag == F_DIFF ? CRT_CLASS_DIFFUSE : CRT_CLASS_GLOSSY);
        group = p;
        if (in_range) A.cls_out[p] = (uint8_t)cls;
    }

    // ---- 4. emit
    if (!in_range) return;
    const int64_t o = REUSE ? i : (int64_t)p;            // output index: the slot, or the path id (row-major order)
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = make_float4(0.f, 0.f, 0.f, -1.f);
    const bool emit = live && has_dir;
    if (emit) {
        const V3 wd = has_wdir ? wdir : to_world(fr, wi);
        const float mx = fmaxf(fabsf(hp.x), fmaxf(fabsf(hp.y), fabsf(hp.z)));
        const float off = mul(1.0f / 32768.0f, add(1.0f, mx));
        r0 = make_float4(add(hp.x, mul(fr.ng.x, off)), add(hp.y, mul(fr.ng.y, off)), add(hp.z, mul(fr.ng.z, off)), 0.f);
        r1 = make_float4(wd.x, wd.y, wd.z, 1e30f);
    }
    if (p >= 0 && (ps.flags & 1u)) {
        // throughput *= weight; a live path that produced no ray ends here
        float4 np = make_float4(ps.tr, ps.tg, ps.tb, 0.f);
        uint32_t fl = ps.flags;
        if (emit) { np.x = mul(ps.tr, weight[0]); np.y = mul(ps.tg, weight[1]); np.z = mul(ps.tb, weight[2]); }
        else fl &= ~1u;
        np.w = __uint_as_float(fl);
        float4* pw = reinterpret_cast<float4*>(A.paths + (A.by_slot ? i : (int64_t)p));
        pw[0] = np;
        if (A.fresh) pw[1] = make_float4(0.f, 0.f, 0.f, 0.f);       // radiance of a path that goes on: nothing collected yet
    }
    if (o >= 0) {
        float4* rp = reinterpret_cast<float4*>(A.rays_out + o);
        rp[0] = r0; rp[1] = r1;
        A.r2p_out[o] = p;
        A.src_out[o] = emit ? src : -1;
        if (A.morton) A.keys_out[o] = emit ? ray_code(A.morton - 1, A.bounds, r0.x, r0.y, r0.z, r1.x, r1.y, r1.z) : 0xFFFFFFFFu;
        else A.gid_out[o] = REUSE ? (int32_t)group : p;
    }
    const unsigned m = __ballot_sync(__activemask(), emit);
    if (emit && (threadIdx.x & 31) == (__ffs(m) - 1)) atomicAdd(A.n_active, (unsigned)__popc(m));
}

__global__ void morton_encode_kernel(Bounds6 B, int code, const crt_ray* __restrict__ rays, int64_t n, uint32_t* __restrict__ keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = __ldg(reinterpret_cast<const float4*>(rays + i)), b = __ldg(reinterpret_cast<const float4*>(rays + i) + 1);
    keys[i] = b.w < 0.f ? 0xFFFFFFFFu : ray_code(code, B, a.x, a.y, a.z, b.x, b.y, b.z);
}

// rays_out[j] = tmp[perm[j]] etc.
__global__ void permute_kernel(const int32_t* __restrict__ perm, const crt_ray* __restrict__ tmp_rays, const int32_t* __restrict__ tmp_src,
                               int64_t n, crt_ray* __restrict__ rays_out, int32_t* __restrict__ r2p_out, int32_t* __restrict__ gid_out,
                               int32_t* __restrict__ src_out)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int32_t p = perm[j];
    const float4* s = reinterpret_cast<const float4*>(tmp_rays + p);
    float4* d = reinterpret_cast<float4*>(rays_out + j);
    d[0] = __ldg(s); d[1] = __ldg(s + 1);
    r2p_out[j] = p; gid_out[j] = p; src_out[j] = __ldg(tmp_src + p);
}

Bounds6 make_bounds(const float* b)
{
    Bounds6 B;
    float maxext = 0.f;
    for (int k = 0; k < 3; ++k) { B.lo[k] = b[k]; float ext = b[3 + k] - b[k]; B.scale[k] = ext > 0.f ? 32.0f / ext : 0.f; if (ext > maxext) maxext = ext; }
    B.len = 0.25f * maxext;
    return B;
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

size_t generate_scratch_bytes(const Layout& L)
{
    if (!crt_mode_sorts(L.mode)) return 256;
    const size_t n = (size_t)L.n_slots;
    return align256(n * sizeof(crt_ray)) + 5 * align256(n * 4) + align256(radix_sort_scratch_bytes(L.n_slots)) + 256;
}

crt_status launch_morton_encode(crt_ctx* ctx, const float* bounds, int code, const crt_ray* rays, int64_t n, uint32_t* keys, cudaStream_t st)
{
    if (n == 0) return CRT_OK;
    morton_encode_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(make_bounds(bounds), code, rays, n, keys);
    CRT_CHECK_LAUNCH(ctx, "morton_encode");
    return CRT_OK;
}

crt_status launch_generate(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats& mats, const crt_frame& f, int bounce, const Layout& L,
                           const crt_ray* prev_rays, const crt_hit* prev_hits, const int32_t* prev_r2p, crt_path_state* paths,
                           crt_ray* rays_out, int32_t* r2p_out, int32_t* gid_out, int32_t* src_out, uint8_t* cls_out,
                           uint32_t* n_active, void* scratch, size_t scratch_bytes, cudaStream_t st, cudaEvent_t* ev4, bool fuse_shade, bool paths_by_slot, bool fresh_paths, const Band* band)
{
    if (band) n_active = band->n_active;                  // a band adds to a count the frame zeroed before it forked
    else CRT_CUDA(ctx, cudaMemsetAsync(n_active, 0, sizeof(uint32_t), st));
    if (L.n_slots == 0 || (band && band->count == 0)) return CRT_OK;
    if (scratch_bytes < generate_scratch_bytes(L)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "generate_secondary: scratch too small");
    GenArgs A;
    A.tris = bvh->d_tris; A.slot_of_prim = bvh->d_slot_of_prim; A.mat_id = bvh->d_mat_id; A.mats = mats.materials;
    A.prev_rays = prev_rays; A.prev_hits = prev_hits; A.prev_r2p = prev_r2p; A.paths = paths;
    A.rays_out = rays_out; A.r2p_out = r2p_out; A.gid_out = gid_out; A.src_out = src_out; A.cls_out = cls_out; A.n_active = n_active;
    A.keys_out = nullptr; A.bounds = make_bounds(bvh->bounds); A.n_slots = band ? band->slot0 + band->count : L.n_slots; A.slot0 = band ? band->slot0 : 0; A.bounce = bounce; A.morton = 0; A.n_tris = (int32_t)bvh->n_tris;
    A.world = (L.mode == CRT_MODE_WORLD_REUSE);
    A.fuse_shade = fuse_shade ? 1 : 0;
    A.fresh = (fresh_paths && fuse_shade) ? 1 : 0;
    A.by_slot = (paths_by_slot && (L.mode == CRT_MODE_DIRECT_REUSE || L.mode == CRT_MODE_WORLD_REUSE)) ? 1 : 0;
    for (int k = 0; k < 6; ++k) A.env[k] = mats.env[k];
    const DevLayout D = make_dev_layout(L, f);
    const int64_t n = band ? band->count : L.n_slots;      // (the sorting modes are never banded: their sort is global)
    if (L.mode == CRT_MODE_DIRECT_REUSE || L.mode == CRT_MODE_WORLD_REUSE) {
        const int block = L.K > 256 ? L.K : 256;
        generate_kernel<true><<<(unsigned)((n + block - 1) / block), block, (size_t)block * 20, st>>>(A, D);
        CRT_CHECK_LAUNCH(ctx, "generate<reuse>");
        return CRT_OK;
    }
    if (L.mode == CRT_MODE_INDEPENDENT) {
        generate_kernel<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(A, D);
        CRT_CHECK_LAUNCH(ctx, "generate<independent>");
        return CRT_OK;
    }
    // morton_reorder and the other sort modes: independent rays by path id into scratch, with their keys; stable sort of (key, path); permute
    char* s = static_cast<char*>(scratch);
    crt_ray* tmp_rays = reinterpret_cast<crt_ray*>(s); s += align256((size_t)n * sizeof(crt_ray));
    int32_t* tmp_src = reinterpret_cast<int32_t*>(s); s += align256((size_t)n * 4);
    uint32_t* keys = reinterpret_cast<uint32_t*>(s); s += align256((size_t)n * 4);
    int32_t* idx = reinterpret_cast<int32_t*>(s); s += align256((size_t)n * 4);
    uint32_t* keys2 = reinterpret_cast<uint32_t*>(s); s += align256((size_t)n * 4);
    int32_t* perm = reinterpret_cast<int32_t*>(s); s += align256((size_t)n * 4);
    A.rays_out = tmp_rays; A.src_out = tmp_src; A.keys_out = keys; A.morton = 1 + crt_mode_sort_code(L.mode);
    A.r2p_out = idx;        // idx[p] = p
    generate_kernel<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(A, D);
    CRT_CHECK_LAUNCH(ctx, "generate<morton>");
    if (ev4) CRT_CUDA(ctx, cudaEventRecord(ev4[0], st));
    crt_status stt = launch_radix_sort(ctx, keys, idx, n, keys2, perm, s, radix_sort_scratch_bytes(n), st);
    if (stt != CRT_OK) return stt;
    permute_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(perm, tmp_rays, tmp_src, n, rays_out, r2p_out, gid_out, src_out);
    CRT_CHECK_LAUNCH(ctx, "permute");
    if (ev4) CRT_CUDA(ctx, cudaEventRecord(ev4[1], st));
    return CRT_OK;
}
