/*
 * crt_oracle.c -- the ORACLE: a plain, slow, single-threaded CPU path tracer for
 * the secondary-bounce loop of "Generate Coherent Rays Directly" (arxiv 2310.07182).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA library
 * (paper_2310_07182_b200/csrc); it was written from PAPER.md and DESIGN.md's
 * readings alone.  Citations "P:Lnn" are /root/reference/PAPER.md line numbers;
 * "D:Rn" are the numbered readings in DESIGN.md section 3.
 *
 * Arithmetic: IEEE binary32, one rounding per written operation (build with
 * -ffp-contract=off, no -ffast-math).  The paper does not fix a precision; the
 * path's floating point decides integers (nearest-hit primitive, material class
 * of the next bounce, Morton code), so both sides take those decisions in the
 * kernel's precision, fp32 (D:R0).  Building with -DORC_REAL=double gives
 * the same procedure in fp64, used by tests to bound the fp32 rounding error.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m not gpu"):
 *   philox            cuRAND's curand_Philox4x32_10 (toolkit header, host build) + libcurand host generator
 *   sincos2pi         libm sin/cos in fp64
 *   trace (BVH)       orc_trace_brute (the plain definition: min t over ALL triangles), analytic
 *                     plane / sphere hits
 *   partition         bijection, exact cover, K members per group, quotient rule
 *   classification    constructed all-diffuse / all-mirror / checker scenes, python recount
 *   reuse rule        bit-identical local directions in a diffuse group, leader == independent sample,
 *                     upper hemisphere, fp64 normalised mean in hybrid groups
 *   cosine sampling   E[cos]=2/3 and chi-square on a histogram
 *   GGX               moments of the sampled half-vector vs fp64 quadrature of the textbook visible-normal
 *                     density D_v(h) = G1(wo) max(0, wo.h) D(h) / wo.z (Heitz 2018); weight <= 1; |wi| = 1;
 *                     white-furnace energy <= 1
 *   morton + sort     bit-by-bit loop encoder vs a python magic-mask encoder, numpy stable argsort
 *   lattice rule      (D:R20) exact cover, members congruent modulo the strides, groups = distinct residue classes, row-major
 *                     member order, one tile written out from the definition, shift varies per tile and frame, furnace == 1
 *   other sort keys   (Origin, Reis, Costa, TwoPoint; D:R19) numpy encoder, hand-derived fixture tests/golden/ray_codes.txt,
 *                     Reis/Costa halves swapped, Origin's top levels == Reis' origin half, TwoPoint with d = 0 repeats the
 *                     origin bits; each sort mode == numpy stable argsort of its key over the independent rays
 *   shade/accumulate  closed-form furnace (white sphere under uniform light == 1), albedo series
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#include <time.h>

#ifndef ORC_REAL
#define ORC_REAL float
#endif
typedef ORC_REAL real;
#define R(x) ((real)(x))
static real rsqrt_(real x) { return sizeof(real) == 4 ? (real)sqrtf((float)x) : (real)sqrt((double)x); }
static real rfloor_(real x) { return (real)floor((double)x); }
static real rabs_(real x) { return x < 0 ? -x : x; }
/* min/max that return the non-NaN operand (fminf/fmaxf semantics) */
static real rmin_(real a, real b) { return (a != a) ? b : ((b != b) ? a : (a < b ? a : b)); }
static real rmax_(real a, real b) { return (a != a) ? b : ((b != b) ? a : (a > b ? a : b)); }

/* ------------------------------------------------------------------ records
 * External records are always binary32 / int32 (D:R1 data layout).          */
typedef struct { float ox, oy, oz, tmin, dx, dy, dz, tmax; } orc_ray;      /* tmax < 0: inactive slot */
typedef struct { float t, u, v; int32_t prim; } orc_hit;                   /* prim = -1: miss */
typedef struct { float tr, tg, tb; uint32_t flags; float lr, lg, lb; uint32_t pad; } orc_path;
typedef struct { float albedo[3]; float roughness; float emission[3]; int32_t type; } orc_material;
typedef struct { int32_t w, h, spp, seed, frame; } orc_frame;
enum { MAT_DIFFUSE = 0, MAT_GLOSSY = 1, MAT_SPECULAR = 2, MAT_EMISSIVE = 3 };
enum { MODE_INDEPENDENT = 0, MODE_MORTON = 1, MODE_REUSE = 2, MODE_WORLD = 3,
       /* further reordering baselines (D:R19): same procedure as MODE_MORTON with another sort key */
       MODE_SORT_ORIGIN = 4, MODE_SORT_REIS = 5, MODE_SORT_COSTA = 6, MODE_SORT_TWOPOINT = 7 };
#define IS_SORTED(m) ((m) == MODE_MORTON || ((m) >= MODE_SORT_ORIGIN && (m) <= MODE_SORT_TWOPOINT))
/* sort key of a mode: 0 AilaCompact, 1 Origin, 2 Reis, 3 Costa, 4 TwoPoint */
#define CODE_OF_MODE(m) ((m) == MODE_MORTON ? 0 : (m) - MODE_SORT_ORIGIN + 1)
#define IS_GROUPED(m) ((m) == MODE_REUSE || (m) == MODE_WORLD)
enum { CLASS_EMPTY = 0, CLASS_DIFFUSE = 1, CLASS_GLOSSY = 2, CLASS_HYBRID = 3 };
enum { PURPOSE_CAMERA = 0, PURPOSE_BSDF = 1, PURPOSE_TILE = 2, PURPOSE_LEADER = 3 };
#define PATH_ALIVE 1u

typedef struct { real x, y, z; } vec3;
static vec3 v3(real x, real y, real z) { vec3 r = { x, y, z }; return r; }
static vec3 vsub(vec3 a, vec3 b) { return v3(a.x - b.x, a.y - b.y, a.z - b.z); }
static real vdot(vec3 a, vec3 b) { return (a.x * b.x + a.y * b.y) + a.z * b.z; }          /* ((x+y)+z) */
static vec3 vcross(vec3 a, vec3 b) { return v3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x); }

/* ------------------------------------------------------------------ RNG (D:R2)
 * Philox4x32-10 (Salmon et al. 2011), counter-based; north_star: "Philox keyed by
 * pixel, sample and bounce".  key = (seed, frame), counter = (index, sample, bounce, purpose). */
void orc_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4])
{
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* uniform in [0,1): top 24 bits, exact in binary32 */
static real u01(uint32_t r) { return R(r >> 8) * R(1.0 / 16777216.0); }
float orc_u01(uint32_t r) { return (float)u01(r); }

/* sin and cos of 2*pi*u, u in [0,1) (D:R9): quadrant reduction (exact), then Taylor
 * polynomials on |x| <= pi/4, Horner, one rounding per operation. */
static void sincos2pi(real u, real* sn, real* cs)
{
    int k = (int)(u * R(4.0) + R(0.5));
    real r = u - R(k) * R(0.25);
    real x = r * R(6.2831853071795864769);
    real x2 = x * x;
    real s = x * (R(1.0) + x2 * (R(-1.0 / 6.0) + x2 * (R(1.0 / 120.0) + x2 * (R(-1.0 / 5040.0) + x2 * R(1.0 / 362880.0)))));
    real c = R(1.0) + x2 * (R(-0.5) + x2 * (R(1.0 / 24.0) + x2 * (R(-1.0 / 720.0) + x2 * R(1.0 / 40320.0))));
    switch (k & 3) {
    case 0: *sn = s; *cs = c; break;
    case 1: *sn = c; *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
    }
}
void orc_sincos2pi(float u, float* s, float* c) { real a, b; sincos2pi(R(u), &a, &b); *s = (float)a; *c = (float)b; }

/* ------------------------------------------------------------------ intersection (D:R10)
 * Nearest hit = over ALL triangles the smallest t with tmin < t < tmax; ties -> lowest
 * primitive id.  Moller-Trumbore, two-sided; NaN/inf (det = 0) rejects. */
typedef struct { real t, u, v; int32_t prim; } hitrec;

static int tri_test(const float* tv, vec3 o, vec3 d, real tmin, real tmax, real* t_, real* u_, real* v_)
{
    vec3 v0 = v3(R(tv[0]), R(tv[1]), R(tv[2]));
    vec3 e1 = vsub(v3(R(tv[3]), R(tv[4]), R(tv[5])), v0);
    vec3 e2 = vsub(v3(R(tv[6]), R(tv[7]), R(tv[8])), v0);
    vec3 p = vcross(d, e2);
    real det = vdot(e1, p);
    real inv = R(1.0) / det;
    vec3 s = vsub(o, v0);
    real u = vdot(s, p) * inv;
    vec3 q = vcross(s, e1);
    real v = vdot(d, q) * inv;
    real t = vdot(e2, q) * inv;
    if (u >= R(0.0) && v >= R(0.0) && u + v <= R(1.0) && t > tmin && t < tmax) { *t_ = t; *u_ = u; *v_ = v; return 1; }
    return 0;
}
static void hit_consider(hitrec* best, real t, real u, real v, int32_t prim)
{
    if (best->prim < 0 || t < best->t || (t == best->t && prim < best->prim)) { best->t = t; best->u = u; best->v = v; best->prim = prim; }
}
static void write_hit(orc_hit* h, const hitrec* b, const orc_ray* r)
{
    if (b->prim >= 0) { h->t = (float)b->t; h->u = (float)b->u; h->v = (float)b->v; h->prim = b->prim; }
    else { h->t = r->tmax; h->u = 0.f; h->v = 0.f; h->prim = -1; }
}

/* The plain definition, no acceleration structure. */
void orc_trace_brute(const float* verts, int64_t n_tris, const orc_ray* rays, int64_t n_rays, orc_hit* hits)
{
    for (int64_t i = 0; i < n_rays; ++i) {
        const orc_ray* r = &rays[i];
        hitrec best = { 0, 0, 0, -1 };
        if (r->tmax >= 0.f) {
            vec3 o = v3(R(r->ox), R(r->oy), R(r->oz)), d = v3(R(r->dx), R(r->dy), R(r->dz));
            for (int64_t k = 0; k < n_tris; ++k) {
                real t, u, v;
                if (tri_test(verts + 9 * k, o, d, R(r->tmin), R(r->tmax), &t, &u, &v)) hit_consider(&best, t, u, v, (int32_t)k);
            }
        }
        write_hit(&hits[i], &best, r);
    }
}

/* ------------------------------------------------------------------ BVH (D:R11)
 * Binary tree, binned surface-area heuristic, leaves of <= 4 triangles.  The result of
 * orc_trace must equal orc_trace_brute exactly, so box tests are conservative: boxes are
 * padded at build time, a subtree is skipped only when its entry distance is strictly
 * beyond the current best t, and leaves apply the same (t, id) tie-break. */
typedef struct { float bmin[3], bmax[3]; int32_t left, right; int32_t first, count; } bnode;
typedef struct {
    const float* verts; int64_t n_tris;
    bnode* nodes; int64_t n_nodes, cap_nodes;
    int32_t* prim; float root_min[3], root_max[3]; int depth; double sah;
} orc_bvh;

#define NBINS 32
#define MAX_LEAF 4

static void tri_bounds(const float* tv, float mn[3], float mx[3])
{
    for (int a = 0; a < 3; ++a) {
        float x0 = tv[a], x1 = tv[3 + a], x2 = tv[6 + a];
        mn[a] = fminf(x0, fminf(x1, x2)); mx[a] = fmaxf(x0, fmaxf(x1, x2));
    }
}
static double half_area(const float mn[3], const float mx[3])
{
    double dx = (double)mx[0] - mn[0], dy = (double)mx[1] - mn[1], dz = (double)mx[2] - mn[2];
    return dx * dy + dy * dz + dz * dx;
}
static int64_t new_node(orc_bvh* b)
{
    if (b->n_nodes == b->cap_nodes) { b->cap_nodes = b->cap_nodes * 2 + 64; b->nodes = (bnode*)realloc(b->nodes, sizeof(bnode) * (size_t)b->cap_nodes); }
    return b->n_nodes++;
}

static void build_range(orc_bvh* b, int64_t node, int64_t lo, int64_t hi, int depth, const float* cen, float pad)
{
    /* bounds of triangles and of centroids */
    float mn[3] = { INFINITY, INFINITY, INFINITY }, mx[3] = { -INFINITY, -INFINITY, -INFINITY };
    float cmn[3] = { INFINITY, INFINITY, INFINITY }, cmx[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (int64_t i = lo; i < hi; ++i) {
        float a[3], c[3]; tri_bounds(b->verts + 9 * (int64_t)b->prim[i], a, c);
        for (int k = 0; k < 3; ++k) {
            mn[k] = fminf(mn[k], a[k]); mx[k] = fmaxf(mx[k], c[k]);
            float ce = cen[3 * (int64_t)b->prim[i] + k];
            cmn[k] = fminf(cmn[k], ce); cmx[k] = fmaxf(cmx[k], ce);
        }
    }
    bnode* nd = &b->nodes[node];
    for (int k = 0; k < 3; ++k) { nd->bmin[k] = mn[k] - pad; nd->bmax[k] = mx[k] + pad; }
    nd->left = nd->right = -1; nd->first = (int32_t)lo; nd->count = (int32_t)(hi - lo);
    if (depth > b->depth) b->depth = depth;
    int64_t n = hi - lo;
    if (n <= MAX_LEAF) { b->sah += half_area(mn, mx) * (double)n; return; }

    int best_axis = -1, best_split = -1; double best_cost = INFINITY;
    for (int axis = 0; axis < 3; ++axis) {
        float ext = cmx[axis] - cmn[axis];
        if (!(ext > 0.f)) continue;
        int64_t cnt[NBINS]; float bmn[NBINS][3], bmx[NBINS][3];
        for (int j = 0; j < NBINS; ++j) { cnt[j] = 0; for (int k = 0; k < 3; ++k) { bmn[j][k] = INFINITY; bmx[j][k] = -INFINITY; } }
        float scale = (float)NBINS / ext;
        for (int64_t i = lo; i < hi; ++i) {
            int64_t p = b->prim[i];
            int j = (int)((cen[3 * p + axis] - cmn[axis]) * scale); if (j >= NBINS) j = NBINS - 1; if (j < 0) j = 0;
            float a[3], c[3]; tri_bounds(b->verts + 9 * p, a, c);
            cnt[j]++;
            for (int k = 0; k < 3; ++k) { bmn[j][k] = fminf(bmn[j][k], a[k]); bmx[j][k] = fmaxf(bmx[j][k], c[k]); }
        }
        /* sweep from the right, then from the left */
        double rarea[NBINS]; int64_t rcnt[NBINS];
        float amn[3] = { INFINITY, INFINITY, INFINITY }, amx[3] = { -INFINITY, -INFINITY, -INFINITY }; int64_t ac = 0;
        for (int j = NBINS - 1; j >= 1; --j) {
            for (int k = 0; k < 3; ++k) { amn[k] = fminf(amn[k], bmn[j][k]); amx[k] = fmaxf(amx[k], bmx[j][k]); }
            ac += cnt[j]; rcnt[j] = ac; rarea[j] = ac ? half_area(amn, amx) : 0.0;
        }
        for (int k = 0; k < 3; ++k) { amn[k] = INFINITY; amx[k] = -INFINITY; } ac = 0;
        for (int j = 0; j < NBINS - 1; ++j) {
            for (int k = 0; k < 3; ++k) { amn[k] = fminf(amn[k], bmn[j][k]); amx[k] = fmaxf(amx[k], bmx[j][k]); }
            ac += cnt[j];
            if (ac == 0 || rcnt[j + 1] == 0) continue;
            double cost = half_area(amn, amx) * (double)ac + rarea[j + 1] * (double)rcnt[j + 1];
            if (cost < best_cost) { best_cost = cost; best_axis = axis; best_split = j; }
        }
    }
    int64_t mid;
    if (best_axis < 0) {
        mid = lo + n / 2;                       /* all centroids coincide: split the list in half */
    } else {
        float ext = cmx[best_axis] - cmn[best_axis], scale = (float)NBINS / ext;
        int64_t i = lo, j = hi - 1;
        while (i <= j) {
            int64_t p = b->prim[i];
            int bin = (int)((cen[3 * p + best_axis] - cmn[best_axis]) * scale); if (bin >= NBINS) bin = NBINS - 1; if (bin < 0) bin = 0;
            if (bin <= best_split) ++i; else { int32_t t = b->prim[i]; b->prim[i] = b->prim[j]; b->prim[j] = t; --j; }
        }
        mid = i;
        if (mid == lo || mid == hi) mid = lo + n / 2;
    }
    int64_t l = new_node(b), r = new_node(b);
    b->nodes[node].left = (int32_t)l; b->nodes[node].right = (int32_t)r; b->nodes[node].count = 0;
    build_range(b, l, lo, mid, depth + 1, cen, pad);
    build_range(b, r, mid, hi, depth + 1, cen, pad);
}

orc_bvh* orc_bvh_build(const float* verts, int64_t n_tris)
{
    orc_bvh* b = (orc_bvh*)calloc(1, sizeof(orc_bvh));
    b->verts = verts; b->n_tris = n_tris;
    b->prim = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_tris > 0 ? n_tris : 1));
    float* cen = (float*)malloc(sizeof(float) * 3 * (size_t)(n_tris > 0 ? n_tris : 1));
    for (int k = 0; k < 3; ++k) { b->root_min[k] = INFINITY; b->root_max[k] = -INFINITY; }
    float maxabs = 0.f;
    for (int64_t i = 0; i < n_tris; ++i) {
        b->prim[i] = (int32_t)i;
        float a[3], c[3]; tri_bounds(verts + 9 * i, a, c);
        for (int k = 0; k < 3; ++k) {
            cen[3 * i + k] = 0.5f * a[k] + 0.5f * c[k];
            b->root_min[k] = fminf(b->root_min[k], a[k]); b->root_max[k] = fmaxf(b->root_max[k], c[k]);
            maxabs = fmaxf(maxabs, fmaxf(fabsf(a[k]), fabsf(c[k])));
        }
    }
    if (n_tris > 0) {
        /* padding: Moller-Trumbore in fp32 can accept a hit whose exact position lies a few
         * ulps of the scene's coordinates outside the triangle's exact box */
        float pad = maxabs * (1.0f / 65536.0f);
        new_node(b);
        build_range(b, 0, 0, n_tris, 1, cen, pad);
    }
    free(cen);
    return b;
}
void orc_bvh_free(orc_bvh* b) { if (b) { free(b->nodes); free(b->prim); free(b); } }
void orc_bvh_info(const orc_bvh* b, int64_t* n_nodes, float root[6], int32_t* depth, double* sah)
{
    *n_nodes = b->n_nodes; *depth = b->depth;
    for (int k = 0; k < 3; ++k) { root[k] = b->root_min[k]; root[3 + k] = b->root_max[k]; }
    double ra = half_area(b->root_min, b->root_max);
    *sah = ra > 0 ? b->sah / ra : 0.0;
}
/* invariants: every primitive in exactly one leaf, parent box contains child boxes and
 * leaf boxes contain their triangles.  Returns 0 when all hold. */
int32_t orc_bvh_check(const orc_bvh* b)
{
    if (b->n_tris == 0) return 0;
    uint8_t* seen = (uint8_t*)calloc((size_t)b->n_tris, 1);
    int32_t bad = 0;
    for (int64_t i = 0; i < b->n_nodes; ++i) {
        const bnode* n = &b->nodes[i];
        if (n->left >= 0) {
            const bnode* ch[2] = { &b->nodes[n->left], &b->nodes[n->right] };
            for (int c = 0; c < 2; ++c) for (int k = 0; k < 3; ++k)
                if (ch[c]->bmin[k] < n->bmin[k] || ch[c]->bmax[k] > n->bmax[k]) bad |= 1;
        } else {
            if (n->count < 1 || n->count > MAX_LEAF) bad |= 2;
            for (int32_t j = 0; j < n->count; ++j) {
                int32_t p = b->prim[n->first + j];
                if (seen[p]) bad |= 4; seen[p] = 1;
                float a[3], c[3]; tri_bounds(b->verts + 9 * (int64_t)p, a, c);
                for (int k = 0; k < 3; ++k) if (a[k] < n->bmin[k] || c[k] > n->bmax[k]) bad |= 8;
            }
        }
    }
    for (int64_t i = 0; i < b->n_tris; ++i) if (!seen[i]) bad |= 16;
    free(seen);
    return bad;
}

/* slab test; returns entry distance in *tn.  Conservative: far side inflated. */
static int box_test(const bnode* n, vec3 o, vec3 inv, real tmin, real tbest, real* tn)
{
    real t0 = (R(n->bmin[0]) - o.x) * inv.x, t1 = (R(n->bmax[0]) - o.x) * inv.x;
    real near = rmin_(t0, t1), far = rmax_(t0, t1);
    t0 = (R(n->bmin[1]) - o.y) * inv.y; t1 = (R(n->bmax[1]) - o.y) * inv.y;
    near = rmax_(near, rmin_(t0, t1)); far = rmin_(far, rmax_(t0, t1));
    t0 = (R(n->bmin[2]) - o.z) * inv.z; t1 = (R(n->bmax[2]) - o.z) * inv.z;
    near = rmax_(near, rmin_(t0, t1)); far = rmin_(far, rmax_(t0, t1));
    near = rmax_(near, tmin);
    far = rmin_(far, tbest) * R(1.0000005);
    *tn = near;
    return near <= far;
}

/* counters[0] += node visits, counters[1] += triangle tests (may be NULL) */
void orc_trace(const orc_bvh* b, const orc_ray* rays, int64_t n_rays, orc_hit* hits, int64_t* counters)
{
    int64_t nv = 0, nt = 0;
    int32_t stack[128];
    for (int64_t i = 0; i < n_rays; ++i) {
        const orc_ray* r = &rays[i];
        hitrec best = { 0, 0, 0, -1 };
        if (r->tmax >= 0.f && b->n_tris > 0) {
            vec3 o = v3(R(r->ox), R(r->oy), R(r->oz)), d = v3(R(r->dx), R(r->dy), R(r->dz));
            vec3 inv = v3(R(1.0) / d.x, R(1.0) / d.y, R(1.0) / d.z);
            real tbest = R(r->tmax);
            int sp = 0; stack[sp++] = 0;
            while (sp) {
                const bnode* n = &b->nodes[stack[--sp]];
                real tn; ++nv;
                if (!box_test(n, o, inv, R(r->tmin), tbest, &tn)) continue;
                if (n->left >= 0) {
                    real ta, tb;
                    int ha = box_test(&b->nodes[n->left], o, inv, R(r->tmin), tbest, &ta);
                    int hb = box_test(&b->nodes[n->right], o, inv, R(r->tmin), tbest, &tb);
                    /* push the farther child first so the nearer is popped first */
                    if (ha && hb) { if (ta <= tb) { stack[sp++] = n->right; stack[sp++] = n->left; } else { stack[sp++] = n->left; stack[sp++] = n->right; } }
                    else if (ha) stack[sp++] = n->left;
                    else if (hb) stack[sp++] = n->right;
                } else {
                    for (int32_t j = 0; j < n->count; ++j) {
                        int32_t p = b->prim[n->first + j]; real t, u, v; ++nt;
                        /* accept t <= current best (ties resolved by id), never beyond the ray's tmax */
                        if (tri_test(b->verts + 9 * (int64_t)p, o, d, R(r->tmin), R(r->tmax), &t, &u, &v) && (best.prim < 0 || t <= best.t)) {
                            hit_consider(&best, t, u, v, p); tbest = best.t;
                        }
                    }
                }
            }
        }
        write_hit(&hits[i], &best, r);
    }
    if (counters) { counters[0] += nv; counters[1] += nt; }
}

/* ------------------------------------------------------------------ partition (D:R3-R5)
 * BASELINE.json's "group gw x gh, interleave stride s"  <->  the paper's tile W x H and
 * group size K:  K = gw*gh, W = gw*s, H = gh*s, M = W*H slots per tile, G = M/K groups. */
typedef struct { int32_t W, H, M, K, G, tiles_x, tiles_y, n_tiles; int64_t n_slots, n_paths; int32_t gw, gh, sx, sy, lattice, sequence; } layout;
static layout make_layout(const orc_frame* f, int mode, int gw, int gh, int s)
{
    layout L; memset(&L, 0, sizeof L);
    L.n_paths = (int64_t)f->spp * f->w * f->h;
    if (!IS_GROUPED(mode)) { L.W = L.H = L.M = L.K = L.G = 1; L.tiles_x = f->w; L.tiles_y = f->h; L.n_tiles = f->w * f->h; L.n_slots = L.n_paths; return L; }
    /* the paper's native parametrisation is a W x H tile and a group size K (tile 8x8, K = 8).  Any power-of-two
     * (W, H, K) is gw = min(K, W), gh = K / gw with separate horizontal / vertical strides W / gw, H / gh; the vertical
     * stride travels in the high 16 bits of s (0 = same as the horizontal one).  DESIGN.md D:R5. */
    int32_t sx = s & 0x3fff, sy = (s >> 16) ? (s >> 16) : sx;
    L.gw = gw; L.gh = gh; L.sx = sx; L.sy = sy; L.lattice = (s >> 14) & 1;      /* bit 14: partition rule LATTICE (D:R20) */
    L.sequence = (s >> 15) & 1;                                                 /* bit 15: partition rule LCG SEQUENCE (D:R21) */
    L.W = gw * sx; L.H = gh * sy; L.M = L.W * L.H; L.K = gw * gh; L.G = L.M / L.K;
    L.tiles_x = (f->w + L.W - 1) / L.W; L.tiles_y = (f->h + L.H - 1) / L.H; L.n_tiles = L.tiles_x * L.tiles_y;
    L.n_slots = (int64_t)f->spp * L.n_tiles * L.M;
    return L;
}
int64_t orc_n_slots(const orc_frame* f, int32_t mode, int32_t gw, int32_t gh, int32_t s) { return make_layout(f, mode, gw, gh, s).n_slots; }
int64_t orc_n_groups(const orc_frame* f, int32_t mode, int32_t gw, int32_t gh, int32_t s) { layout L = make_layout(f, mode, gw, gh, s); return L.n_slots / L.K; }

/* "pixels are numbered based on their order on the screen. These numbers are then shuffled
 * using a linear congruence method": m = (a*n + c) mod M, a odd (D:R3). */
static void tile_lcg(const orc_frame* f, const layout* L, int32_t tile, int32_t sample, uint32_t* a, uint32_t* c)
{
    uint32_t r[4];
    orc_philox((uint32_t)tile, (uint32_t)sample, 0u, PURPOSE_TILE, (uint32_t)f->seed, (uint32_t)f->frame, r);
    *a = (r[0] % (uint32_t)L->M) | 1u;
    *c = r[1] % (uint32_t)L->M;
}
static void tile_raw(const orc_frame* f, int32_t tile, int32_t sample, uint32_t* r0, uint32_t* r1)
{
    uint32_t r[4];
    orc_philox((uint32_t)tile, (uint32_t)sample, 0u, PURPOSE_TILE, (uint32_t)f->seed, (uint32_t)f->frame, r);
    *r0 = r[0]; *r1 = r[1];
}
/* path id p = (sample*h + y)*w + x.  Fills path_of_slot[n_slots] (-1: out-of-image slot). */
static void partition(const orc_frame* f, const layout* L, int mode, int32_t* path_of_slot)
{
    if (!IS_GROUPED(mode)) { for (int64_t p = 0; p < L->n_paths; ++p) path_of_slot[p] = (int32_t)p; return; }
    for (int64_t i = 0; i < L->n_slots; ++i) path_of_slot[i] = -1;
    for (int32_t sg = 0; sg < f->spp; ++sg)
        for (int32_t tile = 0; tile < L->n_tiles; ++tile) {
            uint32_t a, c, a0, c0; tile_lcg(f, L, tile, sg, &a, &c); tile_raw(f, tile, sg, &a0, &c0);
            int32_t tx = tile % L->tiles_x, ty = tile / L->tiles_x;
            /* third reading of "shuffled using a linear congruence method" (S:8c A-1; D:R21): the shuffled number of pixel n is
             * the n-th term of a linear congruential SEQUENCE x_{n+1} = (A x_n + C) mod M of full period (Hull-Dobell for M a power
             * of two: C odd, A = 1 mod 4), started at x_0; A, C, x_0 from the TILE stream, so it varies per tile, sample and frame. */
            uint32_t seqA = 1, seqC = 1, xs = 0;
            if (L->sequence) {
                uint32_t r[4];
                orc_philox((uint32_t)tile, (uint32_t)sg, 0u, PURPOSE_TILE, (uint32_t)f->seed, (uint32_t)f->frame, r);
                seqA = ((r[0] % (uint32_t)L->M) & ~3u) | 1u; seqC = (r[1] % (uint32_t)L->M) | 1u; xs = r[2] % (uint32_t)L->M;
            }
            for (int32_t n = 0; n < L->M; ++n) {
                int32_t lx = n % L->W, ly = n / L->W;                  /* order on the screen inside the tile */
                int32_t x = tx * L->W + lx, y = ty * L->H + ly;
                uint32_t xn = xs;                                      /* n-th term of the sequence; the next pixel number gets the next term */
                xs = (seqA * xs + seqC) % (uint32_t)L->M;
                if (x >= f->w || y >= f->h) continue;
                uint32_t m = (a * (uint32_t)n + c) % (uint32_t)L->M;   /* shuffled number */
                if (L->sequence) m = xn;
                if (L->lattice) {
                    /* alternative reading of BASELINE's "interleave stride" (S:8c A-3; D:R20): a REGULAR lattice.  The tile is
                     * shifted cyclically by an offset drawn per tile, sample and frame ("varies in each tile and in each frame",
                     * P:L113); pixels congruent modulo (sx, sy) form a group: its gw x gh members lie sx apart horizontally and
                     * sy apart vertically.  Group-major position m = group * K + member, as in the shuffled rule. */
                    int32_t px = (lx + (int32_t)(a0 % (uint32_t)L->W)) % L->W, py = (ly + (int32_t)(c0 % (uint32_t)L->H)) % L->H;
                    int32_t g = (py % L->sy) * L->sx + (px % L->sx), j = (py / L->sy) * L->gw + (px / L->sx);
                    m = (uint32_t)(g * L->K + j);
                }
                /* group = m / K ("divided by K, yield the same quotient"); the shuffled number
                 * is also the ray's position inside the tile's slot block (D:R5) */
                int64_t slot = ((int64_t)sg * L->n_tiles + tile) * L->M + m;
                path_of_slot[slot] = (int32_t)(((int64_t)sg * f->h + y) * f->w + x);
            }
        }
}
void orc_partition(const orc_frame* f, int32_t mode, int32_t gw, int32_t gh, int32_t s, int32_t* path_of_slot)
{
    layout L = make_layout(f, mode, gw, gh, s); partition(f, &L, mode, path_of_slot);
}

/* ------------------------------------------------------------------ primary rays (D:R6)
 * cam = eye[3], U[3], V[3], W[3].  One camera ray per path, jittered inside the pixel. */
static void camera_ray(const float* cam, const orc_frame* f, int32_t x, int32_t y, int32_t sample, orc_ray* out)
{
    uint32_t r[4];
    orc_philox((uint32_t)(y * f->w + x), (uint32_t)sample, 0u, PURPOSE_CAMERA, (uint32_t)f->seed, (uint32_t)f->frame, r);
    real jx = u01(r[0]), jy = u01(r[1]);
    real fx = (R(x) + jx) / R(f->w), fy = (R(y) + jy) / R(f->h);
    real sx = R(2.0) * fx - R(1.0), sy = R(1.0) - R(2.0) * fy;
    real d[3];
    for (int k = 0; k < 3; ++k) d[k] = (R(cam[9 + k]) + sx * R(cam[3 + k])) + sy * R(cam[6 + k]);
    real len = rsqrt_((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
    out->ox = cam[0]; out->oy = cam[1]; out->oz = cam[2]; out->tmin = 0.f;
    out->dx = (float)(d[0] / len); out->dy = (float)(d[1] / len); out->dz = (float)(d[2] / len); out->tmax = 1e30f;
}
static void inactive_ray(orc_ray* r) { memset(r, 0, sizeof *r); r->tmax = -1.f; }

void orc_trace_primary(const orc_bvh* b, const float* cam, const orc_frame* f, int32_t mode, int32_t gw, int32_t gh, int32_t s,
                       orc_ray* rays, orc_hit* hits, int32_t* ray_to_path)
{
    layout L = make_layout(f, mode, gw, gh, s);
    partition(f, &L, mode, ray_to_path);
    for (int64_t i = 0; i < L.n_slots; ++i) {
        int32_t p = ray_to_path[i];
        if (p < 0) { inactive_ray(&rays[i]); continue; }
        int32_t x = p % f->w, y = (p / f->w) % f->h, sg = p / (f->w * f->h);
        camera_ray(cam, f, x, y, sg, &rays[i]);
    }
    orc_trace(b, rays, L.n_slots, hits, NULL);
}

/* ------------------------------------------------------------------ shading point (D:R7, R8) */
typedef struct {
    int live; int mtype; int32_t prim; int32_t pixel, sample;
    vec3 ng, tx, ty;       /* frame: tangent, bitangent, face-forwarded geometric normal */
    vec3 p;                /* hit position */
    vec3 wo;               /* -d_prev in local coordinates */
    real albedo[3], rough;
    /* filled by the group rules */
    int has_dir; vec3 wi; real weight[3]; int32_t dir_src;
    int has_wdir; vec3 wdir;   /* world-space reuse: the shared world direction, used as is */
} shadept;

static vec3 to_local(const shadept* s, vec3 w) { return v3(vdot(w, s->tx), vdot(w, s->ty), vdot(w, s->ng)); }
static vec3 to_world(const shadept* s, vec3 l)
{
    return v3((s->tx.x * l.x + s->ty.x * l.y) + s->ng.x * l.z, (s->tx.y * l.x + s->ty.y * l.y) + s->ng.y * l.z,
              (s->tx.z * l.x + s->ty.z * l.y) + s->ng.z * l.z);
}
/* returns 0 if the path must be killed (grazing: d_prev . ng == 0) */
static int shading_point(const float* verts, const int32_t* mat_id, const orc_material* mats, const orc_ray* ray, const orc_hit* hit, shadept* s)
{
    const float* tv = verts + 9 * (int64_t)hit->prim;
    vec3 v0 = v3(R(tv[0]), R(tv[1]), R(tv[2]));
    vec3 e1 = vsub(v3(R(tv[3]), R(tv[4]), R(tv[5])), v0), e2 = vsub(v3(R(tv[6]), R(tv[7]), R(tv[8])), v0);
    vec3 n = vcross(e1, e2);
    real len = rsqrt_(vdot(n, n));
    vec3 ng = v3(n.x / len, n.y / len, n.z / len);
    vec3 d = v3(R(ray->dx), R(ray->dy), R(ray->dz));
    real cosi = vdot(ng, d);
    if (cosi > R(0.0)) ng = v3(-ng.x, -ng.y, -ng.z);          /* face-forward: ng . (-d_prev) > 0 */
    else if (!(cosi < R(0.0))) return 0;
    /* tangent frame = a function of the normal only, so parallel surfaces share the frame and a
     * shared tangent-space direction gives parallel world-space rays.  Branch-free
     * orthonormal basis (Duff et al. 2017). */
    real sign = ng.z >= R(0.0) ? R(1.0) : R(-1.0);
    real a = R(-1.0) / (sign + ng.z);
    real bb = (ng.x * ng.y) * a;
    s->tx = v3(R(1.0) + ((sign * ng.x) * ng.x) * a, sign * bb, (-sign) * ng.x);
    s->ty = v3(bb, sign + (ng.y * ng.y) * a, -ng.y);
    s->ng = ng;
    real u = R(hit->u), v = R(hit->v);
    s->p = v3((v0.x + u * e1.x) + v * e2.x, (v0.y + u * e1.y) + v * e2.y, (v0.z + u * e1.z) + v * e2.z);
    s->wo = to_local(s, v3(-d.x, -d.y, -d.z));
    const orc_material* m = &mats[mat_id[hit->prim]];
    s->mtype = m->type; s->prim = hit->prim; s->rough = R(m->roughness);
    for (int k = 0; k < 3; ++k) s->albedo[k] = R(m->albedo[k]);
    return 1;
}

/* ------------------------------------------------------------------ BSDF sampling (D:R9)
 * (u1,u2) = first two floats of Philox(ctr = (pixel of the stream's owner, sample, bounce, BSDF)). */
static void bsdf_uniforms(const orc_frame* f, int32_t pixel, int32_t sample, int32_t bounce, real* u1, real* u2)
{
    uint32_t r[4];
    orc_philox((uint32_t)pixel, (uint32_t)sample, (uint32_t)bounce, PURPOSE_BSDF, (uint32_t)f->seed, (uint32_t)f->frame, r);
    *u1 = u01(r[0]); *u2 = u01(r[1]);
}
/* cosine-weighted hemisphere; weight = albedo (pdf cancels cos/pi) */
static vec3 sample_cosine(real u1, real u2)
{
    real r = rsqrt_(u1), sn, cs; sincos2pi(u2, &sn, &cs);
    return v3(r * cs, r * sn, rsqrt_(R(1.0) - u1));
}
static real smith_g1(vec3 w, real alpha)
{
    real tan2 = (w.x * w.x + w.y * w.y) / (w.z * w.z);
    return R(2.0) / (R(1.0) + rsqrt_(R(1.0) + (alpha * alpha) * tan2));
}
/* GGX, sampling the distribution of visible normals (Heitz 2018), wi = reflect(wo, h).
 * weight = F_schlick(F0 = albedo, wo.h) * G1(wi)  (separable Smith; G2/G1(wo) = G1(wi)).
 * Returns 0 if the reflected direction is not in the upper hemisphere. */
static int sample_ggx(const shadept* s, real u1, real u2, vec3* wi, real weight[3])
{
    real al = s->rough; vec3 wo = s->wo;
    vec3 vh = v3(al * wo.x, al * wo.y, wo.z);
    real vl = rsqrt_(vdot(vh, vh)); vh = v3(vh.x / vl, vh.y / vl, vh.z / vl);
    real lensq = vh.x * vh.x + vh.y * vh.y;
    vec3 T1 = v3(R(1.0), R(0.0), R(0.0));
    if (lensq > R(0.0)) { real il = rsqrt_(lensq); T1 = v3(-vh.y / il, vh.x / il, R(0.0)); }
    vec3 T2 = vcross(vh, T1);
    real r = rsqrt_(u1), sn, cs; sincos2pi(u2, &sn, &cs);
    real t1 = r * cs, t2 = r * sn;
    real sh = R(0.5) * (R(1.0) + vh.z);
    t2 = (R(1.0) - sh) * rsqrt_(rmax_(R(0.0), R(1.0) - t1 * t1)) + sh * t2;
    real t3 = rsqrt_(rmax_(R(0.0), (R(1.0) - t1 * t1) - t2 * t2));
    vec3 nh = v3((t1 * T1.x + t2 * T2.x) + t3 * vh.x, (t1 * T1.y + t2 * T2.y) + t3 * vh.y, (t1 * T1.z + t2 * T2.z) + t3 * vh.z);
    vec3 h = v3(al * nh.x, al * nh.y, rmax_(R(0.0), nh.z));
    real hl = rsqrt_(vdot(h, h)); h = v3(h.x / hl, h.y / hl, h.z / hl);
    real woh = vdot(wo, h);
    real two = R(2.0) * woh;
    *wi = v3(two * h.x - wo.x, two * h.y - wo.y, two * h.z - wo.z);
    if (!(wi->z > R(0.0))) return 0;
    real g1 = smith_g1(*wi, al);
    real c1 = R(1.0) - woh; if (c1 < R(0.0)) c1 = R(0.0);
    real c2 = c1 * c1, c5 = (c2 * c2) * c1;
    for (int k = 0; k < 3; ++k) weight[k] = (s->albedo[k] + (R(1.0) - s->albedo[k]) * c5) * g1;
    return 1;
}
/* GGX weight of a GIVEN exit direction wi (wi.z > 0) under the member's own material: the same F * G1(wi) as when the
 * direction was sampled from the visible normals, with h = normalize(wo + wi) ("calculating the probability based on the
 * direction and their respective materials").  Returns 0 if wo + wi vanishes. */
static int ggx_weight(const shadept* s, vec3 wi, real weight[3])
{
    vec3 h = v3(s->wo.x + wi.x, s->wo.y + wi.y, s->wo.z + wi.z);
    real hl = rsqrt_(vdot(h, h));
    if (!(hl > R(0.0))) return 0;
    h = v3(h.x / hl, h.y / hl, h.z / hl);
    real woh = vdot(s->wo, h);
    real g1 = smith_g1(wi, s->rough);
    real c1 = R(1.0) - woh; if (c1 < R(0.0)) c1 = R(0.0);
    real c2 = c1 * c1, c5 = (c2 * c2) * c1;
    for (int k = 0; k < 3; ++k) weight[k] = (s->albedo[k] + (R(1.0) - s->albedo[k]) * c5) * g1;
    return 1;
}
/* a glossy or specular member samples from its own stream ("undergo no processing") */
static void sample_own_glossy(const orc_frame* f, int32_t bounce, shadept* s, int32_t path)
{
    real u1, u2; bsdf_uniforms(f, s->pixel, s->sample, bounce, &u1, &u2);
    if (s->mtype == MAT_SPECULAR) {
        s->wi = v3(-s->wo.x, -s->wo.y, s->wo.z); s->has_dir = 1;
        for (int k = 0; k < 3; ++k) s->weight[k] = s->albedo[k];
    } else {
        s->has_dir = sample_ggx(s, u1, u2, &s->wi, s->weight);
    }
    s->dir_src = path;
}

/* ------------------------------------------------------------------ Morton code + sort (P:L43 [AK10]; D:R12)
 * 30 bits: 5 per component, origin bit before direction bit at every level. */
static uint32_t quant5(real x) { real fl = rfloor_(x); int q = (fl < R(0.0)) ? 0 : ((fl > R(31.0)) ? 31 : (int)fl); if (x != x) q = 0; return (uint32_t)q; }
uint32_t orc_morton_code(const orc_ray* r, const float* bounds)
{
    if (r->tmax < 0.f) return 0xFFFFFFFFu;
    uint32_t q[6];
    const float o[3] = { r->ox, r->oy, r->oz }, d[3] = { r->dx, r->dy, r->dz };
    for (int k = 0; k < 3; ++k) {
        real ext = R(bounds[3 + k]) - R(bounds[k]);
        real scale = ext > R(0.0) ? R(32.0) / ext : R(0.0);
        q[k] = quant5((R(o[k]) - R(bounds[k])) * scale);
        q[3 + k] = quant5((R(d[k]) + R(1.0)) * R(16.0));
    }
    uint32_t code = 0;
    for (int l = 0; l < 5; ++l)
        for (int k = 0; k < 6; ++k)
            code |= ((q[k] >> l) & 1u) << (6 * l + (5 - k));
    return code;
}
void orc_morton_encode(const orc_ray* rays, int64_t n, const float* bounds, uint32_t* keys)
{
    for (int64_t i = 0; i < n; ++i) keys[i] = orc_morton_code(&rays[i], bounds);
}

/* ---- the other sort keys of the paper's comparison (section 2.1, section 4; D:R19), all 30 bits.
 *   1 Origin    Morton code of the ray origin alone, 10 bits per axis (x above y above z at every level)
 *   2 Reis      "the higher bits represent the origin and subsequent bits represent the direction" [RCP17]: 15-bit
 *               Morton code of the origin (5 bits per axis) above the 15-bit Morton code of the direction
 *   3 Costa     "the opposite approach, where higher bits represented the direction" [CPJ15]: direction above origin
 *   4 TwoPoint  "interleaved bits from the origin and termination point" [MBK*10, MBGB20] with the fixed-length
 *               estimate of P:L139: end = o + (0.25 * largest extent of the scene box) * d, quantised like the origin
 *               (clamped into the box), in AilaCompact's bit layout with the end point in place of the direction
 * Quantisation of origin and direction components is AilaCompact's (D:R12): separate fp32 multiply and add/subtract. */
static uint32_t quant10(real x) { real fl = rfloor_(x); int q = (fl < R(0.0)) ? 0 : ((fl > R(1023.0)) ? 1023 : (int)fl); if (x != x) q = 0; return (uint32_t)q; }
static uint32_t morton3(uint32_t x, uint32_t y, uint32_t z, int bits)
{
    uint32_t c = 0;
    for (int l = 0; l < bits; ++l)
        c |= (((x >> l) & 1u) << (3 * l + 2)) | (((y >> l) & 1u) << (3 * l + 1)) | (((z >> l) & 1u) << (3 * l));
    return c;
}
uint32_t orc_ray_code(int32_t code, const orc_ray* r, const float* bounds)
{
    if (code == 0) return orc_morton_code(r, bounds);
    if (r->tmax < 0.f) return 0xFFFFFFFFu;
    const float o[3] = { r->ox, r->oy, r->oz }, d[3] = { r->dx, r->dy, r->dz };
    real ext[3], maxext = R(0.0);
    for (int k = 0; k < 3; ++k) { ext[k] = R(bounds[3 + k]) - R(bounds[k]); if (ext[k] > maxext) maxext = ext[k]; }
    uint32_t qo[3], qd[3], qe[3], qo10[3];
    real len = R(0.25) * maxext;
    for (int k = 0; k < 3; ++k) {
        real scale5 = ext[k] > R(0.0) ? R(32.0) / ext[k] : R(0.0), scale10 = ext[k] > R(0.0) ? R(1024.0) / ext[k] : R(0.0);
        qo[k] = quant5((R(o[k]) - R(bounds[k])) * scale5);
        qo10[k] = quant10((R(o[k]) - R(bounds[k])) * scale10);
        qd[k] = quant5((R(d[k]) + R(1.0)) * R(16.0));
        real e = R(o[k]) + len * R(d[k]);
        qe[k] = quant5((e - R(bounds[k])) * scale5);
    }
    switch (code) {
    case 1: return morton3(qo10[0], qo10[1], qo10[2], 10);
    case 2: return (morton3(qo[0], qo[1], qo[2], 5) << 15) | morton3(qd[0], qd[1], qd[2], 5);
    case 3: return (morton3(qd[0], qd[1], qd[2], 5) << 15) | morton3(qo[0], qo[1], qo[2], 5);
    default: {
        uint32_t q[6] = { qo[0], qo[1], qo[2], qe[0], qe[1], qe[2] }, c = 0;
        for (int l = 0; l < 5; ++l) for (int k = 0; k < 6; ++k) c |= ((q[k] >> l) & 1u) << (6 * l + (5 - k));
        return c; }
    }
}
void orc_ray_code_encode(int32_t code, const orc_ray* rays, int64_t n, const float* bounds, uint32_t* keys)
{
    for (int64_t i = 0; i < n; ++i) keys[i] = orc_ray_code(code, &rays[i], bounds);
}
typedef struct { uint32_t key; int32_t idx; } kv;
static int kv_cmp(const void* a, const void* b)
{
    const kv* x = (const kv*)a; const kv* y = (const kv*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx ? 1 : 0);
}
/* stable ascending sort of (key, index): order[j] = index of the j-th ray */
void orc_sort_keys(const uint32_t* keys, int64_t n, int32_t* order)
{
    kv* a = (kv*)malloc(sizeof(kv) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < n; ++i) { a[i].key = keys[i]; a[i].idx = (int32_t)i; }
    qsort(a, (size_t)n, sizeof(kv), kv_cmp);     /* total order on (key, idx) == stable sort by key */
    for (int64_t i = 0; i < n; ++i) order[i] = a[i].idx;
    free(a);
}

/* ------------------------------------------------------------------ secondary-ray generation
 * (P:L95-113 sections 3.2, 3.3; D:R3-R9, R13).  Outputs are in the mode's slot order:
 *   independent   slot = path id (row-major)
 *   direct_reuse  slot = (sample*n_tiles + tile)*M + m  (group-major; group = K consecutive slots)
 *   morton        independent rays, stably sorted by their 30-bit code
 * local_dir_out (optional, float[n_slots][3]) = tangent-space direction per output slot. */
void orc_generate_secondary(const float* verts, const int32_t* mat_id, const orc_material* mats, const orc_frame* f,
                            int32_t bounce, int32_t mode, int32_t gw, int32_t gh, int32_t s, const float* bounds,
                            const orc_ray* prev_rays, const orc_hit* prev_hits, const int32_t* prev_ray_to_path,
                            orc_path* paths, orc_ray* rays_out, int32_t* ray_to_path_out, int32_t* group_id_out,
                            int32_t* dir_src_out, uint8_t* group_class_out, uint32_t* n_active_out, float* local_dir_out)
{
    layout L = make_layout(f, mode, gw, gh, s);
    int64_t n_groups = L.n_slots / L.K;
    shadept* sp = (shadept*)calloc((size_t)L.n_paths, sizeof(shadept));
    /* 1. shading point of every live path (pixel <-> shading point) */
    for (int64_t i = 0; i < L.n_slots; ++i) {
        int32_t p = prev_ray_to_path[i];
        if (p < 0) continue;
        shadept* q = &sp[p];
        q->pixel = p % (f->w * f->h); q->sample = p / (f->w * f->h); q->dir_src = -1;
        if (!(paths[p].flags & PATH_ALIVE) || prev_rays[i].tmax < 0.f || prev_hits[i].prim < 0) { paths[p].flags &= ~PATH_ALIVE; continue; }
        if (!shading_point(verts, mat_id, mats, &prev_rays[i], &prev_hits[i], q)) { paths[p].flags &= ~PATH_ALIVE; continue; }
        q->live = 1;
    }
    /* 2. slot layout of this mode; the partition is per (tile, sample, frame), the same at every bounce (D:R4) */
    int32_t* path_of_slot = (int32_t*)malloc(sizeof(int32_t) * (size_t)L.n_slots);
    partition(f, &L, IS_GROUPED(mode) ? MODE_REUSE : MODE_INDEPENDENT, path_of_slot);
    /* 3. group rules */
    for (int64_t g = 0; g < n_groups; ++g) {
        int64_t base = g * L.K;
        int n_diff = 0, n_gloss = 0;
        for (int j = 0; j < L.K; ++j) {
            int32_t p = path_of_slot[base + j];
            if (p < 0 || !sp[p].live) continue;
            if (sp[p].mtype == MAT_DIFFUSE) ++n_diff; else ++n_gloss;
        }
        int cls = (n_diff + n_gloss == 0) ? CLASS_EMPTY : (n_gloss == 0 ? CLASS_DIFFUSE : (n_diff == 0 ? CLASS_GLOSSY : CLASS_HYBRID));
        group_class_out[g] = (uint8_t)cls;
        if (cls == CLASS_EMPTY) continue;
        if (mode == MODE_WORLD) {
            /* "Direct Direction Reusing" in WORLD space (section 3.1; DESIGN.md D:R18): one randomly selected pixel of the
             * group samples a direction from its own BSDF; the other rays reuse it in world space and weight it with their
             * own material.  A direction below a member's horizon ends that path (the artifact of Fig. 1).  Mirror
             * members cannot evaluate an arbitrary direction (delta lobe) and keep their own reflection. */
            uint32_t r[4];
            int32_t sample = (int32_t)(g / ((int64_t)L.n_tiles * L.G));
            orc_philox((uint32_t)g, (uint32_t)sample, (uint32_t)bounce, PURPOSE_LEADER, (uint32_t)f->seed, (uint32_t)f->frame, r);
            int j0 = (int)(r[0] % (uint32_t)L.K); int32_t leader = -1;
            for (int t = 0; t < L.K && leader < 0; ++t) {
                int32_t p = path_of_slot[base + (j0 + t) % L.K];
                if (p >= 0 && sp[p].live) leader = p;
            }
            /* every live member first takes its own independent sample (the leader's is the shared one; the others keep
             * theirs only if they are mirrors or the leader's sample is invalid) */
            for (int j = 0; j < L.K; ++j) {
                int32_t p = path_of_slot[base + j];
                if (p < 0 || !sp[p].live) continue;
                if (sp[p].mtype == MAT_DIFFUSE) {
                    real u1, u2; bsdf_uniforms(f, sp[p].pixel, sp[p].sample, bounce, &u1, &u2);
                    sp[p].wi = sample_cosine(u1, u2); sp[p].has_dir = 1; sp[p].dir_src = p;
                    for (int k = 0; k < 3; ++k) sp[p].weight[k] = sp[p].albedo[k];
                } else sample_own_glossy(f, bounce, &sp[p], p);
            }
            if (!sp[leader].has_dir) continue;
            vec3 wd = to_world(&sp[leader], sp[leader].wi);
            for (int j = 0; j < L.K; ++j) {
                int32_t p = path_of_slot[base + j];
                if (p < 0 || !sp[p].live || p == leader || sp[p].mtype == MAT_SPECULAR) continue;
                vec3 wl = to_local(&sp[p], wd);
                sp[p].dir_src = leader;
                if (!(wl.z > R(0.0))) { sp[p].has_dir = 0; continue; }
                sp[p].wi = wl; sp[p].has_wdir = 1; sp[p].wdir = wd; sp[p].has_dir = 1;
                if (sp[p].mtype == MAT_DIFFUSE) { for (int k = 0; k < 3; ++k) sp[p].weight[k] = sp[p].albedo[k]; }
                else sp[p].has_dir = ggx_weight(&sp[p], wl, sp[p].weight);
            }
            continue;
        }
        /* glossy / specular members: untouched, in glossy AND hybrid groups */
        vec3 sum = v3(R(0.0), R(0.0), R(0.0)); int n_valid = 0;
        for (int j = 0; j < L.K; ++j) {
            int32_t p = path_of_slot[base + j];
            if (p < 0 || !sp[p].live || sp[p].mtype == MAT_DIFFUSE) continue;
            sample_own_glossy(f, bounce, &sp[p], p);
            if (sp[p].has_dir) { sum = v3(sum.x + sp[p].wi.x, sum.y + sp[p].wi.y, sum.z + sp[p].wi.z); ++n_valid; }   /* ascending slot order */
        }
        if (n_diff == 0) continue;
        if (cls == CLASS_HYBRID && n_valid > 0) {
            /* hybrid: diffuse members take the average tangent-space exit direction of the
             * glossy/specular members; own material's pdf => weight = albedo (D:R13) */
            real len = rsqrt_(vdot(sum, sum));
            vec3 avg = v3(sum.x / len, sum.y / len, sum.z / len);
            for (int j = 0; j < L.K; ++j) {
                int32_t p = path_of_slot[base + j];
                if (p < 0 || !sp[p].live || sp[p].mtype != MAT_DIFFUSE) continue;
                sp[p].wi = avg; sp[p].has_dir = 1; sp[p].dir_src = (int32_t)(-2 - g);
                for (int k = 0; k < 3; ++k) sp[p].weight[k] = sp[p].albedo[k];
            }
            continue;
        }
        /* diffuse group (or hybrid without a valid glossy sample): "randomly selects one pixel"
         * = first live diffuse member in cyclic slot order from j0 (D:R8); only the
         * selected ray samples a direction, the others reuse it in tangent space */
        uint32_t r[4];
        int32_t sample = (int32_t)(g / ((int64_t)L.n_tiles * L.G));
        orc_philox((uint32_t)g, (uint32_t)sample, (uint32_t)bounce, PURPOSE_LEADER, (uint32_t)f->seed, (uint32_t)f->frame, r);
        int j0 = (int)(r[0] % (uint32_t)L.K), leader = -1;
        for (int t = 0; t < L.K && leader < 0; ++t) {
            int32_t p = path_of_slot[base + (j0 + t) % L.K];
            if (p >= 0 && sp[p].live && sp[p].mtype == MAT_DIFFUSE) leader = p;
        }
        real u1, u2; bsdf_uniforms(f, sp[leader].pixel, sp[leader].sample, bounce, &u1, &u2);
        vec3 wi = sample_cosine(u1, u2);
        for (int j = 0; j < L.K; ++j) {
            int32_t p = path_of_slot[base + j];
            if (p < 0 || !sp[p].live || sp[p].mtype != MAT_DIFFUSE) continue;
            sp[p].wi = wi; sp[p].has_dir = 1; sp[p].dir_src = leader;
            for (int k = 0; k < 3; ++k) sp[p].weight[k] = sp[p].albedo[k];
        }
    }
    /* 4. emit rays in slot order; throughput *= weight */
    uint32_t n_active = 0;
    orc_ray* tmp_rays = rays_out; int32_t* tmp_r2p = ray_to_path_out; int32_t* tmp_src = dir_src_out; float* tmp_loc = local_dir_out;
    if (IS_SORTED(mode)) {
        tmp_rays = (orc_ray*)malloc(sizeof(orc_ray) * (size_t)L.n_slots); tmp_r2p = (int32_t*)malloc(4 * (size_t)L.n_slots);
        tmp_src = (int32_t*)malloc(4 * (size_t)L.n_slots); tmp_loc = (float*)malloc(12 * (size_t)L.n_slots);
    }
    for (int64_t i = 0; i < L.n_slots; ++i) {
        int32_t p = path_of_slot[i];
        tmp_r2p[i] = p; tmp_src[i] = -1; inactive_ray(&tmp_rays[i]);
        if (tmp_loc) tmp_loc[3 * i] = tmp_loc[3 * i + 1] = tmp_loc[3 * i + 2] = 0.f;
        if (IS_GROUPED(mode)) group_id_out[i] = (int32_t)(i / L.K);
        if (p < 0 || !sp[p].live) continue;
        shadept* q = &sp[p];
        if (!q->has_dir) { paths[p].flags &= ~PATH_ALIVE; continue; }       /* invalid glossy sample: path ends */
        vec3 wd = q->has_wdir ? q->wdir : to_world(q, q->wi);
        real mx = rmax_(rabs_(q->p.x), rmax_(rabs_(q->p.y), rabs_(q->p.z)));
        real off = R(1.0 / 32768.0) * (R(1.0) + mx);                        /* self-intersection offset (D:R7) */
        orc_ray* o = &tmp_rays[i];
        o->ox = (float)(q->p.x + q->ng.x * off); o->oy = (float)(q->p.y + q->ng.y * off); o->oz = (float)(q->p.z + q->ng.z * off);
        o->dx = (float)wd.x; o->dy = (float)wd.y; o->dz = (float)wd.z; o->tmin = 0.f; o->tmax = 1e30f;
        paths[p].tr = (float)(R(paths[p].tr) * q->weight[0]); paths[p].tg = (float)(R(paths[p].tg) * q->weight[1]); paths[p].tb = (float)(R(paths[p].tb) * q->weight[2]);
        tmp_src[i] = q->dir_src;
        if (tmp_loc) { tmp_loc[3 * i] = (float)q->wi.x; tmp_loc[3 * i + 1] = (float)q->wi.y; tmp_loc[3 * i + 2] = (float)q->wi.z; }
        ++n_active;
    }
    if (IS_SORTED(mode)) {
        /* reordering baseline: encode, sort, permute */
        uint32_t* keys = (uint32_t*)malloc(4 * (size_t)L.n_slots); int32_t* order = (int32_t*)malloc(4 * (size_t)L.n_slots);
        orc_ray_code_encode(CODE_OF_MODE(mode), tmp_rays, L.n_slots, bounds, keys);
        orc_sort_keys(keys, L.n_slots, order);
        for (int64_t j = 0; j < L.n_slots; ++j) {
            int32_t i = order[j];
            rays_out[j] = tmp_rays[i]; ray_to_path_out[j] = tmp_r2p[i]; dir_src_out[j] = tmp_src[i];
            if (local_dir_out) memcpy(local_dir_out + 3 * j, tmp_loc + 3 * (int64_t)i, 12);
        }
        free(keys); free(order); free(tmp_rays); free(tmp_r2p); free(tmp_src); free(tmp_loc);
    }
    if (!IS_GROUPED(mode)) for (int64_t j = 0; j < L.n_slots; ++j) group_id_out[j] = ray_to_path_out[j];
    *n_active_out = n_active;
    free(path_of_slot); free(sp);
}

/* ------------------------------------------------------------------ shading / accumulation (D:R14)
 * Emission on hit, environment on miss, no next-event estimation, no Russian roulette.
 * bounce = index of the segment just traced (0 = primary).  At the last segment every
 * path adds its radiance / spp to its pixel. */
void orc_paths_init(orc_path* paths, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) { paths[i].tr = paths[i].tg = paths[i].tb = 1.f; paths[i].flags = PATH_ALIVE; paths[i].lr = paths[i].lg = paths[i].lb = 0.f; paths[i].pad = 0; }
}
void orc_shade_accumulate(const int32_t* mat_id, const orc_material* mats, const float* env, const orc_frame* f, int32_t bounce, int32_t is_last,
                          const orc_ray* rays, const orc_hit* hits, const int32_t* ray_to_path, int64_t n_rays, orc_path* paths, float* accum)
{
    (void)bounce;
    for (int64_t i = 0; i < n_rays; ++i) {
        int32_t p = ray_to_path[i];
        if (p < 0) continue;
        orc_path* ps = &paths[p];
        if ((ps->flags & PATH_ALIVE) && rays[i].tmax >= 0.f) {
            real T[3] = { R(ps->tr), R(ps->tg), R(ps->tb) }, Le[3]; int ends = 0;
            if (hits[i].prim < 0) {
                real w = R(0.5) * (R(rays[i].dy) + R(1.0));
                for (int k = 0; k < 3; ++k) Le[k] = R(env[k]) + (R(env[3 + k]) - R(env[k])) * w;
                ends = 1;
            } else {
                const orc_material* m = &mats[mat_id[hits[i].prim]];
                if (m->type == MAT_EMISSIVE) { for (int k = 0; k < 3; ++k) Le[k] = R(m->emission[k]); ends = 1; }
            }
            if (ends) {
                ps->lr = (float)(R(ps->lr) + T[0] * Le[0]); ps->lg = (float)(R(ps->lg) + T[1] * Le[1]); ps->lb = (float)(R(ps->lb) + T[2] * Le[2]);
                ps->flags &= ~PATH_ALIVE;
            }
        }
        if (is_last) {
            int32_t pix = p % (f->w * f->h);
            real inv = R(1.0) / R(f->spp);
            accum[3 * pix + 0] = (float)(R(accum[3 * pix + 0]) + R(ps->lr) * inv);
            accum[3 * pix + 1] = (float)(R(accum[3 * pix + 1]) + R(ps->lg) * inv);
            accum[3 * pix + 2] = (float)(R(accum[3 * pix + 2]) + R(ps->lb) * inv);
        }
    }
}

/* ------------------------------------------------------------------ one whole frame (call sequence of DESIGN.md section 2)
 * primary -> shade(0) -> for b = 1..B { generate(b) -> trace -> shade(b) }.
 * times[0..3] += seconds in generate(+encode+sort), trace (secondary), shade, primary;
 * counts[0] += live secondary rays, counts[1..2] += node visits / triangle tests of secondary rays. */
static double now_s(void) { struct timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); return ts.tv_sec + 1e-9 * ts.tv_nsec; }
void orc_render_frame(const orc_bvh* b, const int32_t* mat_id, const orc_material* mats, const float* env, const float* cam,
                      const orc_frame* f, int32_t n_bounces, int32_t mode, int32_t gw, int32_t gh, int32_t s,
                      float* accum, double* times, int64_t* counts)
{
    layout L = make_layout(f, mode, gw, gh, s);
    size_t ns = (size_t)L.n_slots;
    orc_ray* rays[2] = { (orc_ray*)malloc(sizeof(orc_ray) * ns), (orc_ray*)malloc(sizeof(orc_ray) * ns) };
    orc_hit* hits = (orc_hit*)malloc(sizeof(orc_hit) * ns);
    int32_t* r2p[2] = { (int32_t*)malloc(4 * ns), (int32_t*)malloc(4 * ns) };
    int32_t* gid = (int32_t*)malloc(4 * ns); int32_t* src = (int32_t*)malloc(4 * ns);
    uint8_t* cls = (uint8_t*)malloc(ns);
    orc_path* paths = (orc_path*)malloc(sizeof(orc_path) * (size_t)L.n_paths);
    float bounds[6] = { b->root_min[0], b->root_min[1], b->root_min[2], b->root_max[0], b->root_max[1], b->root_max[2] };
    orc_paths_init(paths, L.n_paths);
    double t0 = now_s();
    orc_trace_primary(b, cam, f, mode, gw, gh, s, rays[0], hits, r2p[0]);
    double t1 = now_s(); times[3] += t1 - t0;
    orc_shade_accumulate(mat_id, mats, env, f, 0, n_bounces == 0, rays[0], hits, r2p[0], L.n_slots, paths, accum);
    double t2 = now_s(); times[2] += t2 - t1;
    int cur = 0;
    for (int32_t bn = 1; bn <= n_bounces; ++bn) {
        uint32_t n_active = 0;
        t0 = now_s();
        orc_generate_secondary(b->verts, mat_id, mats, f, bn, mode, gw, gh, s, bounds, rays[cur], hits, r2p[cur], paths,
                               rays[1 - cur], r2p[1 - cur], gid, src, cls, &n_active, NULL);
        cur = 1 - cur;
        t1 = now_s(); times[0] += t1 - t0;
        orc_trace(b, rays[cur], L.n_slots, hits, counts + 1);
        t2 = now_s(); times[1] += t2 - t1;
        orc_shade_accumulate(mat_id, mats, env, f, bn, bn == n_bounces, rays[cur], hits, r2p[cur], L.n_slots, paths, accum);
        times[2] += now_s() - t2;
        counts[0] += n_active;
    }
    free(rays[0]); free(rays[1]); free(hits); free(r2p[0]); free(r2p[1]); free(gid); free(src); free(cls); free(paths);
}

/* ------------------------------------------------------------------ test entry points (sampling routines alone) */
void orc_test_sample_cosine(float u1, float u2, float* wi)
{
    vec3 w = sample_cosine(R(u1), R(u2)); wi[0] = (float)w.x; wi[1] = (float)w.y; wi[2] = (float)w.z;
}
/* albedo = 1 (so F = 1 and weight = G1(wi)); returns validity */
int32_t orc_test_sample_ggx(const float* wo, float alpha, float u1, float u2, float* wi, float* weight)
{
    shadept s; memset(&s, 0, sizeof s);
    s.wo = v3(R(wo[0]), R(wo[1]), R(wo[2])); s.rough = R(alpha); s.albedo[0] = s.albedo[1] = s.albedo[2] = R(1.0);
    vec3 w; real wt[3];
    int ok = sample_ggx(&s, R(u1), R(u2), &w, wt);
    wi[0] = (float)w.x; wi[1] = (float)w.y; wi[2] = (float)w.z; weight[0] = (float)wt[0];
    return ok;
}
/* the same with a given F0 = albedo (RGB), so that the Schlick factor is exercised; returns validity, weight[3] */
int32_t orc_test_sample_ggx_f0(const float* wo, float alpha, const float* albedo, float u1, float u2, float* wi, float* weight)
{
    shadept s; memset(&s, 0, sizeof s);
    s.wo = v3(R(wo[0]), R(wo[1]), R(wo[2])); s.rough = R(alpha);
    for (int k = 0; k < 3; ++k) s.albedo[k] = R(albedo[k]);
    vec3 w; real wt[3] = { R(0.0), R(0.0), R(0.0) };
    int ok = sample_ggx(&s, R(u1), R(u2), &w, wt);
    wi[0] = (float)w.x; wi[1] = (float)w.y; wi[2] = (float)w.z;
    for (int k = 0; k < 3; ++k) weight[k] = (float)wt[k];
    return ok;
}
/* ggx_weight (world-space reuse, D:R18) alone: weight[3] of a GIVEN exit direction wi; returns validity */
int32_t orc_test_ggx_weight(const float* wo, const float* wi, float alpha, const float* albedo, float* weight)
{
    shadept s; memset(&s, 0, sizeof s);
    s.wo = v3(R(wo[0]), R(wo[1]), R(wo[2])); s.rough = R(alpha);
    for (int k = 0; k < 3; ++k) s.albedo[k] = R(albedo[k]);
    real wt[3] = { R(0.0), R(0.0), R(0.0) };
    int ok = ggx_weight(&s, v3(R(wi[0]), R(wi[1]), R(wi[2])), wt);
    for (int k = 0; k < 3; ++k) weight[k] = (float)wt[k];
    return ok;
}
