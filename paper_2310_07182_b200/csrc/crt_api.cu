// C ABI of libcrt (include/crt.h): argument checking, BVH upload, and the per-frame call sequence.
#include <algorithm>
#include <chrono>
#include <cstring>
#include <thread>
#include "crt_internal.h"

bool crt_bvh_build_host(crt_bvh* b, const float* verts, int64_t n, const crt_bvh_params& pr, bool presplit_single = false);
int32_t crt_bvh_check_host(const crt_bvh* b);
void crt_bvh_flatten(const crt_bvh* b, const std::vector<int32_t>& tri_order, std::vector<GpuNode>& gn, std::vector<GpuTri>& gt, std::vector<int32_t>& slot_of_prim);
int32_t crt_bvh_quantise(const crt_bvh* b, const std::vector<GpuNode>& gn, std::vector<QNode>& qn, QGrid* grid, double* inflation);
void crt_bvh_collapse4(const std::vector<GpuNode>& gn, const std::vector<QNode>& qn, std::vector<QNode>& q4);
void crt_bvh_build_wide(const crt_bvh* b, std::vector<WNode>& wn, std::vector<int32_t>& tri_order, int* depth_out);
int32_t crt_bvh_check_wide(const crt_bvh* b, const std::vector<WNode>& wn, const std::vector<int32_t>& tri_order);

static thread_local std::string g_last_error;

crt_status crt_fail(crt_ctx* ctx, crt_status st, const char* fmt, ...)
{
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    if (ctx) ctx->last_error = buf;
    g_last_error = buf;
    return st;
}

static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
static bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

crt_status crt_make_layout(crt_ctx* ctx, const crt_frame* f, const crt_order* o, Layout* L)
{
    if (!f || !o || !L) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "layout: null argument");
    if (f->w < 0 || f->h < 0 || f->spp < 1) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "layout: bad frame %dx%d spp %d", f->w, f->h, f->spp);
    if (o->mode < 0 || o->mode > CRT_MODE_SORT_TWOPOINT) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "layout: mode %d out of range", o->mode);
    memset(L, 0, sizeof *L);
    L->w = f->w; L->h = f->h; L->spp = f->spp; L->mode = o->mode;
    L->n_paths = (int64_t)f->spp * f->w * f->h;
    if (L->n_paths >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "layout: more than 2^31 paths");
    if (o->mode != CRT_MODE_DIRECT_REUSE && o->mode != CRT_MODE_WORLD_REUSE) {
        L->W = L->H = L->M = L->K = L->G = 1; L->tiles_x = f->w; L->tiles_y = f->h; L->n_tiles = f->w * f->h;
        L->n_slots = L->n_paths; L->n_groups = L->n_paths;
        return CRT_OK;
    }
    const int sy = o->stride_y ? o->stride_y : o->stride;
    if (!is_pow2(o->group_w) || !is_pow2(o->group_h) || !is_pow2(o->stride) || !is_pow2(sy) || o->stride > 4096 || sy > 4096 || o->group_w > 1024 || o->group_h > 1024)
        return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "layout: group %dx%d stride %d/%d must be powers of two", o->group_w, o->group_h, o->stride, sy);
    const int64_t M = (int64_t)o->group_w * o->stride * o->group_h * sy, K = (int64_t)o->group_w * o->group_h;
    if (M > 4096 || K > 1024) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "layout: tile of %lld slots / group of %lld exceeds 4096 / 1024", (long long)M, (long long)K);
    if (o->partition_rule < CRT_PARTITION_SHUFFLE || o->partition_rule > CRT_PARTITION_LCG_SEQUENCE) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "layout: partition_rule %d out of range", o->partition_rule);
    L->gw = o->group_w; L->sx = o->stride; L->sy = sy; L->lattice = o->partition_rule;       // 0 shuffle (affine), 1 lattice, 2 LCG sequence
    L->W = o->group_w * o->stride; L->H = o->group_h * sy; L->M = (int)M; L->K = (int)K; L->G = (int)(M / K);
    L->log2W = ilog2(L->W); L->log2M = ilog2(L->M); L->log2K = ilog2(L->K);
    L->tiles_x = (f->w + L->W - 1) / L->W; L->tiles_y = (f->h + L->H - 1) / L->H; L->n_tiles = L->tiles_x * L->tiles_y;
    L->n_slots = (int64_t)f->spp * L->n_tiles * L->M; L->n_groups = L->n_slots / L->K;
    if (L->n_slots >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "layout: more than 2^31 slots");
    return CRT_OK;
}

// The 4-wide form of the 16-bit nodes (trace_kernel 7) is built on first use, from the device's own binary layouts: an alternative kernel should not cost
// every BVH 14-164 MB.  Returns false when it cannot exist (tree too deep for the stack with three pushes per visit, wide triangle order, no 16-bit nodes).
bool crt_bvh_ensure_q4(const crt_bvh* cb)
{
    crt_bvh* b = const_cast<crt_bvh*>(cb);
    if (b->d_q4nodes) return true;
    if (!b->d_nodes || !b->d_qnodes || b->d_wnodes || b->n_gpu_nodes < 1 || (b->depth + 1) / 2 * 3 + 2 > 64) return false;
    std::vector<GpuNode> gn((size_t)b->n_gpu_nodes); std::vector<QNode> qn((size_t)b->n_gpu_nodes), q4;
    if (cudaMemcpy(gn.data(), b->d_nodes, gn.size() * sizeof(GpuNode), cudaMemcpyDeviceToHost) != cudaSuccess) return false;
    if (cudaMemcpy(qn.data(), b->d_qnodes, qn.size() * sizeof(QNode), cudaMemcpyDeviceToHost) != cudaSuccess) return false;
    crt_bvh_collapse4(gn, qn, q4);
    if (cudaMalloc((void**)&b->d_q4nodes, q4.size() * sizeof(QNode)) != cudaSuccess) { b->d_q4nodes = nullptr; return false; }
    if (cudaMemcpy(b->d_q4nodes, q4.data(), q4.size() * sizeof(QNode), cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(b->d_q4nodes); b->d_q4nodes = nullptr; return false; }
    b->n_q4_nodes = (int64_t)q4.size() / 2; b->device_bytes += (int64_t)(q4.size() * sizeof(QNode));
    return true;
}

extern "C" {

crt_status crt_create(int32_t device, crt_ctx** out)
{
    if (!out) return crt_fail(nullptr, CRT_ERR_INVALID_ARG, "crt_create: out is null");
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count == 0) return crt_fail(nullptr, CRT_ERR_CUDA, "crt_create: no CUDA device (%s); libcrt has no CPU fallback", cudaGetErrorString(e));
    if (device < 0 || device >= count) return crt_fail(nullptr, CRT_ERR_INVALID_ARG, "crt_create: device %d out of range [0,%d)", device, count);
    CRT_CUDA(nullptr, cudaSetDevice(device));
    cudaDeviceProp prop;
    CRT_CUDA(nullptr, cudaGetDeviceProperties(&prop, device));
    if (prop.major < 10) return crt_fail(nullptr, CRT_ERR_UNSUPPORTED, "crt_create: device is sm_%d%d; libcrt is built for sm_100a only", prop.major, prop.minor);
    radix_sort_noalloc_setup(device);      // address of the static scratch of crt_radix_sort_pairs_noalloc on this device (sort.cu); not fatal here
    crt_ctx* c = new crt_ctx();
    c->device = device; c->n_sms = prop.multiProcessorCount;
    if (cudaMalloc(&c->d_counter, 4096) != cudaSuccess) { delete c; return crt_fail(nullptr, CRT_ERR_NOMEM, "crt_create: cudaMalloc failed"); }
    *out = c;
    return CRT_OK;
}

crt_status crt_destroy(crt_ctx* ctx)
{
    if (!ctx) return CRT_OK;
    CrtDeviceGuard dev_guard_(ctx->device);
    cudaFree(ctx->d_counter);
    for (cudaEvent_t ev : ctx->ev) cudaEventDestroy(ev);
    for (int k = 0; k < 4; ++k) { if (ctx->band_stream[k]) cudaStreamDestroy(ctx->band_stream[k]); if (ctx->band_join[k]) cudaEventDestroy(ctx->band_join[k]); }
    if (ctx->band_fork) cudaEventDestroy(ctx->band_fork);
    delete ctx;
    return CRT_OK;
}

const char* crt_last_error(const crt_ctx* ctx) { return ctx ? ctx->last_error.c_str() : g_last_error.c_str(); }

crt_status crt_set_option(crt_ctx* ctx, const char* key, int64_t value)
{
    if (!ctx || !key) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "set_option: null argument");
    if (!strcmp(key, "trace_kernel")) { if (value < 0 || value > 9) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_kernel must be 0..9"); ctx->trace_kernel = (int)value; }
    else if (!strcmp(key, "trace_refill_threshold")) { if (value < 0 || value > 32) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_refill_threshold out of range"); ctx->trace_refill_threshold = (int)value; }
    else if (!strcmp(key, "trace_leaf_wait")) { if (value < 0 || value > 31) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_leaf_wait out of range"); ctx->trace_leaf_wait = (int)value; }
    else if (!strcmp(key, "trace_tri_wait")) { if (value < 0 || value > 32) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_tri_wait out of range"); ctx->trace_tri_wait = (int)value; }
    else if (!strcmp(key, "fuse_shade")) { ctx->fuse_shade = value != 0; }
    else if (!strcmp(key, "trace_exact")) { ctx->trace_exact = value != 0; }
    else if (!strcmp(key, "trace_tail_split")) { ctx->trace_tail_split = value != 0; }
    else if (!strcmp(key, "shade_pixel_order")) { ctx->shade_pixel_order = value != 0; }
    else if (!strcmp(key, "frame_bands")) { if (value < 1 || value > 4) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "frame_bands must be 1..4"); ctx->frame_bands = (int)value; }
    else if (!strcmp(key, "trace_blocks_per_sm")) { if (value < 0 || value > 32) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_blocks_per_sm out of range"); ctx->trace_blocks_per_sm = (int)value; }
    else return crt_fail(ctx, CRT_ERR_INVALID_ARG, "set_option: unknown key '%s'", key);
    return CRT_OK;
}

crt_status crt_measure_peaks(crt_ctx* ctx, double* fp32_tflops, double* copy_gbs)
{
    if (!ctx || !fp32_tflops || !copy_gbs) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "measure_peaks: null argument");
    CrtDeviceGuard dev_guard_(ctx->device);
    return measure_peaks(ctx, fp32_tflops, copy_gbs);
}

// ---- BVH ----------------------------------------------------------------------------------------------
static bool is_device_ptr(const void* p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

crt_status crt_build_bvh(crt_ctx* ctx, const float* verts, const int32_t* mat_id, int64_t n_tris, const crt_bvh_params* params, crt_bvh** out)
{
    if (!out) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: out is null");
    *out = nullptr;
    CrtDeviceGuard dev_guard_(ctx ? ctx->device : -1);
    if (n_tris < 0 || (n_tris > 0 && !verts)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: bad triangle array");
    if (n_tris >= ((int64_t)1 << 28)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "build_bvh: more than 2^28 triangles");
    crt_bvh_params pr = {3, 64, 1.0f, 1.0f, 0, 0, 0, 0.0625f, 20};
    if (params) pr = *params;
    if (pr.max_leaf < 1 || pr.max_leaf > 8) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: max_leaf %d not in [1,8]", pr.max_leaf);
    if (pr.sah_bins == 0) pr.sah_bins = 64;
    if (pr.optimize < 0 || pr.optimize > 10000) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: optimize %d not in [0,10000]", pr.optimize);
    if (!(pr.presplit >= 0.f && pr.presplit <= 1.f)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: presplit %g not in [0,1]", (double)pr.presplit);
    std::vector<float> hv; std::vector<int32_t> hm((size_t)n_tris, 0);
    const float* v = verts;
    if (ctx && n_tris > 0 && is_device_ptr(verts)) {
        hv.resize((size_t)n_tris * 9);
        CRT_CUDA(ctx, cudaMemcpy(hv.data(), verts, hv.size() * 4, cudaMemcpyDeviceToHost));
        v = hv.data();
    }
    if (mat_id && n_tris > 0) {
        if (ctx && is_device_ptr(mat_id)) CRT_CUDA(ctx, cudaMemcpy(hm.data(), mat_id, hm.size() * 4, cudaMemcpyDeviceToHost));
        else memcpy(hm.data(), mat_id, hm.size() * 4);
    }
    for (int64_t i = 0; i < 9 * n_tris; ++i) if (!(v[i] == v[i]) || v[i] > 1e30f || v[i] < -1e30f) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: non-finite vertex");
    int32_t max_mat = -1;
    for (int32_t m : hm) { if (m < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: negative material id"); max_mat = std::max(max_mat, m); }
    if (pr.builder < 0 || pr.builder > 3) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: builder %d out of range", pr.builder);
    if ((pr.builder == 1 || pr.builder == 2) && !ctx) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "build_bvh: the device builder needs a context");
    if (n_tris <= pr.max_leaf) pr.builder = 0;            // nothing to cluster: the whole scene is one leaf (or empty)
    crt_bvh* b = new crt_bvh();
    b->max_mat_id = max_mat;
    if (pr.builder == 1 || pr.builder == 2) {
        crt_status bst = crt_bvh_build_device(ctx, b, v, n_tris, pr, pr.builder == 1);
        if (bst != CRT_OK) { crt_bvh_destroy(b); return bst; }
    } else if (pr.builder == 0 && ctx && pr.optimize > 0) {
        // host build; its optimisation step runs on the device (parallel re-insertion, bvh_ploc.cu: every node looks for its best place in every iteration,
        // where the host's own version can afford the worst 2 % only)
        const auto t_opt0 = std::chrono::steady_clock::now();
        crt_bvh_params p0 = pr; p0.optimize = 0;
        // the tree is built and optimised with ONE reference per leaf, so that the re-insertion can move single triangles; subtrees of at most max_leaf
        // references are collapsed into leaves afterwards (interior scene: 8 % fewer triangle tests per ray, secondary traversal -2 %; profiles/r02o)
        const bool fine = pr.max_leaf > 1;
        if (fine) p0.max_leaf = 1;
        crt_bvh_build_host(b, v, n_tris, p0, fine);
        const crt_status rst = crt_bvh_reinsert_device(ctx, b, pr.optimize, fine ? pr.max_leaf : 0);
        if (rst != CRT_OK) { crt_bvh_destroy(b); return rst; }
        if (fine) b->max_leaf = pr.max_leaf;
        if (b->opt_iters > 0 || fine) {          // SAH cost of the new tree, on the unpadded boxes as crt_bvh_build_host reports it
            float maxabs = 0.f; for (int k = 0; k < 6; ++k) maxabs = std::max(maxabs, std::fabs(b->bounds[k]));
            const double pad2 = 2.0 * (double)(maxabs * (1.0f / 131072.0f));
            auto ha = [&](const BuildNode& x) { const double dx = (double)x.bmax[0] - x.bmin[0] - pad2, dy = (double)x.bmax[1] - x.bmin[1] - pad2, dz = (double)x.bmax[2] - x.bmin[2] - pad2; return dx * dy + dy * dz + dz * dx; };
            double cost = 0; for (const BuildNode& x : b->nodes) cost += ha(x) * (x.left >= 0 ? (double)pr.cost_traversal : (double)pr.cost_intersect * x.count);
            const double ra = b->nodes.empty() ? 0 : ha(b->nodes[0]);
            b->sah = ra > 0 ? cost / ra : 0;
        }
        b->build_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_opt0).count();
    } else { crt_bvh_build_host(b, v, n_tris, pr); b->builder = pr.builder == 3 ? 3 : 0; }
    const auto t_layout0 = std::chrono::steady_clock::now();
    if (b->depth > 60) { crt_bvh_destroy(b); return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "build_bvh: tree depth exceeds the traversal stack (64)"); }
    auto up = [&](void** d, const void* h, size_t bytes) -> cudaError_t {
        cudaError_t e = cudaMalloc(d, bytes ? bytes : 256);
        if (e != cudaSuccess) return e;
        b->device_bytes += (int64_t)bytes;
        return bytes ? cudaMemcpy(*d, h, bytes, cudaMemcpyHostToDevice) : cudaMemset(*d, 0, 256);      // empty scene: a defined (degenerate) record
    };
    if (pr.builder == 1) {
        // the device builder wrote the traversal layouts itself (bvh_ploc.cu); only the material ids remain
        cudaError_t e = up((void**)&b->d_mat_id, hm.data(), hm.size() * 4);
        if (e != cudaSuccess) { crt_bvh_destroy(b); return crt_fail(ctx, e == cudaErrorMemoryAllocation ? CRT_ERR_NOMEM : CRT_ERR_CUDA, "build_bvh: upload: %s", cudaGetErrorString(e)); }
    } else {
    // one triangle per leaf: also build the 8-wide compressed layout (the default kernel's); its triangle order is the shared one
    std::vector<WNode> wn; std::vector<int32_t> tri_order;
    if (pr.max_leaf == 1) {
        crt_bvh_build_wide(b, wn, tri_order, &b->wide_depth);
        b->n_wide_nodes = (int64_t)wn.size();
        b->wide_violations = crt_bvh_check_wide(b, wn, tri_order);
        if (b->wide_depth > 40) { crt_bvh_destroy(b); return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "build_bvh: wide tree depth %d exceeds the traversal stack", b->wide_depth); }
    }
    // traversal layouts (host vectors; built without a context too, so that crt_bvh_check / crt_bvh_get_info cover the 16-bit nodes)
    std::vector<GpuNode> gn; std::vector<GpuTri> gt; std::vector<int32_t> sop; std::vector<QNode> qn;
    crt_bvh_flatten(b, tri_order, gn, gt, sop);
    b->q_violations = crt_bvh_quantise(b, gn, qn, &b->qgrid, &b->q_inflation);
    if (ctx) {
        b->device = ctx->device; b->n_gpu_nodes = (int64_t)gn.size();
        cudaError_t e = up((void**)&b->d_nodes, gn.data(), gn.size() * sizeof(GpuNode));
        if (e == cudaSuccess) e = up((void**)&b->d_qnodes, qn.data(), qn.size() * sizeof(QNode));
        if (e == cudaSuccess) e = up((void**)&b->d_tris, gt.data(), gt.size() * sizeof(GpuTri));
        if (e == cudaSuccess && !wn.empty()) e = up((void**)&b->d_wnodes, wn.data(), wn.size() * sizeof(WNode));
        if (e == cudaSuccess) e = up((void**)&b->d_slot_of_prim, sop.data(), sop.size() * 4);
        if (e == cudaSuccess) e = up((void**)&b->d_mat_id, hm.data(), hm.size() * 4);
        if (e != cudaSuccess) { crt_bvh_destroy(b); return crt_fail(ctx, e == cudaErrorMemoryAllocation ? CRT_ERR_NOMEM : CRT_ERR_CUDA, "build_bvh: upload: %s", cudaGetErrorString(e)); }
    }
    }
    b->layout_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_layout0).count();
    *out = b;
    return CRT_OK;
}

crt_status crt_bvh_destroy(crt_bvh* b)
{
    if (!b) return CRT_OK;
    CrtDeviceGuard dev_guard_(b->device);
    cudaFree(b->d_nodes); cudaFree(b->d_qnodes); cudaFree(b->d_q4nodes); cudaFree(b->d_wnodes); cudaFree(b->d_tris); cudaFree(b->d_slot_of_prim); cudaFree(b->d_mat_id);
    delete b;
    return CRT_OK;
}

crt_status crt_bvh_get_info(const crt_bvh* b, crt_bvh_info_t* o)
{
    if (!b || !o) return crt_fail(nullptr, CRT_ERR_INVALID_ARG, "bvh_get_info: null argument");
    o->optimize_iterations = b->opt_iters; o->reserved = 0; o->n_refs = b->n_refs; o->n_tris = b->n_tris; o->n_nodes = b->nodes.empty() ? b->n_tree_nodes : (int64_t)b->nodes.size(); o->device_bytes = b->device_bytes;
    memcpy(o->bounds, b->bounds, sizeof o->bounds);
    o->sah_cost = b->sah; o->depth = b->depth; o->max_leaf = b->max_leaf; o->build_seconds = b->build_seconds;
    o->n_wide_nodes = b->n_wide_nodes; o->wide_depth = b->wide_depth;
    o->q16_inflation_pct = (int32_t)std::min(1e9, b->q_inflation * 100.0 + 0.5);
    o->builder = b->builder; o->build_rounds = b->ploc_rounds; o->device_build_seconds = 1e-3 * b->device_build_ms; o->layout_seconds = b->layout_seconds;
    return CRT_OK;
}

crt_status crt_bvh_check(const crt_bvh* b, int32_t* violations)
{
    if (!b || !violations) return crt_fail(nullptr, CRT_ERR_INVALID_ARG, "bvh_check: null argument");
    CrtDeviceGuard dev_guard_(b->device);
    // host tree (host builder, builder 2) and/or the device layouts themselves (always when they exist: whichever builder wrote them)
    *violations = (b->nodes.empty() && b->n_tris > 0 ? 0 : crt_bvh_check_host(b)) | (b->wide_violations << 8) | (b->q_violations << 16) | crt_layout_check_device(b);
    return CRT_OK;
}

// ---- index spaces ---------------------------------------------------------------------------------------
crt_status crt_layout(const crt_frame* frame, const crt_order* order, int64_t* n_paths, int64_t* n_slots, int64_t* n_groups)
{
    Layout L;
    crt_status st = crt_make_layout(nullptr, frame, order, &L);
    if (st != CRT_OK) return st;
    if (n_paths) *n_paths = L.n_paths;
    if (n_slots) *n_slots = L.n_slots;
    if (n_groups) *n_groups = L.n_groups;
    return CRT_OK;
}

#define NEED_CTX(name) if (!ctx) return crt_fail(nullptr, CRT_ERR_INVALID_ARG, name ": ctx is null"); CrtDeviceGuard dev_guard_(ctx->device)
#define NEED_BVH(name) if (!bvh) return crt_fail(ctx, CRT_ERR_INVALID_ARG, name ": bvh is null"); \
    if (!bvh->d_nodes || bvh->device != ctx->device) return crt_fail(ctx, CRT_ERR_STATE, name ": BVH has no data on this context's device")
#define NEED_ALIGNED(name, p, a) if (!crt_aligned(p, a)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, name ": " #p " is null or not %d-byte aligned", (int)(a))

crt_status crt_paths_init(crt_ctx* ctx, crt_path_state* paths, int64_t n_paths, void* stream)
{
    NEED_CTX("paths_init");
    if (n_paths < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "paths_init: negative size");
    if (n_paths == 0) return CRT_OK;
    NEED_ALIGNED("paths_init", paths, 16);
    return launch_paths_init(ctx, paths, n_paths, (cudaStream_t)stream);
}

crt_status crt_trace_primary(crt_ctx* ctx, const crt_bvh* bvh, const crt_camera* camera, const crt_frame* frame, const crt_order* order,
                             crt_ray* rays, crt_hit* hits, int32_t* ray_to_path, void* stream)
{
    NEED_CTX("trace_primary"); NEED_BVH("trace_primary");
    if (!camera) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_primary: camera is null");
    Layout L; crt_status st = crt_make_layout(ctx, frame, order, &L); if (st != CRT_OK) return st;
    if (L.n_slots == 0) return CRT_OK;
    NEED_ALIGNED("trace_primary", rays, 32); NEED_ALIGNED("trace_primary", hits, 16); NEED_ALIGNED("trace_primary", ray_to_path, 4);
    return launch_primary(ctx, bvh, *camera, *frame, L, rays, hits, ray_to_path, (cudaStream_t)stream);
}

size_t crt_generate_secondary_scratch_bytes(const crt_frame* frame, const crt_order* order)
{
    Layout L; if (crt_make_layout(nullptr, frame, order, &L) != CRT_OK) return 0;
    return generate_scratch_bytes(L);
}

crt_status crt_generate_secondary(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_frame* frame, int32_t bounce, const crt_order* order,
                                  const crt_ray* prev_rays, const crt_hit* prev_hits, const int32_t* prev_ray_to_path, crt_path_state* paths,
                                  crt_ray* rays_out, int32_t* ray_to_path_out, int32_t* group_id_out, int32_t* dir_src_out, uint8_t* group_class_out,
                                  uint32_t* n_active_out, void* scratch, size_t scratch_bytes, void* stream)
{
    NEED_CTX("generate_secondary"); NEED_BVH("generate_secondary");
    if (!mats || !mats->materials) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "generate_secondary: materials are null");
    if (mats->n_materials <= bvh->max_mat_id) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "generate_secondary: %d materials but the BVH's triangles use id %d", mats->n_materials, bvh->max_mat_id);
    if (bounce < 1) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "generate_secondary: bounce %d < 1", bounce);
    Layout L; crt_status st = crt_make_layout(ctx, frame, order, &L); if (st != CRT_OK) return st;
    NEED_ALIGNED("generate_secondary", n_active_out, 4);
    if (L.n_slots > 0) {
        NEED_ALIGNED("generate_secondary", prev_rays, 32); NEED_ALIGNED("generate_secondary", prev_hits, 16);
        NEED_ALIGNED("generate_secondary", prev_ray_to_path, 4); NEED_ALIGNED("generate_secondary", paths, 16);
        NEED_ALIGNED("generate_secondary", rays_out, 32); NEED_ALIGNED("generate_secondary", ray_to_path_out, 4);
        NEED_ALIGNED("generate_secondary", group_id_out, 4); NEED_ALIGNED("generate_secondary", dir_src_out, 4);
        NEED_ALIGNED("generate_secondary", group_class_out, 1); NEED_ALIGNED("generate_secondary", scratch, 16);
        if (rays_out == prev_rays) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "generate_secondary: rays_out aliases prev_rays");
    }
    return launch_generate(ctx, bvh, *mats, *frame, bounce, L, prev_rays, prev_hits, prev_ray_to_path, paths, rays_out, ray_to_path_out, group_id_out,
                           dir_src_out, group_class_out, n_active_out, scratch, scratch_bytes, (cudaStream_t)stream, nullptr);
}

crt_status crt_morton_encode(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, uint32_t* keys, void* stream)
{
    NEED_CTX("morton_encode");
    if (!bvh) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "morton_encode: bvh is null");
    if (n < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "morton_encode: negative size");
    if (n == 0) return CRT_OK;
    NEED_ALIGNED("morton_encode", rays, 32); NEED_ALIGNED("morton_encode", keys, 4);
    return launch_morton_encode(ctx, bvh->bounds, 0, rays, n, keys, (cudaStream_t)stream);
}

crt_status crt_ray_code_encode(crt_ctx* ctx, const crt_bvh* bvh, int32_t code, const crt_ray* rays, int64_t n, uint32_t* keys, void* stream)
{
    NEED_CTX("ray_code_encode");
    if (!bvh) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "ray_code_encode: bvh is null");
    if (code < 0 || code > CRT_CODE_TWOPOINT) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "ray_code_encode: code %d out of range", code);
    if (n < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "ray_code_encode: negative size");
    if (n == 0) return CRT_OK;
    NEED_ALIGNED("ray_code_encode", rays, 32); NEED_ALIGNED("ray_code_encode", keys, 4);
    return launch_morton_encode(ctx, bvh->bounds, code, rays, n, keys, (cudaStream_t)stream);
}

size_t crt_radix_sort_scratch_bytes(int64_t n) { return n < 0 ? 0 : radix_sort_scratch_bytes(n); }

crt_status crt_radix_sort_pairs(crt_ctx* ctx, const uint32_t* keys_in, const int32_t* vals_in, int64_t n, uint32_t* keys_out, int32_t* vals_out,
                                void* scratch, size_t scratch_bytes, void* stream)
{
    NEED_CTX("radix_sort_pairs");
    if (n < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "radix_sort_pairs: negative size");
    if (n == 0) return CRT_OK;
    NEED_ALIGNED("radix_sort_pairs", keys_in, 4); NEED_ALIGNED("radix_sort_pairs", vals_in, 4);
    NEED_ALIGNED("radix_sort_pairs", keys_out, 4); NEED_ALIGNED("radix_sort_pairs", vals_out, 4); NEED_ALIGNED("radix_sort_pairs", scratch, 16);
    if (keys_out == keys_in || vals_out == vals_in) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "radix_sort_pairs: in-place sort is not supported");
    return launch_radix_sort(ctx, keys_in, vals_in, n, keys_out, vals_out, scratch, scratch_bytes, (cudaStream_t)stream);
}

int64_t crt_radix_sort_noalloc_max_n(void) { return radix_sort_noalloc_max_n(); }

crt_status crt_radix_sort_pairs_noalloc(crt_ctx* ctx, const uint32_t* keys_in, const int32_t* vals_in, int64_t n, uint32_t* keys_out, int32_t* vals_out, void* stream)
{
    NEED_CTX("radix_sort_pairs_noalloc");
    if (n < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "radix_sort_pairs_noalloc: negative size");
    if (n == 0) return CRT_OK;
    NEED_ALIGNED("radix_sort_pairs_noalloc", keys_in, 4); NEED_ALIGNED("radix_sort_pairs_noalloc", vals_in, 4);
    NEED_ALIGNED("radix_sort_pairs_noalloc", keys_out, 4); NEED_ALIGNED("radix_sort_pairs_noalloc", vals_out, 4);
    if (keys_out == keys_in || vals_out == vals_in) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "radix_sort_pairs_noalloc: in-place sort is not supported");
    return launch_radix_sort_noalloc(ctx, keys_in, vals_in, n, keys_out, vals_out, (cudaStream_t)stream);
}

crt_status crt_trace(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, crt_hit* hits, void* stream)
{
    NEED_CTX("trace"); NEED_BVH("trace");
    if (n_rays < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace: negative ray count");
    if (n_rays == 0) return CRT_OK;
    if (n_rays >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_UNSUPPORTED, "trace: more than 2^31 rays per call");
    NEED_ALIGNED("trace", rays, 32); NEED_ALIGNED("trace", hits, 16);
    return launch_trace(ctx, bvh, rays, n_rays, hits, (cudaStream_t)stream);
}

crt_status crt_trace_timeline(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, crt_hit* hits, uint64_t* marks, int64_t marks_capacity_warps, int32_t* n_warps, void* stream)
{
    NEED_CTX("trace_timeline"); NEED_BVH("trace_timeline");
    if (!n_warps || !marks || marks_capacity_warps < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_timeline: null argument");
    if (n_rays < 0 || n_rays >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_timeline: bad ray count");
    NEED_ALIGNED("trace_timeline", marks, 8);
    if (n_rays == 0) { *n_warps = 0; return CRT_OK; }
    NEED_ALIGNED("trace_timeline", rays, 32); NEED_ALIGNED("trace_timeline", hits, 16);
    return launch_trace_timeline(ctx, bvh, rays, n_rays, hits, marks, marks_capacity_warps, n_warps, (cudaStream_t)stream);
}

crt_status crt_trace_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, int64_t* counters, void* stream)
{
    NEED_CTX("trace_stats"); NEED_BVH("trace_stats");
    if (n_rays < 0 || n_rays >= ((int64_t)1 << 31)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "trace_stats: bad ray count");
    NEED_ALIGNED("trace_stats", counters, 8);
    if (n_rays == 0) return CRT_OK;
    NEED_ALIGNED("trace_stats", rays, 32);
    return launch_trace_stats(ctx, bvh, rays, n_rays, counters, (cudaStream_t)stream);
}

crt_status crt_shade_accumulate(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_frame* frame, int32_t bounce, int32_t is_last,
                                const crt_ray* rays, const crt_hit* hits, const int32_t* ray_to_path, int64_t n_rays, crt_path_state* paths, float* accum, void* stream)
{
    NEED_CTX("shade_accumulate"); NEED_BVH("shade_accumulate");
    if (!mats || !mats->materials || !frame) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "shade_accumulate: null argument");
    if (mats->n_materials <= bvh->max_mat_id) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "shade_accumulate: %d materials but the BVH's triangles use id %d", mats->n_materials, bvh->max_mat_id);
    if (bounce < 0 || n_rays < 0 || frame->spp < 1) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "shade_accumulate: bad bounce / size");
    if (n_rays == 0) return CRT_OK;
    NEED_ALIGNED("shade_accumulate", rays, 32); NEED_ALIGNED("shade_accumulate", hits, 16); NEED_ALIGNED("shade_accumulate", ray_to_path, 4);
    NEED_ALIGNED("shade_accumulate", paths, 16); NEED_ALIGNED("shade_accumulate", accum, 4);
    return launch_shade(ctx, bvh, *mats, *frame, is_last, rays, hits, ray_to_path, n_rays, paths, accum, (cudaStream_t)stream);
}

// ---- whole frame ------------------------------------------------------------------------------------------
static size_t al(size_t x) { return (x + 255) & ~(size_t)255; }
struct Workspace {
    crt_ray* rays[2]; crt_hit* hits; int32_t* r2p[2]; int32_t* gid; int32_t* src; uint8_t* cls; crt_path_state* paths; uint32_t* n_active; void* scratch; size_t scratch_bytes;
    size_t total;
};
static Workspace carve(const Layout& L, void* base)
{
    Workspace W; char* p = static_cast<char*>(base); size_t off = 0;
    const size_t ns = (size_t)L.n_slots;
    auto take = [&](size_t bytes) { void* r = p ? p + off : nullptr; off += al(bytes); return r; };
    W.rays[0] = (crt_ray*)take(ns * 32); W.rays[1] = (crt_ray*)take(ns * 32); W.hits = (crt_hit*)take(ns * 16);
    W.r2p[0] = (int32_t*)take(ns * 4); W.r2p[1] = (int32_t*)take(ns * 4); W.gid = (int32_t*)take(ns * 4); W.src = (int32_t*)take(ns * 4);
    W.cls = (uint8_t*)take((size_t)L.n_groups); W.paths = (crt_path_state*)take((size_t)L.n_slots * 32);       // n_slots >= n_paths: grouped orders keep the path state by slot
    W.n_active = (uint32_t*)take(256);
    W.scratch_bytes = generate_scratch_bytes(L); W.scratch = take(W.scratch_bytes);
    W.total = off;
    return W;
}

size_t crt_frame_workspace_bytes(const crt_frame* frame, const crt_order* order)
{
    Layout L; if (crt_make_layout(nullptr, frame, order, &L) != CRT_OK) return 0;
    return carve(L, nullptr).total;
}

static crt_status mark(crt_ctx* ctx, int stage, cudaStream_t st)
{
    if ((size_t)ctx->ev_used == ctx->ev.size()) { cudaEvent_t e; CRT_CUDA(ctx, cudaEventCreate(&e)); ctx->ev.push_back(e); ctx->ev_stage.push_back(-1); }
    ctx->ev_stage[ctx->ev_used] = stage;
    CRT_CUDA(ctx, cudaEventRecord(ctx->ev[ctx->ev_used++], st));
    return CRT_OK;
}

crt_status crt_render_frame(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_camera* camera, const crt_frame* frame,
                            const crt_order* order, int32_t n_bounces, float* accum, uint32_t* n_secondary_out, void* workspace, size_t workspace_bytes,
                            int32_t record_times, void* stream)
{
    NEED_CTX("render_frame"); NEED_BVH("render_frame");
    if (!mats || !mats->materials || !camera) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "render_frame: null argument");
    if (mats->n_materials <= bvh->max_mat_id) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "render_frame: %d materials but the BVH's triangles use id %d", mats->n_materials, bvh->max_mat_id);
    if (n_bounces < 0 || n_bounces > 64) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "render_frame: n_bounces out of range");
    Layout L; crt_status st = crt_make_layout(ctx, frame, order, &L); if (st != CRT_OK) return st;
    if (L.n_slots == 0) return CRT_OK;
    NEED_ALIGNED("render_frame", workspace, 256); NEED_ALIGNED("render_frame", accum, 4);
    Workspace W = carve(L, workspace);
    if (workspace_bytes < W.total) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "render_frame: workspace %zu < %zu bytes", workspace_bytes, W.total);
    cudaStream_t s = (cudaStream_t)stream;
    ctx->ev_used = 0;
#define STEP(call) do { st = (call); if (st != CRT_OK) return st; } while (0)
#define MARK(stage) do { if (record_times) STEP(mark(ctx, stage, s)); } while (0)
    // grouped orders: path state indexed by slot (fixed for the frame), so that shading and generation stream it instead of
    // gathering 32-byte records in the shuffled pixel order of the tiles; the image is unaffected (tested against the staged calls)
    const bool by_slot = (L.mode == CRT_MODE_DIRECT_REUSE || L.mode == CRT_MODE_WORLD_REUSE);
    // option fuse_shade: the shading of every segment but the last runs inside the generation kernel of the next bounce, and the first
    // generation kernel also sets the initial path state (no paths_init launch)
    // (not for the sorting modes: their ray order is a permutation of the paths, and the fused read-modify-write of the state of ended
    // paths would be a scattered access inside the generation kernel: measured 2.3x slower generation on the landscape scene)
    const bool fuse = ctx->fuse_shade != 0 && !crt_mode_sorts(L.mode);
    // Bands (option "frame_bands", default 1 = off): tiles are independent (groups never span tiles), so a frame can be cut into bands of whole tiles,
    // every band running its whole sequence on its own library-owned stream, so that the tail of one band's traversal launch (the last rays finishing on
    // a nearly empty machine, 0.08-0.11 ms per launch) is filled by the others' work inside ONE frame.  Measured (profiles/r02f): two bands +0.8 % (interior)
    // / +4.2 % (landscape) for one frame at a time, three bands less, four a loss (every band launch has its own tail and the bands' persistent grids
    // queue behind each other); with several frames in flight (bench.py's headline) bands cost 2-3 %, hence off by default.
    // Never with per-stage timing (stage times of overlapping bands mean nothing), for the sorting modes (their sort is global), with the alternative
    // kernels that use the context's single work counter, or for small frames.
    const int64_t unit = std::max<int64_t>(by_slot ? L.M : 1, 256);
    const int64_t n_units = (L.n_slots + unit - 1) / unit;
    int n_bands = ctx->frame_bands;
    if (record_times || crt_mode_sorts(L.mode) || ctx->trace_kernel == 2 || ctx->trace_kernel == 5 || L.n_slots < (int64_t)n_bands * 262144) n_bands = 1;
    uint32_t* d_nact = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(ctx->d_counter) + 1024);      // [64] live rays per bounce of a banded frame
    if (n_bands > 1) {
        for (int k = 1; k < n_bands; ++k) {
            if (!ctx->band_stream[k]) CRT_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->band_stream[k], cudaStreamNonBlocking));
            if (!ctx->band_join[k]) CRT_CUDA(ctx, cudaEventCreateWithFlags(&ctx->band_join[k], cudaEventDisableTiming));
        }
        if (!ctx->band_fork) CRT_CUDA(ctx, cudaEventCreateWithFlags(&ctx->band_fork, cudaEventDisableTiming));
        CRT_CUDA(ctx, cudaMemsetAsync(d_nact, 0, 64 * sizeof(uint32_t), s));
        CRT_CUDA(ctx, cudaEventRecord(ctx->band_fork, s));
    }
    for (int k = 0; k < n_bands; ++k) {
        Band band; const Band* bp = nullptr; cudaStream_t sb = s;
        if (n_bands > 1) {
            const int64_t u0 = n_units * k / n_bands, u1 = n_units * (k + 1) / n_bands;
            band.slot0 = u0 * unit; band.count = std::min(u1 * unit, L.n_slots) - band.slot0;
            band.counter = ctx->d_counter + 16 * k; band.n_active = nullptr;
            bp = &band;
            if (k > 0) { sb = ctx->band_stream[k]; CRT_CUDA(ctx, cudaStreamWaitEvent(sb, ctx->band_fork, 0)); }
        }
        const int64_t n_here = bp ? band.count : L.n_slots;
        if (!(fuse && n_bands >= 1 && n_bounces >= 1)) STEP(launch_paths_init(ctx, W.paths + (bp ? band.slot0 : 0), bp ? band.count : (by_slot ? L.n_slots : L.n_paths), sb));
        if (k == 0) MARK(-1);
        STEP(launch_primary(ctx, bvh, *camera, *frame, L, W.rays[0], W.hits, W.r2p[0], sb, bp));
        if (k == 0) MARK(0);
        if (n_bounces == 0 || !fuse) STEP(launch_shade(ctx, bvh, *mats, *frame, n_bounces == 0, W.rays[0], W.hits, W.r2p[0], L.n_slots, W.paths, accum, sb, by_slot, by_slot ? &L : nullptr, bp));
        if (k == 0) MARK(1);
        int cur = 0;
        for (int b = 1; b <= n_bounces; ++b) {
            cudaEvent_t ev4[2] = {nullptr, nullptr};
            if (record_times && crt_mode_sorts(L.mode)) {
                // events bracketing encode+sort+permute inside generate
                while (ctx->ev.size() < (size_t)ctx->ev_used + 2) { cudaEvent_t e; CRT_CUDA(ctx, cudaEventCreate(&e)); ctx->ev.push_back(e); ctx->ev_stage.push_back(-1); }
                ev4[0] = ctx->ev[ctx->ev_used]; ctx->ev_stage[ctx->ev_used++] = -2;     // after the generate kernel: opens stage 4
                ev4[1] = ctx->ev[ctx->ev_used]; ctx->ev_stage[ctx->ev_used++] = 4;      // after permute: closes stage 4
            }
            if (bp) band.n_active = d_nact + (b - 1);
            STEP(launch_generate(ctx, bvh, *mats, *frame, b, L, W.rays[cur], W.hits, W.r2p[cur], W.paths, W.rays[1 - cur], W.r2p[1 - cur], W.gid, W.src, W.cls,
                                 W.n_active, W.scratch, W.scratch_bytes, sb, ev4[0] ? ev4 : nullptr, fuse, by_slot, b == 1, bp));
            cur = 1 - cur;
            if (!bp && n_secondary_out) CRT_CUDA(ctx, cudaMemcpyAsync(n_secondary_out + (b - 1), W.n_active, 4, cudaMemcpyDeviceToDevice, sb));
            MARK(2);
            STEP(launch_trace(ctx, bvh, W.rays[cur] + (bp ? band.slot0 : 0), n_here, W.hits + (bp ? band.slot0 : 0), sb, false, bp ? band.counter : nullptr));
            MARK(3);
            if (b == n_bounces || !fuse) STEP(launch_shade(ctx, bvh, *mats, *frame, b == n_bounces, W.rays[cur], W.hits, W.r2p[cur], L.n_slots, W.paths, accum, sb, by_slot, by_slot ? &L : nullptr, bp));
            MARK(1);
        }
        if (bp && k > 0) { CRT_CUDA(ctx, cudaEventRecord(ctx->band_join[k], sb)); CRT_CUDA(ctx, cudaStreamWaitEvent(s, ctx->band_join[k], 0)); }
    }
    if (n_bands > 1 && n_secondary_out && n_bounces > 0) CRT_CUDA(ctx, cudaMemcpyAsync(n_secondary_out, d_nact, 4 * (size_t)std::min(n_bounces, 64), cudaMemcpyDeviceToDevice, s));
#undef STEP
#undef MARK
    return CRT_OK;
}

crt_status crt_frame_times(crt_ctx* ctx, float* stage_ms)
{
    NEED_CTX("frame_times");
    if (!stage_ms) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "frame_times: null argument");
    if (ctx->ev_used == 0) return CRT_OK;
    CRT_CUDA(ctx, cudaEventSynchronize(ctx->ev[ctx->ev_used - 1]));
    // events are recorded in stream order; an event with stage >= 0 closes the interval opened by the previous event
    // on the main timeline (stage 4 intervals are nested inside a stage-2 interval)
    int prev_main = -1, open4 = -1;
    for (int i = 0; i < ctx->ev_used; ++i) {
        const int stg = ctx->ev_stage[i];
        if (stg == -2) { open4 = i; continue; }
        if (stg == 4) { float ms = 0; CRT_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[open4], ctx->ev[i])); stage_ms[4] += ms; continue; }
        if (stg >= 0 && prev_main >= 0) { float ms = 0; CRT_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[prev_main], ctx->ev[i])); stage_ms[stg] += ms; }
        prev_main = i;
    }
    return CRT_OK;
}

crt_status crt_frame_bounce_times(crt_ctx* ctx, int32_t n_bounces, float* bounce_ms)
{
    NEED_CTX("frame_bounce_times");
    if (!bounce_ms || n_bounces < 0) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "frame_bounce_times: bad argument");
    if (ctx->ev_used == 0) return CRT_OK;
    CRT_CUDA(ctx, cudaEventSynchronize(ctx->ev[ctx->ev_used - 1]));
    int prev_main = -1, open4 = -1, bounce = 0;          // bounce: index of the bounce whose generation interval was closed last
    for (int i = 0; i < ctx->ev_used; ++i) {
        const int stg = ctx->ev_stage[i];
        if (stg == -2) { open4 = i; continue; }
        float ms = 0;
        if (stg == 4) {
            CRT_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[open4], ctx->ev[i]));
            if (bounce < n_bounces) { bounce_ms[3 * bounce + 1] += ms; bounce_ms[3 * bounce + 0] -= ms; }     // nested inside the generation interval that closes next
            continue;
        }
        if (stg >= 0 && prev_main >= 0) {
            CRT_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev[prev_main], ctx->ev[i]));
            if (stg == 2 && bounce < n_bounces) bounce_ms[3 * bounce + 0] += ms;
            if (stg == 3 && bounce < n_bounces) { bounce_ms[3 * bounce + 2] += ms; ++bounce; }
        }
        prev_main = i;
    }
    return CRT_OK;
}

size_t crt_frame_host_extra_bytes(const crt_frame* frame, int32_t n_materials)
{
    if (!frame || n_materials < 0) return 0;
    return al((size_t)n_materials * sizeof(crt_material)) + al((size_t)frame->w * frame->h * 12) + al(64 * 4) + 256;
}

// shared body of the two host-buffer entry points.  resident: the accumulation image lives in the workspace between calls
// (zeroed when reset != 0) and is only copied OUT; otherwise it is copied in from image_host first.
static crt_status render_frame_host_impl(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials, const float* env,
                                         const crt_camera* camera, const crt_frame* frame, const crt_order* order, int32_t n_bounces, float* image_host,
                                         uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream, bool resident, bool reset, bool sync, const char* name)
{
    if (!ctx) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "%s: ctx is null", name);
    CrtDeviceGuard dev_guard_(ctx->device);
    if (!bvh || !bvh->d_nodes || bvh->device != ctx->device) return crt_fail(ctx, bvh ? CRT_ERR_STATE : CRT_ERR_INVALID_ARG, "%s: BVH missing or not on this context's device", name);
    if (!materials_host || !env || !camera || !frame || !image_host || n_materials < 1) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "%s: null argument", name);
    if (n_materials <= bvh->max_mat_id) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "%s: %d materials but the BVH's triangles use id %d", name, n_materials, bvh->max_mat_id);
    Layout L; crt_status st = crt_make_layout(ctx, frame, order, &L); if (st != CRT_OK) return st;
    if (!crt_aligned(workspace, 256)) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "%s: workspace is null or not 256-byte aligned", name);
    const size_t core = carve(L, nullptr).total, extra = crt_frame_host_extra_bytes(frame, n_materials);
    if (workspace_bytes < core + extra) return crt_fail(ctx, CRT_ERR_INVALID_ARG, "%s: workspace %zu < %zu bytes", name, workspace_bytes, core + extra);
    cudaStream_t s = (cudaStream_t)stream;
    char* p = static_cast<char*>(workspace) + core;
    crt_material* d_mats = (crt_material*)p; p += al((size_t)n_materials * sizeof(crt_material));
    float* d_accum = (float*)p; p += al((size_t)frame->w * frame->h * 12);
    uint32_t* d_nsec = (uint32_t*)p;
    const size_t img = (size_t)frame->w * frame->h * 12;
    CRT_CUDA(ctx, cudaMemcpyAsync(d_mats, materials_host, (size_t)n_materials * sizeof(crt_material), cudaMemcpyHostToDevice, s));
    if (!resident) CRT_CUDA(ctx, cudaMemcpyAsync(d_accum, image_host, img, cudaMemcpyHostToDevice, s));
    else if (reset) CRT_CUDA(ctx, cudaMemsetAsync(d_accum, 0, img, s));
    crt_scene_mats sm; sm.materials = d_mats; sm.n_materials = n_materials; memcpy(sm.env, env, sizeof sm.env);
    st = crt_render_frame(ctx, bvh, &sm, camera, frame, order, n_bounces, d_accum, n_secondary_host ? d_nsec : nullptr, workspace, core, 0, stream);
    if (st != CRT_OK) return st;
    CRT_CUDA(ctx, cudaMemcpyAsync(image_host, d_accum, img, cudaMemcpyDeviceToHost, s));
    if (n_secondary_host && n_bounces > 0) CRT_CUDA(ctx, cudaMemcpyAsync(n_secondary_host, d_nsec, 4 * (size_t)n_bounces, cudaMemcpyDeviceToHost, s));
    if (sync) CRT_CUDA(ctx, cudaStreamSynchronize(s));
    return CRT_OK;
}

crt_status crt_render_frame_host(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials, const float* env,
                                 const crt_camera* camera, const crt_frame* frame, const crt_order* order, int32_t n_bounces, float* accum_host,
                                 uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream)
{
    return render_frame_host_impl(ctx, bvh, materials_host, n_materials, env, camera, frame, order, n_bounces, accum_host, n_secondary_host,
                                  workspace, workspace_bytes, stream, false, false, true, "render_frame_host");
}

crt_status crt_render_frame_host_resident(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials, const float* env,
                                          const crt_camera* camera, const crt_frame* frame, const crt_order* order, int32_t n_bounces, int32_t reset,
                                          float* image_host, uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream)
{
    return render_frame_host_impl(ctx, bvh, materials_host, n_materials, env, camera, frame, order, n_bounces, image_host, n_secondary_host,
                                  workspace, workspace_bytes, stream, true, reset != 0, true, "render_frame_host_resident");
}

crt_status crt_render_frame_host_resident_async(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials, const float* env,
                                                const crt_camera* camera, const crt_frame* frame, const crt_order* order, int32_t n_bounces, int32_t reset,
                                                float* image_host, uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream)
{
    return render_frame_host_impl(ctx, bvh, materials_host, n_materials, env, camera, frame, order, n_bounces, image_host, n_secondary_host,
                                  workspace, workspace_bytes, stream, true, reset != 0, false, "render_frame_host_resident_async");
}

}  // extern "C"
