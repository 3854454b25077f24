// Internal declarations of libcrt (host side).  Not installed; the public ABI is include/crt.h.
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <string>
#include <vector>
#include "crt.h"

struct crt_ctx {
    int device = 0;
    int n_sms = 0;
    std::string last_error;
    // options
    int trace_kernel = 3;        // 0: binary BVH, one thread per ray; 1: binary BVH with fp32 64-byte nodes, persistent warps; 2: 8-wide compressed BVH, persistent warps (needs max_leaf == 1; else falls back to 1); 3 (default): binary BVH with 16-bit 32-byte nodes, persistent warps
    int trace_refill_threshold = 16;   // idle lanes refetch when fewer than this many lanes of the warp are busy
    int trace_leaf_wait = 6;           // leave the inner-node phase when at most this many converged lanes still lack a leaf
    int trace_tri_wait = 8;            // wide kernel: a warp enters its triangle phase when at least this many lanes hold triangle hits
    int trace_blocks_per_sm = 0; // 0 = from occupancy
    int shade_pixel_order = 1;   // crt_render_frame, grouped orders: the last segment's shading walks the tile in pixel order (coalesced image updates)
    int trace_tail_split = 0;    // default kernel: in the drain phase of a launch idle lanes take over stack entries of their warp's busy lanes (trace.cu)
    int trace_exact = 1;         // 1: the bit-exact triangle test (D:R0); 0: fused multiply-adds + approximate reciprocal (north_star's tolerances only)
    int fuse_shade = 1;          // crt_render_frame: shade non-final segments inside the next generation kernel (default; measured: DESIGN.md 5.4)
    // persistent-kernel work counters (one per band of a frame, 64 bytes apart) and, 1 KB in, the per-bounce live-ray counts of a banded frame
    unsigned int* d_counter = nullptr;
    // crt_render_frame in bands (option "frame_bands"): library-owned streams on which the bands of one frame run side by side
    int frame_bands = 1;
    cudaStream_t band_stream[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t band_fork = nullptr, band_join[4] = {nullptr, nullptr, nullptr, nullptr};
    // events for crt_render_frame(record_times)
    std::vector<cudaEvent_t> ev;
    std::vector<int> ev_stage;   // stage index closed by event i (-1: opening event)
    int ev_used = 0;
};

// build-time tree node (host)
struct BuildNode {
    float bmin[3], bmax[3];
    int32_t left = -1, right = -1;   // inner
    int32_t first = 0, count = 0;    // leaf: range in prim order
};

// traversal layout (device): 64 bytes = two identical 32-byte child records, each fetched with one 256-bit load
struct GpuChild {
    float min_x, max_x, min_y, max_y, min_z, max_z;
    int32_t ref;     // >= 0: node index; < 0: ~((tri_offset << 3) | (count - 1))
    int32_t pad;
};
struct alignas(64) GpuNode { GpuChild c[2]; };
// quantised traversal layout (device): 32 bytes = ONE 256-bit load per node.  Box planes are 16-bit positions on a grid
// over the (padded) scene box, rounded outward (bvh_build.cpp: crt_bvh_quantise); word k < 3 = child 0, axis k; word 3 + k =
// child 1, axis k; low half = min plane, high half = max plane.  ref as in GpuChild.
struct alignas(32) QNode { uint32_t planes[6]; int32_t ref[2]; };
// leaf triangle, 64 bytes = two 256-bit loads: v0 | prim id, e1 | 0, e2 | 0, padding
// (e = v - v0 rounded once, as the intersection formula needs)
struct alignas(64) GpuTri { float4 v0p; float4 e1; float4 e2; float4 pad; };
// 8-wide compressed node, 128 bytes = four 256-bit loads (layout and rounding rules: bvh_wide.cpp)
struct alignas(128) WNode {
    float px, py, pz;        // origin of the node's box
    float ex;                // E.x: power of two >= extent
    uint32_t eyz;            // E.y (high half) | E.z (low half) as bf16
    uint32_t child_base;     // index of the first inner child
    uint32_t tri_base;       // position of the first triangle child
    uint32_t masks;          // imask (inner children) | lmask << 8 (triangle children)
    uint32_t planes[3][8];   // per axis: 4 words of LO planes, 4 words of HI planes; word k = children 2k (low half), 2k+1 (high half)
};
static_assert(sizeof(WNode) == 128 && sizeof(GpuTri) == 64 && sizeof(QNode) == 32, "device layouts");
// grid of the quantised layout: position q (0..65535) on axis k is the coordinate gmin[k] + q / scale[k]
struct QGrid { float gmin[3], scale[3], inv_scale[3]; };

struct crt_bvh {
    int64_t n_tris = 0;
    int64_t n_refs = 0;               // triangle references = records of the device triangle array (> n_tris when the host build pre-split large triangles)
    int max_leaf = 4;
    std::vector<BuildNode> nodes;     // host tree (root = 0)
    std::vector<int32_t> prim;        // leaf order -> caller's triangle id
    std::vector<float> verts;         // host copy of the caller's vertices (for crt_bvh_check)
    float bounds[6] = {0, 0, 0, 0, 0, 0};
    double sah = 0; int depth = 0; double build_seconds = 0;
    int opt_iters = 0;                 // iterations of tree optimisation run and kept (host: re-insertion of bvh_build.cpp; builder 1: parallel re-insertion of bvh_ploc.cu)
    int builder = 0; int ploc_rounds = 0; float device_build_ms = 0.f; double layout_seconds = 0;      // device builder (bvh_ploc.cu)
    // device data
    int device = -1;
    GpuNode* d_nodes = nullptr; int64_t n_gpu_nodes = 0; int64_t n_tree_nodes = 0;      // n_tree_nodes: nodes of the (collapsed) tree when no host tree exists (device builder)
    QNode* d_qnodes = nullptr; QGrid qgrid = {}; int32_t q_violations = 0; double q_inflation = 1.0;   // 16-bit layout of the same nodes (trace_kernel 3)
    QNode* d_q4nodes = nullptr; int64_t n_q4_nodes = 0;       // 4-wide form of the 16-bit nodes: node j = records 2j, 2j + 1 (trace_kernel 7; built on first use)
    GpuTri* d_tris = nullptr;          // leaf order (wide order when the wide layout exists)
    WNode* d_wnodes = nullptr; int64_t n_wide_nodes = 0; int wide_depth = 0; int32_t wide_violations = 0;   // 8-wide layout (only when max_leaf == 1)
    int32_t* d_slot_of_prim = nullptr; // caller's triangle id -> index into d_tris
    int32_t* d_mat_id = nullptr;       // by caller's triangle id
    int32_t max_mat_id = -1;           // largest material id of any triangle (ids are checked >= 0 at build time)
    int64_t device_bytes = 0;
};

// error helpers -----------------------------------------------------------------------------------
crt_status crt_fail(crt_ctx* ctx, crt_status st, const char* fmt, ...);
#define CRT_CUDA(ctx, call)                                                                         \
    do {                                                                                            \
        cudaError_t e_ = (call);                                                                    \
        if (e_ != cudaSuccess) return crt_fail(ctx, CRT_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)
#define CRT_CHECK_LAUNCH(ctx, what)                                                                 \
    do {                                                                                            \
        cudaError_t e_ = cudaGetLastError();                                                        \
        if (e_ != cudaSuccess) return crt_fail(ctx, CRT_ERR_CUDA, "launch %s: %s", what, cudaGetErrorString(e_)); \
    } while (0)
// makes the context's device current for the duration of an entry point (a C caller or another thread may have a different
// current device; allocations, launches and event calls must land on the context's)
struct CrtDeviceGuard {
    int prev = -1; bool switched = false;
    explicit CrtDeviceGuard(int device)
    {
        if (device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~CrtDeviceGuard() { if (switched) cudaSetDevice(prev); }
    CrtDeviceGuard(const CrtDeviceGuard&) = delete; CrtDeviceGuard& operator=(const CrtDeviceGuard&) = delete;
};
static inline bool crt_aligned(const void* p, size_t a) { return p != nullptr && (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// layout of the slot space ---------------------------------------------------------------------------
struct Layout {
    int32_t w, h, spp, mode;
    int32_t W, H, M, K, G, tiles_x, tiles_y, n_tiles;
    int32_t log2W, log2M, log2K;
    int32_t gw, sx, sy, lattice;       // group width, strides, partition rule (crt_partition_rule; D:R3, R20, R21)
    int64_t n_paths, n_slots, n_groups;
};
crt_status crt_make_layout(crt_ctx* ctx, const crt_frame* f, const crt_order* o, Layout* L);

// a contiguous range of slots of a frame processed on its own stream (crt_render_frame in bands): tiles are independent (groups never span
// tiles), so every stage can run on a band of whole tiles; counter = the band's traversal work counter; n_active = where generation counts its
// live rays (added to, not zeroed, when band != nullptr)
struct Band { int64_t slot0, count; unsigned int* counter; uint32_t* n_active; };

// kernels' host launchers (defined in the .cu files) ------------------------------------------------------
crt_status crt_bvh_build_device(crt_ctx* ctx, crt_bvh* b, const float* verts, int64_t n, const crt_bvh_params& pr, bool full_device);
int32_t crt_layout_check_device(const crt_bvh* b);
bool crt_bvh_ensure_q4(const crt_bvh* b);
crt_status launch_trace(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, cudaStream_t st, bool far_origins = false, unsigned int* counter = nullptr, bool camera_rays = false);
bool trace_queue_supported(const crt_bvh* bvh);
crt_status launch_trace_queue(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st);
crt_status launch_trace_timeline(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, uint64_t* marks, int64_t max_warps, int32_t* n_warps, cudaStream_t st);
int crt_bvh_optimize_tree(crt_bvh* b, const crt_bvh_params& pr, int built_depth);
crt_status crt_bvh_reinsert_device(crt_ctx* ctx, crt_bvh* b, int iterations, int collapse_max_leaf = 0);
bool trace_group_supported(const crt_bvh* bvh);
crt_status launch_trace_group(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, unsigned long long* stats, cudaStream_t st, unsigned int* counter, int group);
crt_status launch_trace_wide(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, crt_hit* hits, cudaStream_t st);
crt_status launch_trace_wide_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, int64_t* counters, cudaStream_t st);
crt_status launch_trace_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, int64_t* counters, cudaStream_t st);
crt_status launch_primary(crt_ctx* ctx, const crt_bvh* bvh, const crt_camera& cam, const crt_frame& f, const Layout& L,
                          crt_ray* rays, crt_hit* hits, int32_t* r2p, cudaStream_t st, const Band* band = nullptr);
crt_status launch_generate(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats& mats, const crt_frame& f, int bounce, const Layout& L,
                           const crt_ray* prev_rays, const crt_hit* prev_hits, const int32_t* prev_r2p, crt_path_state* paths,
                           crt_ray* rays_out, int32_t* r2p_out, int32_t* gid_out, int32_t* src_out, uint8_t* cls_out,
                           uint32_t* n_active, void* scratch, size_t scratch_bytes, cudaStream_t st, cudaEvent_t* ev4, bool fuse_shade = false, bool paths_by_slot = false, bool fresh_paths = false, const Band* band = nullptr);
crt_status launch_morton_encode(crt_ctx* ctx, const float* bounds, int code, const crt_ray* rays, int64_t n, uint32_t* keys, cudaStream_t st);
// reordering modes (encode + sort + permute) and their sort key: 0 AilaCompact, 1 Origin, 2 Reis, 3 Costa, 4 TwoPoint
static inline bool crt_mode_sorts(int mode) { return mode == CRT_MODE_MORTON_REORDER || (mode >= CRT_MODE_SORT_ORIGIN && mode <= CRT_MODE_SORT_TWOPOINT); }
static inline int crt_mode_sort_code(int mode) { return mode == CRT_MODE_MORTON_REORDER ? 0 : mode - CRT_MODE_SORT_ORIGIN + 1; }
crt_status launch_radix_sort(crt_ctx* ctx, const uint32_t* kin, const int32_t* vin, int64_t n, uint32_t* kout, int32_t* vout,
                             void* scratch, size_t scratch_bytes, cudaStream_t st);
size_t radix_sort_scratch_bytes(int64_t n);
void radix_sort_noalloc_setup(int device);
int64_t radix_sort_noalloc_max_n();
crt_status launch_radix_sort_noalloc(crt_ctx* ctx, const uint32_t* kin, const int32_t* vin, int64_t n, uint32_t* kout, int32_t* vout, cudaStream_t st);
crt_status launch_shade(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats& mats, const crt_frame& f, int is_last,
                        const crt_ray* rays, const crt_hit* hits, const int32_t* r2p, int64_t n, crt_path_state* paths, float* accum, cudaStream_t st, bool paths_by_slot = false, const Layout* pixel_order = nullptr, const Band* band = nullptr);
crt_status launch_paths_init(crt_ctx* ctx, crt_path_state* paths, int64_t n, cudaStream_t st);
crt_status measure_peaks(crt_ctx* ctx, double* tflops, double* gbs);
namespace crt { struct DevLayout; }
size_t generate_scratch_bytes(const Layout& L);
