/*
 * crt.h -- C ABI of libcrt: the secondary-bounce hot path of "Generate Coherent Rays
 * Directly" (arxiv 2310.07182) for NVIDIA B200 (sm_100a).
 *
 * Citations: "P:Lnn" = PAPER.md line nn; "D:Rn" = reading n in DESIGN.md section 3.
 *
 * Conventions
 *  - Every function returns a crt_status; crt_last_error(ctx) gives the message of the
 *    last failure on that context.  No exceptions cross this boundary.
 *  - Pointers marked [device] are CUDA device pointers of the context's device, owned by
 *    the caller (e.g. torch CUDA tensors) and must be 16-byte aligned (crt_ray: 32-byte).
 *    Pointers marked [host] are ordinary host memory.  [host|device] is detected.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue
 *    work on it and return without synchronising, except where stated.
 *  - The library allocates nothing in the per-frame calls; scratch comes from the caller
 *    (sizes from the *_scratch_bytes queries).  The only library-owned objects are
 *    crt_ctx and crt_bvh.
 *  - There is no CPU fallback: without a usable CUDA device crt_create fails.
 *
 * Index spaces (D:R3-R5)
 *  path  p = (sample*h + y)*w + x,             n_paths = spp*w*h
 *  mode independent / morton_reorder:           n_slots = n_paths
 *  mode direct_reuse / world_reuse with group gw x gh and interleave stride s (all powers of two):
 *      tile W x H = (gw*s) x (gh*s), M = W*H slots per tile, K = gw*gh rays per group,
 *      slot = (sample*n_tiles + tile)*M + m,  m = (a*n + c) mod M the shuffled number of
 *      pixel n = ly*W + lx of the tile;  group = slot / K;  n_slots = spp*n_tiles*M.
 */
#ifndef CRT_H_
#define CRT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CRT_OK = 0,
    CRT_ERR_INVALID_ARG = 1,   /* null / misaligned pointer, negative size, bad enum */
    CRT_ERR_UNSUPPORTED = 2,   /* valid request outside what the kernels implement */
    CRT_ERR_CUDA = 3,          /* a CUDA runtime call failed; message has the CUDA error */
    CRT_ERR_STATE = 4,         /* object used before it is ready (e.g. BVH without device data) */
    CRT_ERR_NOMEM = 5
} crt_status;

/* CRT_MODE_WORLD_REUSE: the paper's first variant, "Direct Direction Reusing" in WORLD space (section 3.1; D:R18): same
 * groups and slot order as CRT_MODE_DIRECT_REUSE, but the selected pixel's world direction is shared as is; members for which
 * it lies below the horizon end (the artifact of Fig. 1).  Kept as the ablation the paper argues from, not as the method. */
/* CRT_MODE_SORT_*: the other reordering baselines of the paper's comparison (section 2.1, section 4; D:R19): the same
 * procedure as CRT_MODE_MORTON_REORDER (independent rays, stable radix sort by a 30-bit key, permute) with another key:
 * ORIGIN = Morton code of the origin, 10 bits per axis; REIS = 15-bit origin code above 15-bit direction code [RCP17]; COSTA = direction
 * above origin [CPJ15]; TWOPOINT = origin and end point o + 0.25 * (largest scene extent) * d interleaved [MBGB20, fixed length]. */
typedef enum { CRT_MODE_INDEPENDENT = 0, CRT_MODE_MORTON_REORDER = 1, CRT_MODE_DIRECT_REUSE = 2, CRT_MODE_WORLD_REUSE = 3,
               CRT_MODE_SORT_ORIGIN = 4, CRT_MODE_SORT_REIS = 5, CRT_MODE_SORT_COSTA = 6, CRT_MODE_SORT_TWOPOINT = 7 } crt_mode;
/* sort keys for crt_ray_code_encode (crt_morton_encode = AILA_COMPACT) */
typedef enum { CRT_CODE_AILA_COMPACT = 0, CRT_CODE_ORIGIN = 1, CRT_CODE_REIS = 2, CRT_CODE_COSTA = 3, CRT_CODE_TWOPOINT = 4 } crt_ray_code;
typedef enum { CRT_MAT_DIFFUSE = 0, CRT_MAT_GLOSSY = 1, CRT_MAT_SPECULAR = 2, CRT_MAT_EMISSIVE = 3 } crt_mat_type;
typedef enum { CRT_CLASS_EMPTY = 0, CRT_CLASS_DIFFUSE = 1, CRT_CLASS_GLOSSY = 2, CRT_CLASS_HYBRID = 3 } crt_group_class;

typedef struct crt_ctx crt_ctx;
typedef struct crt_bvh crt_bvh;

/* 32 bytes.  tmax < 0 marks an inactive slot (dead path or out-of-image slot). */
typedef struct { float ox, oy, oz, tmin, dx, dy, dz, tmax; } crt_ray;
/* 16 bytes.  prim indexes the CALLER's triangle array; -1 = miss (then t = ray.tmax, u = v = 0). */
typedef struct { float t, u, v; int32_t prim; } crt_hit;
/* 32 bytes, indexed by path id.  flags bit 0 = alive.  (tr,tg,tb) throughput, (lr,lg,lb) radiance so far. */
typedef struct { float tr, tg, tb; uint32_t flags; float lr, lg, lb; uint32_t pad; } crt_path_state;
/* 32 bytes.  type is a crt_mat_type; roughness = GGX alpha; emission only read for CRT_MAT_EMISSIVE. */
typedef struct { float albedo[3]; float roughness; float emission[3]; int32_t type; } crt_material;
typedef struct { int32_t w, h, spp, seed, frame; } crt_frame;
/* pinhole camera (D:R6): a pixel at normalised screen position (sx,sy) in [-1,1]^2, sy up, looks along W + sx*U + sy*V */
typedef struct { float eye[3], U[3], V[3], W[3]; } crt_camera;
/* stride = horizontal interleave stride; stride_y = vertical one (0 = same as stride).  The tile is (group_w*stride) x
 * (group_h*stride_y) and K = group_w*group_h, which expresses every power-of-two (W, H, K) of the paper's own
 * parametrisation, e.g. tile 8x8 with K = 8 as group 8x1, stride 1, stride_y 8 (D:R5). */
/* partition_rule: how the pixels of a tile are dealt to its groups.  CRT_PARTITION_SHUFFLE (0, default): the paper's rule,
 * pixel numbers "shuffled using a linear congruence method" (D:R3).  CRT_PARTITION_LATTICE (1): a regular lattice, the
 * literal reading of "interleave stride" (D:R20): after a cyclic shift of the tile drawn per tile, sample and frame, the pixels
 * congruent modulo (stride, stride_y) form a group; its members lie stride / stride_y pixels apart. */
/* CRT_PARTITION_LCG_SEQUENCE (2): the other reading of "shuffled using a linear congruence method" (D:R21): the shuffled
 * number of pixel n is the n-th TERM of a full-period linear congruential sequence x -> (A x + C) mod M (C odd, A = 1 mod 4;
 * A, C and the start x_0 drawn per tile, sample and frame), instead of the affine image a*n + c of the number itself. */
typedef enum { CRT_PARTITION_SHUFFLE = 0, CRT_PARTITION_LATTICE = 1, CRT_PARTITION_LCG_SEQUENCE = 2 } crt_partition_rule;
typedef struct { int32_t mode, group_w, group_h, stride, stride_y, partition_rule; } crt_order;
/* materials: [device] table indexed by the per-triangle material id given to crt_build_bvh.
 * env: radiance on a miss = lerp(env[0..2], env[3..5], 0.5*(d.y+1)) (D:R14). */
typedef struct { const crt_material* materials; int32_t n_materials; float env[6]; } crt_scene_mats;
/* builder: 0 = host (binned surface-area heuristic, threaded; with a context its optimisation step runs on the device, see `optimize`); 3 = host entirely
 * (what 0 does without a context); 1 = device (parallel locally-ordered clustering AND the traversal layouts
 * written by the GPU, csrc/bvh_ploc.cu; needs a context); 2 = the device's clustering with the host's tree optimisation (`optimize`) and layout code
 * (cross-check of 1; profiles/r02n);
 * ploc_radius: neighbours searched on either side of a cluster in Morton order (0 = 8; at most 128).
 * presplit (host builder, max_leaf > 1): a triangle whose box is longer than presplit x the scene's diagonal on some axis is given several REFERENCES,
 * one per cell of a recursive midpoint split of its box, each with the box of the part of the triangle inside the cell, and the tree is built over
 * references (at most n_tris / 4 + 4096 extra ones).  The triangle itself is unchanged -- same record, same id, tested whole -- so every traversal
 * returns the same hit; only the boxes that lead to it are tighter (walls and floors no longer overlap every object in front of them: interior scene
 * -8 % primary, -2 % secondary traversal time, profiles/r02k).  0 = off; NULL params = 1/16.
 * optimize (host builder): iterations of insertion-based optimisation of the built tree (Bittner et al. 2013): each takes the 2 % worst-looking inner
 * nodes (at most 20,000), detaches their children and puts each back where it adds the least surface area.  Same leaves, same hits; interior scene: SAH
 * cost -8 %, traversal -2 to -4 % for +0.8 s of build time (profiles/r02k); stops early when four iterations gain less than 0.2 % (a terrain grid).
 * 0 = off; NULL params = 20.  With a context, builders 0 and 1 run (at most) that many iterations of PARALLEL re-insertion on the device instead (bvh_ploc.cu:
 * every node searches its best position in every iteration, conflicting moves are resolved by locks; stronger and two orders of magnitude faster than the
 * host's version: profiles/r02o); builders 2 and 3 and host-only builds run the host's.  For builder 0 with a context the tree is built and optimised with one
 * triangle reference per leaf and subtrees of at most max_leaf references are collapsed into leaves afterwards. */
typedef struct { int32_t max_leaf; int32_t sah_bins; float cost_traversal, cost_intersect; int32_t n_threads; int32_t builder; int32_t ploc_radius; float presplit; int32_t optimize; } crt_bvh_params;
typedef struct {
    int64_t n_tris, n_nodes, device_bytes;
    float bounds[6];            /* exact min/max over the vertices (unpadded); used by the Morton code */
    double sah_cost; int32_t depth, max_leaf;
    double build_seconds;
    int64_t n_wide_nodes;       /* 8-wide compressed nodes (128 bytes each); 0 when max_leaf != 1 */
    int32_t wide_depth;
    int32_t q16_inflation_pct;  /* summed surface area of the boxes the 16-bit nodes decode to, in percent of the fp32 boxes' (100 = no
                                 * loss); above 200 the default kernel reads the fp32 nodes instead (grid too coarse for the scene) */
    int32_t builder;            /* 0 host SAH, 1 device PLOC, 2 device PLOC + host optimisation and layout, 3 host SAH with the host's own optimisation */
    int32_t build_rounds;       /* device builder: clustering rounds */
    double device_build_seconds;/* device builder: boxes + Morton sort + clustering on the GPU (CUDA events); build_seconds is the whole
                                 * hierarchy build including the copy back and the leaf collapse; layout_seconds the flattening, 16-bit
                                 * quantisation and upload of the traversal layouts (either builder) */
    double layout_seconds;
    int64_t n_refs;             /* triangle references = records of the device triangle array (n_tris unless large triangles were pre-split) */
    int32_t optimize_iterations;/* iterations of tree optimisation that ran and were kept (crt_bvh_params.optimize is the upper limit) */
    int32_t reserved;
} crt_bvh_info_t;

/* ---- context ------------------------------------------------------------------------------------ */
/* Creates a context on CUDA device `device`.  Fails with CRT_ERR_CUDA when no device is usable. */
/* A context serialises its own calls (its traversal work counter and its event pool are per context): to keep several frames in
 * flight on different streams, create one context per stream; BVHs and device buffers may be shared between contexts of a device. */
crt_status crt_create(int32_t device, crt_ctx** out);
crt_status crt_destroy(crt_ctx* ctx);
/* Message of the last failed call on ctx (ctx may be NULL: last failure of a call that had no context). */
const char* crt_last_error(const crt_ctx* ctx);
/* Tunables (for experiments; defaults are what bench.py times): "trace_kernel" (0 = binary BVH, one thread per ray;
 * 1 = binary BVH with fp32 64-byte nodes, persistent warps with per-lane dynamic fetch; 2 = 8-wide compressed BVH, persistent warps;
 * 3 = the persistent kernel of 1 on 16-bit 32-byte nodes, plane distances by packed FFMA2 -- the default; 4 = as 3 with a box test that
 * is conservative for ANY ray origin (3 is for origins within 16 scene extents of the scene, 1 within about 128), 3-4 % slower;
 * 5 = warp-cooperative triangle phase: the triangles of a warp's parked leaves become one work list in shared memory, tested one
 * item per lane (same hit records; measured 15-25 % slower, profiles/r02a); 6 = as 3 with the top 512 nodes of the tree staged in shared
 * memory per block (same hit records; measured 8-16 % slower, profiles/r02a); 7 = the 4-wide form of the 16-bit nodes, two 32-byte records per node, built
 * on first use (half the node visits, same hit records; measured 5-23 % slower, profiles/r02a); 8 / 9 = group-coherent descent: the 16 rays of a
 * half-warp (one group at K = 16) / the 32 rays of a warp walk one shared stack, a node is fetched once per packet (same hit records; measured
 * 1.2-6x slower, profiles/r02h)), "trace_exact" (1 = default: the bit-exact triangle
 * test of D:R0; 0 = fused multiply-adds and an approximate reciprocal in the triangle test: 3-5 % faster, ids equal on >= 99.999 % of
 * rays but t of grazing hits off by up to 4e-4 relative, i.e. outside north_star's 1e-4: an option, not the default),
 * "trace_tail_split" (0 = default; 1: once the ray list is exhausted, idle lanes of a warp take over the bottom stack entries of its busy lanes;
 * same hit records; the drain of a launch gets no shorter and the node loop 8 % slower, profiles/r02i),
 * "trace_leaf_wait" (0..31: a warp leaves its inner-node
 * phase when at most this many descending lanes hold no leaf), "trace_refill_threshold" (0..32: idle lanes fetch new rays when
 * fewer lanes than this are busy), "trace_blocks_per_sm" (0 = from the occupancy calculator), "trace_tri_wait" (8-wide kernel: lanes holding triangle hits
 * before a warp enters its triangle phase), "fuse_shade" (crt_render_frame shades non-final segments inside the next generation
 * kernel; on by default: 2.5-3 % faster on both bench scenes, the image is bit-identical), "shade_pixel_order" (1 = default: under a grouped
 * order the last segment is shaded in the tile's pixel order through the partition's forward map, so that image updates coalesce: +2-3 % per
 * frame, identical image), "frame_bands" (1..4, default 1: crt_render_frame cuts a frame into that many bands of whole tiles, each on its own
 * library-owned stream, so that one band's traversal tail overlaps the others' work; identical image; 2 bands: +1-4 % for one frame at a
 * time, -2-3 % when several frames are in flight on several contexts, profiles/r02f). */
crt_status crt_set_option(crt_ctx* ctx, const char* key, int64_t value);
/* Measures the device's FP32 FFMA rate (TFLOP/s) and a streaming copy rate (GB/s) with small kernels;
 * synchronous. Used only as roofline denominators by bench.py. */
crt_status crt_measure_peaks(crt_ctx* ctx, double* fp32_tflops, double* copy_gbs);

/* ---- a0: acceleration structure (D:R11) ------------------------------------------------ */
/* Builds a binary BVH (binned surface-area heuristic, leaves <= max_leaf triangles) on the host with
 * n_threads threads and uploads it in the traversal layouts: the binary fp32 64-byte-node layout and its 16-bit
 * 32-byte-node form (planes on a 65536-step grid over the scene box, rounded outward; read by the default trace_kernel 3,
 * whose box test is conservative for ray origins within 16 scene extents of the scene) always, and, when
 * max_leaf == 1, its collapse into 8-wide compressed 128-byte nodes (read by trace_kernel 2; measured slower than the
 * binary layout on both bench workloads, profiles/r01b, so not the default).
 * verts: [host|device] float[n_tris][3][3]; mat_id: [host|device] int32[n_tris].  Synchronous.  params may be
 * NULL (defaults: max_leaf 3, 64 bins, costs 1/1, all hardware threads, host builder).  params->builder = 1 builds the hierarchy on
 * the device instead (bvh_ploc.cu: two orders of magnitude faster, traversal within a few percent: profiles/r02b); the traversal
 * layouts, the checks and every other call are the same.  With ctx == NULL only the host tree is built (for crt_bvh_check /
 * crt_bvh_get_info; such a BVH is rejected by the device calls with CRT_ERR_STATE). */
crt_status crt_build_bvh(crt_ctx* ctx, const float* verts, const int32_t* mat_id, int64_t n_tris,
                         const crt_bvh_params* params, crt_bvh** out);
crt_status crt_bvh_destroy(crt_bvh* bvh);
crt_status crt_bvh_get_info(const crt_bvh* bvh, crt_bvh_info_t* out);
/* Structural invariants of the host tree: *violations = 0 iff every triangle is in exactly one leaf (pre-split builds: in at least one, and the boxes
 * of its leaves together cover it), every
 * leaf has 1..max_leaf triangles, every node's box contains its children's boxes / its triangles, and (wide
 * layout, bits 8 and up) every triangle lies inside the box the kernel decodes for each of its ancestors, and (16-bit
 * layout, bit 16) every quantised plane lies at least one grid step outside the fp32 box it replaces. */
crt_status crt_bvh_check(const crt_bvh* bvh, int32_t* violations);

/* ---- index spaces -------------------------------------------------------------------------------- */
/* CRT_ERR_UNSUPPORTED unless group_w, group_h, stride are powers of two with tile size M <= 4096 and K <= 1024. */
crt_status crt_layout(const crt_frame* frame, const crt_order* order, int64_t* n_paths, int64_t* n_slots, int64_t* n_groups);

/* ---- path state ---------------------------------------------------------------------------------- */
/* paths: [device] crt_path_state[n_paths] <- throughput 1, radiance 0, alive. */
crt_status crt_paths_init(crt_ctx* ctx, crt_path_state* paths, int64_t n_paths, void* stream);

/* ---- a1: primary rays (one path per pixel, shading point = first hit) ---------------------- */
/* For every slot of the order: camera ray of its path (jitter from Philox purpose CAMERA), nearest hit.
 * rays, hits, ray_to_path: [device] arrays of n_slots; out-of-image slots get an inactive ray and path -1. */
crt_status crt_trace_primary(crt_ctx* ctx, const crt_bvh* bvh, const crt_camera* camera /*[host]*/, const crt_frame* frame,
                             const crt_order* order, crt_ray* rays, crt_hit* hits, int32_t* ray_to_path, void* stream);

/* ---- a2-a4: secondary-ray generation (P:L95-113 sections 3.2-3.3; P:L43 for morton_reorder) -------- */
/* From the previous segment (prev_* arrays in the SAME order, n_slots entries) generate the rays of bounce
 * `bounce` >= 1.  Outputs (all [device]): rays_out, ray_to_path_out, group_id_out, dir_src_out: n_slots entries;
 * group_class_out: n_groups bytes (crt_group_class); n_active_out: one uint32 (zeroed by the call, then counted).
 *   group_id_out[slot] = slot / K (direct_reuse, world_reuse) or the path id (other modes)
 *   dir_src_out[slot]  = path id whose random numbers produced the direction: own id (glossy/specular member or
 *                        independent sampling), the group leader's id (diffuse group), -2 - group (diffuse member of
 *                        a hybrid group: mean direction of the glossy members), -1 (no ray); world_reuse: the selected
 *                        pixel's id for every member that reuses its world direction
 * paths[path].throughput is multiplied by the BSDF weight; paths whose sample is invalid are killed.
 * scratch: [device], at least crt_generate_secondary_scratch_bytes(). */
crt_status crt_generate_secondary(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_frame* frame,
                                  int32_t bounce, const crt_order* order,
                                  const crt_ray* prev_rays, const crt_hit* prev_hits, const int32_t* prev_ray_to_path,
                                  crt_path_state* paths, crt_ray* rays_out, int32_t* ray_to_path_out, int32_t* group_id_out,
                                  int32_t* dir_src_out, uint8_t* group_class_out, uint32_t* n_active_out,
                                  void* scratch, size_t scratch_bytes, void* stream);
size_t crt_generate_secondary_scratch_bytes(const crt_frame* frame, const crt_order* order);

/* Parts of morton_reorder, exported for testing and timing (P:L43 [AK10]; D:R12).
 * keys[i] = 30-bit interleaved origin+direction code of rays[i] inside bvh bounds, 0xFFFFFFFF if inactive. */
crt_status crt_morton_encode(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n, uint32_t* keys, void* stream);
/* The same for any of the sort keys above (code: crt_ray_code; out of range -> CRT_ERR_INVALID_ARG). */
crt_status crt_ray_code_encode(crt_ctx* ctx, const crt_bvh* bvh, int32_t code, const crt_ray* rays, int64_t n, uint32_t* keys, void* stream);
/* Stable LSD radix sort of (key, value) pairs, 4 passes of 8 bits, hand-written (no CUB).  All [device];
 * keys_in/vals_in are left intact; scratch >= crt_radix_sort_scratch_bytes(n). */
crt_status crt_radix_sort_pairs(crt_ctx* ctx, const uint32_t* keys_in, const int32_t* vals_in, int64_t n,
                                uint32_t* keys_out, int32_t* vals_out, void* scratch, size_t scratch_bytes, void* stream);
size_t crt_radix_sort_scratch_bytes(int64_t n);
/* The same sort for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the scratch is a static device array inside the library (17.3 MB per GPU that loads the library, held until the process
 * exits), so this call performs no cudaMalloc / cudaFree and calls no allocating library routine; the caller passes inputs and outputs
 * only.  n <= crt_radix_sort_noalloc_max_n() = 2,097,152 pairs, else CRT_ERR_UNSUPPORTED (use crt_radix_sort_pairs); CRT_ERR_STATE if
 * the array's device address could not be resolved when the context was created.  Same result as crt_radix_sort_pairs, bit for bit.
 * Every call on a device shares the one array (it keeps the last call's contents; nothing in it has to start at zero): calls whose
 * kernels OVERLAP on the GPU -- different streams, or different contexts of one device -- race; serialise them. */
crt_status crt_radix_sort_pairs_noalloc(crt_ctx* ctx, const uint32_t* keys_in, const int32_t* vals_in, int64_t n,
                                        uint32_t* keys_out, int32_t* vals_out, void* stream);
int64_t crt_radix_sort_noalloc_max_n(void);

/* ---- a5: BVH traversal ("the most time-consuming segment") ------------------------------- */
/* hits[i] = nearest intersection of rays[i] with tmin < t < tmax; ties -> lowest primitive id (D:R10).
 * Inactive rays (tmax < 0) give a miss.  rays, hits: [device], n_rays entries.
 * Ray origins: the default kernel's box test is conservative for origins within 16 scene extents of the scene box (rays that start on surfaces or at a
 * camera near the scene; crt_trace_primary checks the camera and switches by itself).  For rays from farther away set "trace_kernel" 4, the same kernel with
 * the any-origin test (3-4 % slower).  A per-ray check inside the default kernel was built twice (far rays traversed by their lane at fetch time; far rays
 * set aside and traversed by the last block) and removed: either form costs the persistent kernel 2-7 % through register pressure alone. */
crt_status crt_trace(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, crt_hit* hits, void* stream);
/* Work counters of the same traversal (a counting build of the kernel; used by bench.py for the roofline's
 * algorithmic FLOPs and by tests).  counters: [device] int64[4], ADDED to: [0] node visits (one visit = one 64-byte
 * node fetched and its two child boxes tested), [1] triangle tests, [2] active rays, [3] trace_kernel 8 only: node visits of
 * the 16-ray packets (one per half-warp and node; [0] then counts the lanes inside each visited node's box). */
crt_status crt_trace_stats(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, int64_t* counters, void* stream);

/* Diagnostic: crt_trace with the default kernel (16-bit nodes) plus four time marks per warp of the launch, for reading the tail of a
 * persistent launch (profiles/r02i).  marks: [device] uint64[4 * marks_capacity_warps]; warp w writes [4w] start, [4w+1] the moment it first
 * saw the ray list exhausted (0: never), [4w+2] end (all %globaltimer, ns), [4w+3] the largest number of node visits one of its lanes made
 * after [4w+1].  *n_warps (host) = warps of the launch; CRT_ERR_INVALID_ARG if the buffer is too small (148 SMs x 8 blocks x 4 warps fit in 4736). */
crt_status crt_trace_timeline(crt_ctx* ctx, const crt_bvh* bvh, const crt_ray* rays, int64_t n_rays, crt_hit* hits,
                              uint64_t* marks, int64_t marks_capacity_warps, int32_t* n_warps, void* stream);

/* ---- a6: shading and accumulation (D:R14) --------------------------------------------- */
/* For the segment just traced: miss -> radiance += throughput*env(d), path ends; emissive hit -> radiance +=
 * throughput*Le, path ends.  If is_last: accum[pixel] += radiance/spp for every path (accum: [device] float[h][w][3]). */
crt_status crt_shade_accumulate(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_frame* frame,
                                int32_t bounce, int32_t is_last, const crt_ray* rays, const crt_hit* hits,
                                const int32_t* ray_to_path, int64_t n_rays, crt_path_state* paths, float* accum, void* stream);

/* ---- whole frame ---------------------------------------------------------------------------------- */
/* primary -> shade(0) -> for b = 1..n_bounces { generate(b) -> trace -> shade(b) } on `stream`, using a caller
 * workspace of crt_frame_workspace_bytes() [device] bytes.  accum: [device] float[h][w][3], added to.
 * stage_ms (may be NULL, [host] float[8]): after the call has been synchronised with crt_frame_times(), the device
 * times of  0 primary, 1 shade, 2 generate(+encode+sort+permute), 3 secondary trace, 4 encode+sort+permute only.
 * n_secondary_out (may be NULL): [device] uint32[n_bounces] live secondary rays per bounce. */
crt_status crt_render_frame(crt_ctx* ctx, const crt_bvh* bvh, const crt_scene_mats* mats, const crt_camera* camera /*[host]*/,
                            const crt_frame* frame, const crt_order* order, int32_t n_bounces, float* accum,
                            uint32_t* n_secondary_out, void* workspace, size_t workspace_bytes, int32_t record_times, void* stream);
size_t crt_frame_workspace_bytes(const crt_frame* frame, const crt_order* order);
/* Synchronises the events recorded by the last crt_render_frame(record_times = 1) and adds their durations
 * (milliseconds) into stage_ms[0..4] ([host]). */
crt_status crt_frame_times(crt_ctx* ctx, float* stage_ms);
/* The same events per bounce (BASELINE config 5: encode+sort, traversal and throughput per bounce): adds to bounce_ms[3*(b-1) + k], b = 1 ..
 * n_bounces ([host] float[3*n_bounces]), k = 0 generation kernel, 1 encode+sort+permute, 2 traversal.  Call after crt_frame_times (which
 * synchronises) or any other synchronisation of the frame's stream. */
crt_status crt_frame_bounce_times(crt_ctx* ctx, int32_t n_bounces, float* bounce_ms);
/* Same frame through HOST buffers: materials [host] crt_material[n_materials], accum_host [host] float[h][w][3]
 * (read, added to, written back).  Copies materials + camera in and the image out on `stream` and synchronises.
 * workspace as above plus crt_frame_host_extra_bytes(). */
crt_status crt_render_frame_host(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials,
                                 const float* env /*[host] 6*/, const crt_camera* camera, const crt_frame* frame,
                                 const crt_order* order, int32_t n_bounces, float* accum_host, uint32_t* n_secondary_host,
                                 void* workspace, size_t workspace_bytes, void* stream);
/* The same with the accumulation image RESIDENT on the device between calls (it lives in the workspace, which the caller must
 * keep and not reuse for another image): reset != 0 zeroes it before this frame; image_host [host] float[h][w][3] only receives
 * the sum so far.  Per frame this moves the materials + camera in and one image out, half the bytes of crt_render_frame_host. */
crt_status crt_render_frame_host_resident(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials,
                                          const float* env /*[host] 6*/, const crt_camera* camera, const crt_frame* frame,
                                          const crt_order* order, int32_t n_bounces, int32_t reset, float* image_host,
                                          uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream);
/* As crt_render_frame_host_resident, but returns without synchronising: the copies and the frame are only ENQUEUED on `stream`;
 * image_host and n_secondary_host (both should be pinned memory, or the copies serialise) are valid once the caller has synchronised
 * the stream.  With one context + stream + workspace + host image per lane this keeps several host frames in flight. */
crt_status crt_render_frame_host_resident_async(crt_ctx* ctx, const crt_bvh* bvh, const crt_material* materials_host, int32_t n_materials,
                                                const float* env /*[host] 6*/, const crt_camera* camera, const crt_frame* frame,
                                                const crt_order* order, int32_t n_bounces, int32_t reset, float* image_host,
                                                uint32_t* n_secondary_host, void* workspace, size_t workspace_bytes, void* stream);
size_t crt_frame_host_extra_bytes(const crt_frame* frame, int32_t n_materials);

#ifdef __cplusplus
}
#endif
#endif /* CRT_H_ */
