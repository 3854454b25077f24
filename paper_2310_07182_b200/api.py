"""Thin ctypes binding of libcrt.so (include/crt.h).  Argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; this module converts torch CUDA
tensors to the raw device pointers of the C ABI and raises CrtError on a non-zero status.
torch is used for device memory and streams only.  There is NO CPU fallback: importing this
module without a built libcrt.so, or calling it without a CUDA device, fails loudly.

Buffer conventions (all torch tensors on the context's device, contiguous):
    rays   float32[n, 8]   ox oy oz tmin dx dy dz tmax          (crt_ray, 32-byte aligned)
    hits   float32[n, 4]   t u v prim(int32 bits)                (crt_hit); hit_prims() views the ids
    paths  float32[n, 8]   tr tg tb flags(u32 bits) lr lg lb pad (crt_path_state)
    mats   uint8[n_mat*32] crt_material records (from the numpy structured array of crt_inputs)
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

MODE_INDEPENDENT, MODE_MORTON_REORDER, MODE_DIRECT_REUSE = 0, 1, 2
MODES = {"independent": 0, "morton_reorder": 1, "direct_reuse": 2, "world_reuse": 3,
         "sort_origin": 4, "sort_reis": 5, "sort_costa": 6, "sort_twopoint": 7}
RAY_CODES = {"aila_compact": 0, "origin": 1, "reis": 2, "costa": 3, "twopoint": 4}
CRT_OK, CRT_ERR_INVALID_ARG, CRT_ERR_UNSUPPORTED, CRT_ERR_CUDA, CRT_ERR_STATE, CRT_ERR_NOMEM = range(6)
STATUS_NAMES = ["CRT_OK", "CRT_ERR_INVALID_ARG", "CRT_ERR_UNSUPPORTED", "CRT_ERR_CUDA", "CRT_ERR_STATE", "CRT_ERR_NOMEM"]

# every symbol include/crt.h declares (tests check that the library exports each of them)
EXPORTS = [
    "crt_create", "crt_destroy", "crt_last_error", "crt_set_option", "crt_measure_peaks",
    "crt_build_bvh", "crt_bvh_destroy", "crt_bvh_get_info", "crt_bvh_check", "crt_layout", "crt_paths_init",
    "crt_trace_primary", "crt_generate_secondary", "crt_generate_secondary_scratch_bytes",
    "crt_morton_encode", "crt_ray_code_encode", "crt_radix_sort_pairs", "crt_radix_sort_scratch_bytes", "crt_radix_sort_pairs_noalloc", "crt_radix_sort_noalloc_max_n", "crt_trace", "crt_trace_stats", "crt_trace_timeline",
    "crt_shade_accumulate", "crt_render_frame", "crt_frame_workspace_bytes", "crt_frame_times", "crt_frame_bounce_times",
    "crt_render_frame_host", "crt_render_frame_host_resident", "crt_render_frame_host_resident_async", "crt_frame_host_extra_bytes",
]


class CrtError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else status}: {message}")
        self.status = status


class Frame(C.Structure):
    _fields_ = [("w", C.c_int32), ("h", C.c_int32), ("spp", C.c_int32), ("seed", C.c_int32), ("frame", C.c_int32)]


class Order(C.Structure):
    _fields_ = [("mode", C.c_int32), ("group_w", C.c_int32), ("group_h", C.c_int32), ("stride", C.c_int32), ("stride_y", C.c_int32), ("partition_rule", C.c_int32)]


class Camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("U", C.c_float * 3), ("V", C.c_float * 3), ("W", C.c_float * 3)]


class SceneMats(C.Structure):
    _fields_ = [("materials", C.c_void_p), ("n_materials", C.c_int32), ("env", C.c_float * 6)]


class BvhParams(C.Structure):
    _fields_ = [("max_leaf", C.c_int32), ("sah_bins", C.c_int32), ("cost_traversal", C.c_float), ("cost_intersect", C.c_float),
                ("n_threads", C.c_int32), ("builder", C.c_int32), ("ploc_radius", C.c_int32), ("presplit", C.c_float), ("optimize", C.c_int32)]


class BvhInfo(C.Structure):
    _fields_ = [("n_tris", C.c_int64), ("n_nodes", C.c_int64), ("device_bytes", C.c_int64), ("bounds", C.c_float * 6),
                ("sah_cost", C.c_double), ("depth", C.c_int32), ("max_leaf", C.c_int32), ("build_seconds", C.c_double),
                ("n_wide_nodes", C.c_int64), ("wide_depth", C.c_int32), ("q16_inflation_pct", C.c_int32),
                ("builder", C.c_int32), ("build_rounds", C.c_int32), ("device_build_seconds", C.c_double), ("layout_seconds", C.c_double),
                ("n_refs", C.c_int64), ("optimize_iterations", C.c_int32), ("reserved", C.c_int32)]


_lib = None


def lib():
    """Loads libcrt.so (building it with nvcc first when the sources are newer).  Raises if it cannot."""
    global _lib
    if _lib is None:
        path = _build.LIB
        try:
            path = _build.build()
        except Exception as e:  # no nvcc on this machine: use the shipped library if there is one
            if not os.path.exists(path):
                raise ImportError(f"libcrt.so is missing and could not be built ({e}); there is no CPU fallback") from e
        L = C.CDLL(path)
        L.crt_last_error.restype = C.c_char_p
        L.crt_last_error.argtypes = [C.c_void_p]
        for name in ("crt_generate_secondary_scratch_bytes", "crt_radix_sort_scratch_bytes", "crt_frame_workspace_bytes",
                     "crt_frame_host_extra_bytes"):
            getattr(L, name).restype = C.c_size_t
        L.crt_radix_sort_noalloc_max_n.restype = C.c_int64
        _lib = L
    return _lib


def _ptr(t):
    if t is None:
        return C.c_void_p(None)
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous(), "libcrt buffers must be contiguous"
        return C.c_void_p(t.data_ptr())
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    raise TypeError(type(t))


def _stream(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def make_frame(w, h, spp=1, seed=0, frame=0):
    return Frame(int(w), int(h), int(spp), int(seed), int(frame))


def make_order(mode, group_w=1, group_h=1, stride=1, stride_y=0, partition_rule=0):
    """partition_rule: 0 = the paper's shuffled numbers (affine map), 1 = regular lattice, 2 = LCG sequence (include/crt.h).  `stride` also
    accepts the packed form the tests use: bits 0-13 horizontal stride, bit 14 lattice rule, bit 15 LCG-sequence rule, high half vertical stride."""
    stride = int(stride)
    if stride >> 14:
        partition_rule = partition_rule or (1 if (stride >> 14) & 1 else (2 if (stride >> 15) & 1 else 0))
        stride, stride_y = stride & 0x3fff, (stride >> 16) or stride_y
    return Order(MODES[mode] if isinstance(mode, str) else int(mode), int(group_w), int(group_h), int(stride), int(stride_y), int(partition_rule))


def order_for_tile(mode, tile_w, tile_h, k):
    """The paper's native parametrisation: a tile_w x tile_h tile and groups of k rays, all powers of two."""
    gw = min(k, tile_w); gh = k // gw
    return make_order(mode, gw, gh, tile_w // gw, tile_h // gh)


def make_camera(cam12):
    c = np.asarray(cam12, np.float32).reshape(12)
    return Camera((C.c_float * 3)(*c[0:3]), (C.c_float * 3)(*c[3:6]), (C.c_float * 3)(*c[6:9]), (C.c_float * 3)(*c[9:12]))


def crt_layout(frame, order):
    """(n_paths, n_slots, n_groups) of the slot space (include/crt.h 'Index spaces')."""
    a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
    st = lib().crt_layout(C.byref(frame), C.byref(order), C.byref(a), C.byref(b), C.byref(c))
    if st != CRT_OK:
        raise CrtError(st, lib().crt_last_error(None).decode())
    return a.value, b.value, c.value


class Bvh:
    def __init__(self, ctx, handle):
        self.ctx, self.handle = ctx, handle

    def info(self):
        o = BvhInfo()
        self.ctx._check(lib().crt_bvh_get_info(self.handle, C.byref(o)))
        return {"n_tris": o.n_tris, "n_nodes": o.n_nodes, "device_bytes": o.device_bytes, "bounds": np.array(list(o.bounds), np.float32),
                "sah_cost": o.sah_cost, "depth": o.depth, "max_leaf": o.max_leaf, "build_seconds": o.build_seconds,
                "n_wide_nodes": o.n_wide_nodes, "wide_depth": o.wide_depth, "q16_inflation_pct": o.q16_inflation_pct,
                "builder": o.builder, "build_rounds": o.build_rounds, "device_build_seconds": o.device_build_seconds, "layout_seconds": o.layout_seconds, "n_refs": o.n_refs, "optimize_iterations": o.optimize_iterations}

    def check(self):
        v = C.c_int32(-1)
        self.ctx._check(lib().crt_bvh_check(self.handle, C.byref(v)))
        return v.value

    def destroy(self):
        if self.handle:
            lib().crt_bvh_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Context:
    """crt_ctx on one CUDA device.  Method names are the C entry points'."""

    def __init__(self, device=0):
        if not torch.cuda.is_available():
            raise CrtError(CRT_ERR_CUDA, "no CUDA device; libcrt has no CPU fallback")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        torch.zeros(1, device=self.device)          # make sure torch's primary context is current
        h = C.c_void_p()
        st = lib().crt_create(C.c_int32(device), C.byref(h))
        if st != CRT_OK:
            raise CrtError(st, lib().crt_last_error(None).decode())
        self.handle = h

    def _check(self, st):
        if st != CRT_OK:
            raise CrtError(st, lib().crt_last_error(self.handle).decode())

    def close(self):
        if getattr(self, "handle", None):
            lib().crt_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers ----------------------------------------------------------------------------------
    def empty(self, shape, dtype=torch.float32):
        return torch.empty(shape, dtype=dtype, device=self.device)

    def upload(self, a, dtype=None):
        a = np.ascontiguousarray(a)
        if a.dtype.fields is not None:                 # structured array -> bytes
            a = a.view(np.uint8)
        t = torch.from_numpy(a).to(self.device)
        return t if dtype is None else t.to(dtype)

    def scene_mats(self, materials_dev, n_materials, env):
        e = np.asarray(env, np.float32).reshape(6)
        return SceneMats(C.c_void_p(materials_dev.data_ptr()), int(n_materials), (C.c_float * 6)(*e))

    def crt_set_option(self, key, value):
        self._check(lib().crt_set_option(self.handle, key.encode(), C.c_int64(int(value))))

    def crt_measure_peaks(self):
        a, b = C.c_double(), C.c_double()
        self._check(lib().crt_measure_peaks(self.handle, C.byref(a), C.byref(b)))
        return a.value, b.value

    # ---- a0 -----------------------------------------------------------------------------------------
    def crt_build_bvh(self, verts, mat_id, max_leaf=3, sah_bins=64, n_threads=0, cost_traversal=1.0, cost_intersect=1.0, builder=0, ploc_radius=0, presplit=1.0 / 16, optimize=20):
        """verts: numpy float32[n,3,3] or torch tensor (host or device); mat_id int32[n].  builder: 0 host SAH, 1 device PLOC."""
        if isinstance(verts, np.ndarray):
            verts = np.ascontiguousarray(verts, np.float32)
            mat_id = np.ascontiguousarray(mat_id, np.int32)
            n = verts.size // 9
        else:
            n = verts.numel() // 9
        pr = BvhParams(max_leaf, sah_bins, cost_traversal, cost_intersect, n_threads, int(builder), int(ploc_radius), float(presplit), int(optimize))
        h = C.c_void_p()
        self._check(lib().crt_build_bvh(self.handle, _ptr(verts), _ptr(mat_id), C.c_int64(n), C.byref(pr), C.byref(h)))
        return Bvh(self, h)

    # ---- path state -----------------------------------------------------------------------------------
    def crt_paths_init(self, paths, stream=None):
        self._check(lib().crt_paths_init(self.handle, _ptr(paths), C.c_int64(paths.shape[0]), _stream(stream)))

    # ---- a1 -----------------------------------------------------------------------------------------
    def crt_trace_primary(self, bvh, camera, frame, order, stream=None):
        _, ns, _ = crt_layout(frame, order)
        rays, hits, r2p = self.empty((ns, 8)), self.empty((ns, 4)), self.empty((ns,), torch.int32)
        self._check(lib().crt_trace_primary(self.handle, bvh.handle, C.byref(camera), C.byref(frame), C.byref(order), _ptr(rays), _ptr(hits),
                                            _ptr(r2p), _stream(stream)))
        return rays, hits, r2p

    # ---- a2-a4 ----------------------------------------------------------------------------------------
    def crt_generate_secondary(self, bvh, mats, frame, bounce, order, prev_rays, prev_hits, prev_r2p, paths, stream=None):
        """Returns dict(rays, ray_to_path, group_id, dir_src, group_class, n_active(tensor uint32 as int32[1]))."""
        _, ns, ng = crt_layout(frame, order)
        out = dict(rays=self.empty((ns, 8)), ray_to_path=self.empty((ns,), torch.int32), group_id=self.empty((ns,), torch.int32),
                   dir_src=self.empty((ns,), torch.int32), group_class=torch.zeros((max(ng, 1),), dtype=torch.uint8, device=self.device),
                   n_active=torch.zeros((1,), dtype=torch.int32, device=self.device))
        nb = lib().crt_generate_secondary_scratch_bytes(C.byref(frame), C.byref(order))
        scratch = self.empty((max(nb, 256),), torch.uint8)
        self._check(lib().crt_generate_secondary(self.handle, bvh.handle, C.byref(mats), C.byref(frame), C.c_int32(bounce), C.byref(order),
                                                 _ptr(prev_rays), _ptr(prev_hits), _ptr(prev_r2p), _ptr(paths), _ptr(out["rays"]),
                                                 _ptr(out["ray_to_path"]), _ptr(out["group_id"]), _ptr(out["dir_src"]), _ptr(out["group_class"]),
                                                 _ptr(out["n_active"]), _ptr(scratch), C.c_size_t(scratch.numel()), _stream(stream)))
        out["group_class"] = out["group_class"][:ng]
        return out

    def crt_morton_encode(self, bvh, rays, stream=None):
        keys = self.empty((rays.shape[0],), torch.int32)
        self._check(lib().crt_morton_encode(self.handle, bvh.handle, _ptr(rays), C.c_int64(rays.shape[0]), _ptr(keys), _stream(stream)))
        return keys

    def crt_ray_code_encode(self, bvh, code, rays, stream=None):
        keys = self.empty((rays.shape[0],), torch.int32)
        self._check(lib().crt_ray_code_encode(self.handle, bvh.handle, C.c_int32(int(code)), _ptr(rays), C.c_int64(rays.shape[0]), _ptr(keys), _stream(stream)))
        return keys

    def crt_radix_sort_pairs(self, keys, vals, stream=None):
        n = keys.shape[0]
        ko, vo = torch.empty_like(keys), torch.empty_like(vals)
        nb = lib().crt_radix_sort_scratch_bytes(C.c_int64(n))
        scratch = self.empty((max(nb, 256),), torch.uint8)
        self._check(lib().crt_radix_sort_pairs(self.handle, _ptr(keys), _ptr(vals), C.c_int64(n), _ptr(ko), _ptr(vo), _ptr(scratch),
                                               C.c_size_t(scratch.numel()), _stream(stream)))
        return ko, vo

    def crt_radix_sort_pairs_noalloc(self, keys, vals, keys_out, vals_out, stream=None):
        """The same sort with the library's static scratch (no allocation inside the call; n <= crt_radix_sort_noalloc_max_n()).
        The caller passes the output tensors; calls that overlap on the GPU race (include/crt.h)."""
        self._check(lib().crt_radix_sort_pairs_noalloc(self.handle, _ptr(keys), _ptr(vals), C.c_int64(keys.shape[0]), _ptr(keys_out), _ptr(vals_out), _stream(stream)))
        return keys_out, vals_out

    # ---- a5 -----------------------------------------------------------------------------------------
    def crt_trace(self, bvh, rays, hits=None, stream=None):
        n = rays.shape[0]
        if hits is None:
            hits = self.empty((n, 4))
        self._check(lib().crt_trace(self.handle, bvh.handle, _ptr(rays), C.c_int64(n), _ptr(hits), _stream(stream)))
        return hits

    def crt_trace_stats(self, bvh, rays, stream=None, full=False):
        """(node_visits, triangle_tests, active_rays) of one traversal of `rays` (counting variant of the kernel); full: all four counters
        (the fourth: half-warp node visits of trace_kernel 8, else 0)."""
        cnt = torch.zeros((4,), dtype=torch.int64, device=self.device)
        self._check(lib().crt_trace_stats(self.handle, bvh.handle, _ptr(rays), C.c_int64(rays.shape[0]), _ptr(cnt), _stream(stream)))
        c = cnt.cpu().tolist()
        return tuple(c) if full else (c[0], c[1], c[2])

    def crt_trace_timeline(self, bvh, rays, hits=None, stream=None):
        """crt_trace with per-warp time marks: returns (hits, marks) with marks an int64 array [n_warps, 4] on the host:
        start ns, ray-list-exhausted ns (0: never seen), end ns, largest number of node visits of a lane after exhaustion."""
        n = rays.shape[0]
        if hits is None:
            hits = self.empty((n, 4))
        cap = 148 * 8 * 4 * 2
        marks = torch.zeros((cap, 4), dtype=torch.int64, device=self.device)
        nw = C.c_int32(0)
        self._check(lib().crt_trace_timeline(self.handle, bvh.handle, _ptr(rays), C.c_int64(n), _ptr(hits), _ptr(marks), C.c_int64(cap), C.byref(nw), _stream(stream)))
        return hits, marks[: nw.value].cpu().numpy()

    # ---- a6 -----------------------------------------------------------------------------------------
    def crt_shade_accumulate(self, bvh, mats, frame, bounce, is_last, rays, hits, r2p, paths, accum, stream=None):
        self._check(lib().crt_shade_accumulate(self.handle, bvh.handle, C.byref(mats), C.byref(frame), C.c_int32(bounce), C.c_int32(int(is_last)),
                                               _ptr(rays), _ptr(hits), _ptr(r2p), C.c_int64(rays.shape[0]), _ptr(paths), _ptr(accum), _stream(stream)))

    # ---- whole frame ----------------------------------------------------------------------------------
    def frame_workspace(self, frame, order, host_materials=0):
        nb = lib().crt_frame_workspace_bytes(C.byref(frame), C.byref(order))
        if host_materials:
            nb += lib().crt_frame_host_extra_bytes(C.byref(frame), C.c_int32(host_materials))
        return self.empty((nb + 256,), torch.uint8)

    def crt_render_frame(self, bvh, mats, camera, frame, order, n_bounces, accum, workspace, n_secondary=None, record_times=False, stream=None):
        self._check(lib().crt_render_frame(self.handle, bvh.handle, C.byref(mats), C.byref(camera), C.byref(frame), C.byref(order),
                                           C.c_int32(n_bounces), _ptr(accum), _ptr(n_secondary), _ptr(workspace), C.c_size_t(workspace.numel()),
                                           C.c_int32(int(record_times)), _stream(stream)))

    def crt_frame_times(self, stage_ms=None):
        """Adds the device times (ms) of the last recorded frame into stage_ms (numpy float32[8])."""
        if stage_ms is None:
            stage_ms = np.zeros(8, np.float32)
        self._check(lib().crt_frame_times(self.handle, _ptr(stage_ms)))
        return stage_ms

    def crt_frame_bounce_times(self, n_bounces, bounce_ms=None):
        """Adds the last recorded frame's device times (ms) per bounce into bounce_ms (numpy float32[n_bounces, 3]: generate, encode+sort+permute, trace)."""
        if bounce_ms is None:
            bounce_ms = np.zeros((n_bounces, 3), np.float32)
        self._check(lib().crt_frame_bounce_times(self.handle, C.c_int32(n_bounces), _ptr(bounce_ms)))
        return bounce_ms

    def crt_render_frame_host(self, bvh, materials_host, env, camera, frame, order, n_bounces, accum_host, n_secondary_host, workspace, stream=None):
        """materials_host: numpy structured array; accum_host: numpy/pinned torch float32[h,w,3]; n_secondary_host: numpy uint32[n_bounces]."""
        e = np.asarray(env, np.float32).reshape(6)
        mh = np.ascontiguousarray(materials_host)
        self._check(lib().crt_render_frame_host(self.handle, bvh.handle, C.c_void_p(mh.ctypes.data), C.c_int32(len(mh)), _ptr(e), C.byref(camera),
                                                C.byref(frame), C.byref(order), C.c_int32(n_bounces), _ptr(accum_host), _ptr(n_secondary_host),
                                                _ptr(workspace), C.c_size_t(workspace.numel()), _stream(stream)))

    def crt_render_frame_host_resident(self, bvh, materials_host, env, camera, frame, order, n_bounces, reset, image_host, n_secondary_host, workspace, stream=None,
                                       wait=True):
        """as crt_render_frame_host, with the accumulation image resident in `workspace` between calls; image_host receives the sum so far.
        wait=False: only enqueue (crt_render_frame_host_resident_async); the outputs are valid after the stream has been synchronised."""
        e = np.asarray(env, np.float32).reshape(6)
        mh = np.ascontiguousarray(materials_host)
        fn = lib().crt_render_frame_host_resident if wait else lib().crt_render_frame_host_resident_async
        self._check(fn(self.handle, bvh.handle, C.c_void_p(mh.ctypes.data), C.c_int32(len(mh)), _ptr(e), C.byref(camera),
                                                         C.byref(frame), C.byref(order), C.c_int32(n_bounces), C.c_int32(1 if reset else 0), _ptr(image_host),
                                                         _ptr(n_secondary_host), _ptr(workspace), C.c_size_t(workspace.numel()), _stream(stream)))


def hit_prims(hits):
    """int32 view of the primitive ids of a hits tensor."""
    return hits.view(torch.int32)[:, 3]


def path_flags(paths):
    return paths.view(torch.int32)[:, 3]
