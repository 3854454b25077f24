"""ctypes binding of oracle/crt_oracle.c (TEST INFRASTRUCTURE ONLY).

Argument marshalling only; every computation is in the C file, which cites the
paper.  `build()` compiles liboracle.so (fp32, the parity oracle) and
liboracle64.so (same procedure in fp64, used to bound rounding error).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "crt_oracle.c")

RAY_DTYPE = np.dtype([("o", "<f4", 3), ("tmin", "<f4"), ("d", "<f4", 3), ("tmax", "<f4")])
HIT_DTYPE = np.dtype([("t", "<f4"), ("u", "<f4"), ("v", "<f4"), ("prim", "<i4")])
PATH_DTYPE = np.dtype([("T", "<f4", 3), ("flags", "<u4"), ("L", "<f4", 3), ("pad", "<u4")])
MODE_INDEPENDENT, MODE_MORTON, MODE_REUSE = 0, 1, 2
MODES = {"independent": 0, "morton_reorder": 1, "direct_reuse": 2, "world_reuse": 3,
         "sort_origin": 4, "sort_reis": 5, "sort_costa": 6, "sort_twopoint": 7}
RAY_CODES = {"aila_compact": 0, "origin": 1, "reis": 2, "costa": 3, "twopoint": 4}
CLASS_EMPTY, CLASS_DIFFUSE, CLASS_GLOSSY, CLASS_HYBRID = 0, 1, 2, 3


class Frame(C.Structure):
    _fields_ = [("w", C.c_int32), ("h", C.c_int32), ("spp", C.c_int32), ("seed", C.c_int32), ("frame", C.c_int32)]


# ORACLE_SANITIZE=1: the same two libraries built with AddressSanitizer + UndefinedBehaviorSanitizer.  Run the CPU suite as
#   ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests/test_oracle_*.py -q
_SAN = os.environ.get("ORACLE_SANITIZE") == "1"
_SUFFIX = "_san" if _SAN else ""
_SAN_FLAGS = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"] if _SAN else []


def build(force=False):
    outs = []
    for name, flags in ((f"liboracle{_SUFFIX}.so", _SAN_FLAGS), (f"liboracle64{_SUFFIX}.so", ["-DORC_REAL=double"] + _SAN_FLAGS)):
        out = os.path.join(_HERE, name)
        outs.append(out)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-Wall", "-Wno-misleading-indentation", "-D_POSIX_C_SOURCE=200809L", *flags, "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return outs


_libs = {}


def _lib(fp64=False):
    key = bool(fp64)
    if key not in _libs:
        build()
        lib = C.CDLL(os.path.join(_HERE, f"liboracle64{_SUFFIX}.so" if fp64 else f"liboracle{_SUFFIX}.so"))
        lib.orc_bvh_build.restype = C.c_void_p
        lib.orc_bvh_build.argtypes = [C.c_void_p, C.c_int64]
        lib.orc_bvh_free.argtypes = [C.c_void_p]
        lib.orc_bvh_check.argtypes = [C.c_void_p]
        lib.orc_bvh_check.restype = C.c_int32
        lib.orc_n_slots.restype = C.c_int64
        lib.orc_n_groups.restype = C.c_int64
        lib.orc_u01.restype = C.c_float
        lib.orc_u01.argtypes = [C.c_uint32]
        lib.orc_morton_code.restype = C.c_uint32
        _libs[key] = lib
    return _libs[key]


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, np.float32)


def philox(c0, c1, c2, c3, k0, k1):
    out = (C.c_uint32 * 4)()
    _lib().orc_philox(C.c_uint32(c0), C.c_uint32(c1), C.c_uint32(c2), C.c_uint32(c3), C.c_uint32(k0), C.c_uint32(k1), out)
    return tuple(int(x) for x in out)


def u01(r):
    return float(_lib().orc_u01(r))


def sincos2pi(u, fp64=False):
    s, c = C.c_float(), C.c_float()
    _lib(fp64).orc_sincos2pi(C.c_float(u), C.byref(s), C.byref(c))
    return s.value, c.value


def trace_brute(verts, rays, fp64=False):
    verts = _f32(verts); rays = np.ascontiguousarray(rays)
    hits = np.zeros(len(rays), HIT_DTYPE)
    _lib(fp64).orc_trace_brute(_p(verts), C.c_int64(len(verts)), _p(rays), C.c_int64(len(rays)), _p(hits))
    return hits


class Bvh:
    """Owns the oracle's BVH (and keeps the vertex array alive)."""

    def __init__(self, verts, fp64=False):
        self.lib = _lib(fp64)
        self.verts = _f32(verts).reshape(-1, 3, 3)
        self.handle = C.c_void_p(self.lib.orc_bvh_build(_p(self.verts), C.c_int64(len(self.verts))))

    def __del__(self):
        if getattr(self, "handle", None):
            self.lib.orc_bvh_free(self.handle); self.handle = None

    def info(self):
        n = C.c_int64(); root = (C.c_float * 6)(); depth = C.c_int32(); sah = C.c_double()
        self.lib.orc_bvh_info(self.handle, C.byref(n), root, C.byref(depth), C.byref(sah))
        return {"n_nodes": n.value, "bounds": np.array(list(root), np.float32), "depth": depth.value, "sah": sah.value}

    def check(self):
        return int(self.lib.orc_bvh_check(self.handle))

    def trace(self, rays, counters=None):
        rays = np.ascontiguousarray(rays)
        hits = np.zeros(len(rays), HIT_DTYPE)
        cnt = np.zeros(2, np.int64)
        self.lib.orc_trace(self.handle, _p(rays), C.c_int64(len(rays)), _p(hits), _p(cnt))
        if counters is not None:
            counters += cnt
        return hits


def frame(w, h, spp=1, seed=0, frame=0):
    return Frame(w, h, spp, seed, frame)


def n_slots(fr, mode, gw=1, gh=1, s=1):
    return int(_lib().orc_n_slots(C.byref(fr), mode, gw, gh, s))


def n_groups(fr, mode, gw=1, gh=1, s=1):
    return int(_lib().orc_n_groups(C.byref(fr), mode, gw, gh, s))


def partition(fr, mode, gw=1, gh=1, s=1):
    out = np.empty(n_slots(fr, mode, gw, gh, s), np.int32)
    _lib().orc_partition(C.byref(fr), mode, gw, gh, s, _p(out))
    return out


def trace_primary(bvh, cam, fr, mode, gw=1, gh=1, s=1):
    n = n_slots(fr, mode, gw, gh, s)
    rays = np.zeros(n, RAY_DTYPE); hits = np.zeros(n, HIT_DTYPE); r2p = np.zeros(n, np.int32)
    cam = _f32(cam)
    bvh.lib.orc_trace_primary(bvh.handle, _p(cam), C.byref(fr), mode, gw, gh, s, _p(rays), _p(hits), _p(r2p))
    return rays, hits, r2p


def paths_init(n):
    p = np.zeros(n, PATH_DTYPE)
    _lib().orc_paths_init(_p(p), C.c_int64(n))
    return p


def generate_secondary(scene, fr, bounce, mode, gw, gh, s, bounds, prev_rays, prev_hits, prev_r2p, paths, fp64=False):
    """paths is updated in place.  Returns dict of outputs."""
    n = n_slots(fr, mode, gw, gh, s)
    ng = n_groups(fr, mode, gw, gh, s)
    out = dict(rays=np.zeros(n, RAY_DTYPE), ray_to_path=np.zeros(n, np.int32), group_id=np.zeros(n, np.int32),
               dir_src=np.zeros(n, np.int32), group_class=np.zeros(ng, np.uint8), local_dir=np.zeros((n, 3), np.float32))
    na = C.c_uint32()
    verts = _f32(scene.verts); mid = np.ascontiguousarray(scene.mat_id, np.int32); mats = np.ascontiguousarray(scene.materials)
    bounds = _f32(bounds)
    _lib(fp64).orc_generate_secondary(_p(verts), _p(mid), _p(mats), C.byref(fr), bounce, mode, gw, gh, s, _p(bounds),
                                      _p(np.ascontiguousarray(prev_rays)), _p(np.ascontiguousarray(prev_hits)),
                                      _p(np.ascontiguousarray(prev_r2p)), _p(paths),
                                      _p(out["rays"]), _p(out["ray_to_path"]), _p(out["group_id"]), _p(out["dir_src"]),
                                      _p(out["group_class"]), C.byref(na), _p(out["local_dir"]))
    out["n_active"] = na.value
    return out


def morton_encode(rays, bounds):
    rays = np.ascontiguousarray(rays); keys = np.zeros(len(rays), np.uint32); bounds = _f32(bounds)
    _lib().orc_morton_encode(_p(rays), C.c_int64(len(rays)), _p(bounds), _p(keys))
    return keys


def ray_code_encode(code, rays, bounds):
    """sort key of every ray for one of RAY_CODES (D:R12, R19)"""
    rays = np.ascontiguousarray(rays); keys = np.zeros(len(rays), np.uint32); bounds = _f32(bounds)
    _lib().orc_ray_code_encode(C.c_int32(int(code)), _p(rays), C.c_int64(len(rays)), _p(bounds), _p(keys))
    return keys


def sort_keys(keys):
    keys = np.ascontiguousarray(keys, np.uint32); order = np.zeros(len(keys), np.int32)
    _lib().orc_sort_keys(_p(keys), C.c_int64(len(keys)), _p(order))
    return order


def shade_accumulate(scene, fr, bounce, is_last, rays, hits, r2p, paths, accum):
    mid = np.ascontiguousarray(scene.mat_id, np.int32); mats = np.ascontiguousarray(scene.materials); env = _f32(scene.env)
    _lib().orc_shade_accumulate(_p(mid), _p(mats), _p(env), C.byref(fr), bounce, int(is_last), _p(np.ascontiguousarray(rays)),
                                _p(np.ascontiguousarray(hits)), _p(np.ascontiguousarray(r2p)), C.c_int64(len(rays)), _p(paths), _p(accum))


def render_frame(bvh, scene, fr, n_bounces, mode, gw=1, gh=1, s=1, accum=None):
    """Whole frame; returns (accum[h,w,3], times[4] = generate, trace, shade, primary seconds, counts[3])."""
    if accum is None:
        accum = np.zeros((fr.h, fr.w, 3), np.float32)
    times = np.zeros(4, np.float64); counts = np.zeros(3, np.int64)
    mid = np.ascontiguousarray(scene.mat_id, np.int32); mats = np.ascontiguousarray(scene.materials)
    env = _f32(scene.env); cam = _f32(scene.camera)
    bvh.lib.orc_render_frame(bvh.handle, _p(mid), _p(mats), _p(env), _p(cam), C.byref(fr), n_bounces, mode, gw, gh, s,
                             _p(accum), _p(times), _p(counts))
    return accum, times, counts


def sample_cosine(u1, u2):
    wi = (C.c_float * 3)()
    _lib().orc_test_sample_cosine(C.c_float(u1), C.c_float(u2), wi)
    return np.array(list(wi))


def sample_ggx(wo, alpha, u1, u2, fp64=False):
    wi = (C.c_float * 3)(); wt = (C.c_float * 3)()
    wo = (C.c_float * 3)(*[float(x) for x in wo])
    ok = _lib(fp64).orc_test_sample_ggx(wo, C.c_float(alpha), C.c_float(u1), C.c_float(u2), wi, wt)
    return bool(ok), np.array(list(wi)), float(wt[0])


def sample_ggx_f0(wo, alpha, albedo, u1, u2, fp64=False):
    """sample_ggx with F0 = albedo (RGB): (valid, wi[3], weight[3])"""
    wi = (C.c_float * 3)(); wt = (C.c_float * 3)()
    wo = (C.c_float * 3)(*[float(x) for x in wo]); al = (C.c_float * 3)(*[float(x) for x in albedo])
    ok = _lib(fp64).orc_test_sample_ggx_f0(wo, C.c_float(alpha), al, C.c_float(u1), C.c_float(u2), wi, wt)
    return bool(ok), np.array(list(wi)), np.array(list(wt))


def ggx_weight(wo, wi, alpha, albedo, fp64=False):
    """weight of a GIVEN exit direction under a GGX material (world-space reuse, D:R18): (valid, weight[3])"""
    wt = (C.c_float * 3)()
    wo = (C.c_float * 3)(*[float(x) for x in wo]); wi = (C.c_float * 3)(*[float(x) for x in wi])
    al = (C.c_float * 3)(*[float(x) for x in albedo])
    ok = _lib(fp64).orc_test_ggx_weight(wo, wi, C.c_float(alpha), al, wt)
    return bool(ok), np.array(list(wt))
