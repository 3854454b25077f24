"""Test helpers: the oracle's stage-by-stage frame (CPU) and the same calls through libcrt (GPU).

Both take the same seeded scene from crt_inputs; neither side's values ever feed the other's expectations
except where a test deliberately feeds the ORACLE's buffers into one GPU stage (stage-wise parity).
"""
from __future__ import annotations

import numpy as np


def tol_close(a, b, rel, floor=1.0):
    """|a-b| <= rel * max(floor, |b|) elementwise"""
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return np.abs(a - b) <= rel * np.maximum(floor, np.abs(b))


def oracle_frame(O, scene, fr, n_bounces, mode, gw=1, gh=1, s=1, bvh=None, keep=True):
    """Runs the oracle stage by stage; returns dict with per-stage buffers (lists indexed by segment)."""
    bvh = bvh or O.Bvh(scene.verts)
    bounds = bvh.info()["bounds"]
    n_paths = fr.spp * fr.w * fr.h
    rays, hits, r2p = O.trace_primary(bvh, scene.camera, fr, mode, gw, gh, s)
    paths = O.paths_init(n_paths)
    accum = np.zeros((fr.h, fr.w, 3), np.float32)
    st = dict(bvh=bvh, bounds=bounds, rays=[rays], hits=[hits], r2p=[r2p], paths_before_gen=[], paths_after_gen=[], gen=[None], paths_after_shade=[])
    O.shade_accumulate(scene, fr, 0, n_bounces == 0, rays, hits, r2p, paths, accum)
    st["paths_after_shade"].append(paths.copy())
    for b in range(1, n_bounces + 1):
        st["paths_before_gen"].append(paths.copy())
        g = O.generate_secondary(scene, fr, b, mode, gw, gh, s, bounds, rays, hits, r2p, paths)
        st["paths_after_gen"].append(paths.copy())
        rays, r2p = g["rays"], g["ray_to_path"]
        hits = bvh.trace(rays)
        O.shade_accumulate(scene, fr, b, b == n_bounces, rays, hits, r2p, paths, accum)
        st["gen"].append(g); st["rays"].append(rays); st["hits"].append(hits); st["r2p"].append(r2p)
        st["paths_after_shade"].append(paths.copy())
    st["accum"] = accum
    return st


class GpuScene:
    """A scene uploaded through the binding: context, BVH, device materials."""

    def __init__(self, crt, scene, ctx=None, **bvh_kw):
        self.crt = crt
        self.ctx = ctx or crt.Context(0)
        self.scene = scene
        self.bvh = self.ctx.crt_build_bvh(scene.verts, scene.mat_id, **bvh_kw)
        self.mats_dev = self.ctx.upload(scene.materials)
        self.mats = self.ctx.scene_mats(self.mats_dev, len(scene.materials), scene.env)
        self.camera = crt.make_camera(scene.camera)

    def rays_to_dev(self, rays_struct):
        return self.ctx.upload(np.ascontiguousarray(rays_struct).view(np.float32).reshape(-1, 8))

    def hits_to_dev(self, hits_struct):
        return self.ctx.upload(np.ascontiguousarray(hits_struct).view(np.float32).reshape(-1, 4))

    def paths_to_dev(self, paths_struct):
        return self.ctx.upload(np.ascontiguousarray(paths_struct).view(np.float32).reshape(-1, 8))


def hits_np(O, hits_dev):
    return np.ascontiguousarray(hits_dev.cpu().numpy()).view(O.HIT_DTYPE).reshape(-1)


def rays_np(O, rays_dev):
    return np.ascontiguousarray(rays_dev.cpu().numpy()).view(O.RAY_DTYPE).reshape(-1)


def paths_np(O, paths_dev):
    return np.ascontiguousarray(paths_dev.cpu().numpy()).view(O.PATH_DTYPE).reshape(-1)


def compare_hits(h_gpu, h_orc, rays=None):
    """north_star's bar: ids identical for >= 99.99 % of rays, the rest only at t-ties within 1e-5 relative;
    t, u, v within 1e-4 relative.  Returns the fraction of identical ids."""
    same = h_gpu["prim"] == h_orc["prim"]
    frac = float(same.mean()) if len(same) else 1.0
    assert frac >= 0.9999, f"hit ids identical for only {frac:.6f}"
    diff = ~same
    if diff.any():
        assert np.all((h_gpu["prim"][diff] >= 0) & (h_orc["prim"][diff] >= 0)), "hit/miss disagreement"
        assert np.all(tol_close(h_gpu["t"][diff], h_orc["t"][diff], 1e-5, floor=0.0)), "id mismatch away from a t-tie"
    m = same & (h_orc["prim"] >= 0)
    assert np.all(tol_close(h_gpu["t"][m], h_orc["t"][m], 1e-4, floor=0.0))
    assert np.all(tol_close(h_gpu["u"][m], h_orc["u"][m], 1e-4)) and np.all(tol_close(h_gpu["v"][m], h_orc["v"][m], 1e-4))
    miss = same & (h_orc["prim"] < 0)
    assert np.array_equal(h_gpu["t"][miss], h_orc["t"][miss])
    return frac


def compare_rays(r_gpu, r_orc):
    """A-26: directions within 1e-5 absolute, origins within 1e-4 relative; activity flags identical."""
    act_g = r_gpu["tmax"] >= 0; act_o = r_orc["tmax"] >= 0
    assert np.array_equal(act_g, act_o)
    assert np.all(np.abs(r_gpu["d"][act_o].astype(np.float64) - r_orc["d"][act_o]) <= 1e-5)
    assert np.all(tol_close(r_gpu["o"][act_o], r_orc["o"][act_o], 1e-4))
    assert np.array_equal(r_gpu["tmin"][act_o], r_orc["tmin"][act_o]) and np.array_equal(r_gpu["tmax"][act_o], r_orc["tmax"][act_o])
    return float(np.mean(r_gpu[act_o].tobytes() == r_orc[act_o].tobytes())) if act_o.any() else 1.0


def rmse(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return float(np.sqrt(np.mean((a - b) ** 2)))
