"""Pins for the oracle's intersection: brute force (the plain definition), analytic
plane and sphere hits, BVH invariants, fp64 cross-check (CPU only)."""
import numpy as np
import pytest

import crt_inputs as I


def _rays(arr, O):
    return np.ascontiguousarray(arr).view(O.RAY_DTYPE).reshape(-1)


@pytest.mark.parametrize("scene_fn,n_rays", [
    (lambda: I.cornell(), 3000),
    (lambda: I.interior(n_boxes=20, n_spheres=5, subdiv=2), 1500),
    (lambda: I.landscape(n=48, n_trees=10), 1500),
    (lambda: I.furnace_sphere(2), 2000),
])
def test_bvh_equals_brute_force(oracle, scene_fn, n_rays):
    s = scene_fn()
    b = oracle.Bvh(s.verts)
    assert b.check() == 0
    info = b.info()
    v = s.verts.reshape(-1, 3)
    assert np.array_equal(info["bounds"], np.concatenate([v.min(0), v.max(0)]))
    rays = _rays(I.random_rays(3, n_rays, info["bounds"][:3], info["bounds"][3:], inactive_frac=0.05), oracle)
    # half the rays start on geometry-aligned positions / axis-aligned directions (zeros in d)
    rays["d"][::7] = np.eye(3, dtype=np.float32)[np.arange(len(rays[::7])) % 3]
    hb = oracle.trace_brute(s.verts, rays)
    ht = b.trace(rays)
    assert np.array_equal(hb, ht)                       # 100 %, including t, u, v bits
    assert (hb["prim"] >= 0).mean() > 0.2
    assert np.all(hb["prim"][rays["tmax"] < 0] == -1)


def test_tie_break_lowest_primitive_id(oracle):
    s = I.cornell()
    verts = np.concatenate([s.verts, s.verts[::-1]])     # every triangle twice, second copy reversed order
    n = len(s.verts)
    b = oracle.Bvh(verts)
    rays = _rays(I.random_rays(5, 1500, [0, 0, 0], [1, 1, 1]), oracle)
    h = b.trace(rays)
    hb = oracle.trace_brute(verts, rays)
    assert np.array_equal(h, hb)
    hit = h["prim"] >= 0
    assert hit.sum() > 500 and np.all(h["prim"][hit] < n)


def test_tmin_tmax_window(oracle):
    q = I.floor_plane(tess=2)
    b = oracle.Bvh(q.verts)
    r = np.zeros(4, oracle.RAY_DTYPE)
    r["o"] = (0.1, 2.0, 0.2); r["d"] = (0, -1, 0); r["tmin"] = (0, 0, 2.5, 0); r["tmax"] = (1e30, 1.5, 1e30, -1)
    h = b.trace(r)
    assert h["prim"][0] >= 0 and abs(h["t"][0] - 2.0) < 1e-6
    assert list(h["prim"][1:]) == [-1, -1, -1]
    assert h["t"][1] == np.float32(1.5) and h["t"][3] == -1.0


def test_analytic_plane_hits_cornell(oracle):
    """Rays from inside the box toward the axis-aligned walls: t = (c - o_k)/d_k."""
    s = I.cornell()
    b = oracle.Bvh(s.verts)
    rng = np.random.default_rng(11)
    n = 2000
    r = np.zeros(n, oracle.RAY_DTYPE)
    r["o"] = (0.5, 0.8, 0.9) + rng.uniform(-0.05, 0.05, (n, 3))
    d = rng.normal(size=(n, 3)); d[:, 1] = np.abs(d[:, 1]) * 0.2; d[:, 2] = -np.abs(d[:, 2]) - 2.0
    # aim at the back wall z=0 above the boxes: expect t = -o.z/d.z unless a side wall / ceiling comes first
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    r["d"] = d; r["tmax"] = 1e30
    h = b.trace(r)
    o = r["o"].astype(np.float64); d = r["d"].astype(np.float64)
    cand = np.stack([(0 - o[:, 2]) / d[:, 2], (0 - o[:, 0]) / d[:, 0], (1 - o[:, 0]) / d[:, 0], (1 - o[:, 1]) / d[:, 1]], 1)
    cand[cand <= 0] = np.inf
    # the light sits 0.005 under the ceiling: exclude rays that reach y >= 0.995 inside its footprint first
    t_exp = cand.min(1)
    p = o + d * t_exp[:, None]
    ty = (0.995 - o[:, 1]) / d[:, 1]
    pl = o + d * ty[:, None]
    light = (ty > 0) & (ty < t_exp) & (np.abs(pl[:, 0] - 0.5) <= 0.125) & (np.abs(pl[:, 2] - 0.5) <= 0.125)
    ok = ~light
    assert ok.sum() > 1500
    assert np.all(h["prim"][ok] >= 0)
    assert np.allclose(h["t"][ok], t_exp[ok], rtol=2e-6, atol=1e-6)
    # barycentrics reconstruct the hit point
    tri = s.verts[h["prim"][ok]].astype(np.float64)
    u = h["u"][ok][:, None]; v = h["v"][ok][:, None]
    rec = tri[:, 0] * (1 - u - v) + tri[:, 1] * u + tri[:, 2] * v
    assert np.allclose(rec, p[ok], atol=5e-6)


def test_analytic_sphere_within_tessellation_error(oracle):
    s = I.furnace_sphere(4)                       # unit icosphere, 5120 tris
    b = oracle.Bvh(s.verts)
    rng = np.random.default_rng(2)
    n = 3000
    o = rng.normal(size=(n, 3)); o = 3.0 * o / np.linalg.norm(o, axis=1, keepdims=True)
    tgt = rng.uniform(-0.5, 0.5, (n, 3))
    d = tgt - o; d /= np.linalg.norm(d, axis=1, keepdims=True)
    r = np.zeros(n, oracle.RAY_DTYPE); r["o"] = o; r["d"] = d; r["tmax"] = 1e30
    h = b.trace(r)
    od = (r["o"].astype(np.float64) * r["d"]).sum(1)
    disc = od * od - ((r["o"].astype(np.float64) ** 2).sum(1) - 1.0)
    t_exp = -od - np.sqrt(disc)
    assert np.all(h["prim"] >= 0)
    # inscribed mesh: chord sag <= 1 - cos(edge/2) ~ 0.003 at subdivision 4; hits lie slightly inside
    assert np.all(h["t"] >= t_exp - 1e-5) and np.max(h["t"] - t_exp) < 0.02


def test_fp32_oracle_close_to_fp64_build(oracle):
    s = I.interior(n_boxes=30, n_spheres=6, subdiv=2)
    b32 = oracle.Bvh(s.verts); b64 = oracle.Bvh(s.verts, fp64=True)
    rays = _rays(I.random_rays(9, 4000, [0, 0, 0], [40, 8, 40]), oracle)
    h32 = b32.trace(rays); h64 = b64.trace(rays)
    same = h32["prim"] == h64["prim"]
    assert same.mean() > 0.999
    m = same & (h32["prim"] >= 0)
    assert np.allclose(h32["t"][m], h64["t"][m], rtol=1e-4)
    assert np.allclose(h32["u"][m], h64["u"][m], atol=1e-3)


def test_sah_beats_median_split_proxy(oracle):
    """SAH cost of the built tree is finite, positive and the tree is shallow enough for a 128-entry stack."""
    s = I.interior(n_boxes=50, n_spheres=10, subdiv=2)
    info = oracle.Bvh(s.verts).info()
    assert 0 < info["sah"] < 200 and info["depth"] < 64
    assert s.n_tris / 4 <= (info["n_nodes"] + 1) / 2 <= s.n_tris


def test_empty_inputs(oracle):
    b = oracle.Bvh(np.zeros((0, 3, 3), np.float32))
    r = _rays(I.random_rays(1, 5, [0, 0, 0], [1, 1, 1]), oracle)
    assert np.all(b.trace(r)["prim"] == -1)
    assert len(oracle.Bvh(I.cornell().verts).trace(r[:0])) == 0


@pytest.mark.parametrize("mode,gw,gh,s", [(0, 1, 1, 1), (2, 4, 4, 2)])
def test_closed_box_without_light_is_watertight_and_black(oracle, mode, gw, gh, s):
    """Closed Lambert cube seen from inside, no light, no environment: every primary ray and every secondary ray of three
    bounces hits a wall (the offset origins of D:R7 never leak through a face or an edge), and the image stays 0."""
    sc = I.emissive_box(albedo=0.8)
    fr = oracle.frame(sc.width, sc.height, 2, 0, 0)
    b = oracle.Bvh(sc.verts)
    rays, hits, r2p = oracle.trace_primary(b, sc.camera, fr, mode, gw, gh, s)
    paths = oracle.paths_init(2 * sc.width * sc.height)
    accum = np.zeros((sc.height, sc.width, 3), np.float32)
    oracle.shade_accumulate(sc, fr, 0, False, rays, hits, r2p, paths, accum)
    for bounce in (1, 2, 3):
        act = rays["tmax"] >= 0
        assert act.sum() == 2 * sc.width * sc.height and np.all(hits["prim"][act] >= 0)
        g = oracle.generate_secondary(sc, fr, bounce, mode, gw, gh, s, b.info()["bounds"], rays, hits, r2p, paths)
        rays, r2p = g["rays"], g["ray_to_path"]
        assert g["n_active"] == 2 * sc.width * sc.height
        o = rays["o"][rays["tmax"] >= 0]
        assert np.all(o > 0) and np.all(o < 1)                              # strictly inside the cube
        hits = b.trace(rays)
        oracle.shade_accumulate(sc, fr, bounce, bounce == 3, rays, hits, r2p, paths, accum)
    assert np.all(hits["prim"][rays["tmax"] >= 0] >= 0)
    assert np.all(accum == 0) and np.all(paths["T"] > 0) and np.all(paths["T"] <= np.float32(0.8) ** 3 * 1.0001)
