"""GPU parity tests: libcrt (through its C ABI, via the ctypes binding) against the CPU oracle, element by element
on the same seeded inputs.  Bars are north_star's: integer outputs bit-exact; hit ids identical >= 99.99 % with the rest
only at t-ties within 1e-5 relative; t/u/v within 1e-4 relative; images within 1e-3 RMSE.  Ray tolerance: reading A-26.
"""
import numpy as np
import pytest

import crt_inputs as I
from pipeline import GpuScene, compare_hits, compare_rays, hits_np, oracle_frame, paths_np, rays_np, rmse

pytestmark = pytest.mark.gpu

MODES = {"independent": 0, "morton_reorder": 1, "direct_reuse": 2, "world_reuse": 3,
         "sort_origin": 4, "sort_reis": 5, "sort_costa": 6, "sort_twopoint": 7}


@pytest.fixture(scope="module")
def crt():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2310_07182_b200 as crt
    return crt


@pytest.fixture(scope="module")
def ctx(crt):
    return crt.Context(0)


def _small_interior():
    return I.interior(seed=1, width=96, height=64, n_boxes=60, n_spheres=12, subdiv=2)


SCENES = {
    "landscape_small": lambda: I.landscape(seed=2, width=96, height=64, n=192, n_trees=150),
    "cornell": lambda: I.cornell(),
    "interior_small": _small_interior,
    "checker": lambda: I.checker_floor(seed=3, width=48, height=40),
}


# ------------------------------------------------------------------ full size, in the launch configuration bench.py times
def test_full_size_config2_stagewise_and_sampled(crt, ctx, oracle):
    """BASELINE config 2 at full size (1,024,704 triangles, 1920x1080, direct_reuse 4x4 stride 4): the partition covers every
    pixel exactly once; generation fed the GPU's own primary hits equals the oracle's generation on the same buffers
    (integer maps bit-exact, rays bit-identical), for both bounces; ALL hits of the primary segment and of both bounces equal the
    oracle's (ids >= 99.99 %, t-tie rule), and a sample of them the all-triangles definition."""
    scene = I.interior(seed=1).with_camera(1920, 1080)
    G = GpuScene(crt, scene, ctx)
    w, h, spp, gw, gh, s = 1920, 1080, 1, 4, 4, 4
    fr = crt.make_frame(w, h, spp, 1, 3); ofr = oracle.frame(w, h, spp, 1, 3)
    order = crt.make_order("direct_reuse", gw, gh, s)
    n_paths, n_slots, n_groups = crt.crt_layout(fr, order)
    assert (n_paths, n_slots, n_groups) == (2073600, 2088960, 130560)
    rays0, hits0, r2p0 = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    r2p = r2p0.cpu().numpy()
    assert np.array_equal(np.sort(r2p[r2p >= 0]), np.arange(n_paths))            # exact cover
    assert np.array_equal(r2p, oracle.partition(ofr, 2, gw, gh, s))
    import torch
    paths = ctx.empty((n_paths, 8)); ctx.crt_paths_init(paths)
    accum = torch.zeros((h, w, 3), device=ctx.device)
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 0, False, rays0, hits0, r2p0, paths, accum)
    paths_before = paths_np(oracle, paths).copy()
    out = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 1, order, rays0, hits0, r2p0, paths)
    bounds = np.asarray(G.bvh.info()["bounds"], np.float32)
    g = oracle.generate_secondary(scene, ofr, 1, 2, gw, gh, s, bounds, rays_np(oracle, rays0), hits_np(oracle, hits0), r2p, paths_before)
    for k in ("ray_to_path", "group_id", "dir_src", "group_class"):
        assert np.array_equal(out[k].cpu().numpy(), g[k]), k
    assert int(out["n_active"].cpu().numpy().view(np.uint32)[0]) == g["n_active"] > 1500000
    assert set(np.unique(g["group_class"])) == {0, 1, 2, 3}                      # empty, diffuse, glossy and hybrid groups all occur
    rg = rays_np(oracle, out["rays"])
    assert rg.tobytes() == g["rays"].tobytes()
    hits1 = ctx.crt_trace(G.bvh, out["rays"])
    # second bounce, stage-wise again: shade(1), generate(2) on the GPU's own buffers against the oracle's on the same buffers
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 1, False, out["rays"], hits1, out["ray_to_path"], paths, accum)
    paths_before2 = paths_np(oracle, paths).copy()
    out2 = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 2, order, out["rays"], hits1, out["ray_to_path"], paths)
    g2 = oracle.generate_secondary(scene, ofr, 2, 2, gw, gh, s, bounds, rg, hits_np(oracle, hits1), g["ray_to_path"], paths_before2)
    for k in ("ray_to_path", "group_id", "dir_src", "group_class"):
        assert np.array_equal(out2[k].cpu().numpy(), g2[k]), k
    assert rays_np(oracle, out2["rays"]).tobytes() == g2["rays"].tobytes()
    pg = paths_np(oracle, paths)                                              # (the oracle updated paths_before2 in place)
    assert np.array_equal(pg["flags"] & 1, paths_before2["flags"] & 1) and np.array_equal(pg["T"], paths_before2["T"])
    hits2 = ctx.crt_trace(G.bvh, out2["rays"])
    # EVERY hit of the primary segment and of both bounces (3 x 2.07 M rays) against the oracle's BVH, which is itself checked
    # against the all-triangles definition on a sample of the same rays
    ob = oracle.Bvh(scene.verts)
    assert ob.check() == 0
    rng = np.random.default_rng(11)
    n_rays_compared = 0
    for rays_dev, hits_dev, n_s in ((rays0, hits0, 120), (out["rays"], hits1, 360), (out2["rays"], hits2, 240)):
        r = rays_np(oracle, rays_dev); hh = hits_np(oracle, hits_dev)
        ho = ob.trace(r)
        frac = compare_hits(hh, ho)
        assert frac >= 0.9999
        act = np.flatnonzero(r["tmax"] >= 0)
        n_rays_compared += len(act)
        pick = rng.choice(act, n_s, replace=False)
        brute = oracle.trace_brute(scene.verts, r[pick])
        assert np.array_equal(ho[pick], brute)                               # the oracle's BVH == the plain definition, bit for bit
        compare_hits(hh[pick], brute)
        assert np.all(hh["prim"][r["tmax"] < 0] == -1)
    assert n_rays_compared > 5000000


# ------------------------------------------------------------------ a0 / a5: BVH + traversal
@pytest.mark.parametrize("scene_name", ["cornell", "interior_small", "landscape_small"])
@pytest.mark.parametrize("kernel", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9])
def test_trace_matches_oracle_on_random_rays(crt, ctx, oracle, scene_name, kernel):
    scene = SCENES[scene_name]()
    # kernel 2 reads the 8-wide compressed layout, which exists when every leaf holds one triangle
    G = GpuScene(crt, scene, ctx, **({"max_leaf": 1} if kernel == 2 else {}))
    assert G.bvh.check() == 0
    info = G.bvh.info()
    assert (info["n_wide_nodes"] > 0) == (kernel == 2)
    assert info["n_tris"] == scene.n_tris
    ob = oracle.Bvh(scene.verts)
    assert np.array_equal(info["bounds"], ob.info()["bounds"])
    n = 20000 + 37                                    # several blocks and a ragged tail
    r = I.random_rays(5, n, info["bounds"][:3], info["bounds"][3:], inactive_frac=0.05)
    ctx.crt_set_option("trace_kernel", kernel)
    try:
        h = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    finally:
        ctx.crt_set_option("trace_kernel", 3)
    ho = ob.trace(r.view(oracle.RAY_DTYPE).reshape(-1))
    compare_hits(h, ho)
    # the triangle test is the same fp32 operation sequence on both sides: where ids agree the record is bit-identical
    same = h["prim"] == ho["prim"]
    assert (h[same].tobytes() == ho[same].tobytes())


@pytest.mark.parametrize("scene_name", ["cornell", "interior_small", "landscape_small"])
@pytest.mark.parametrize("max_leaf,radius", [(3, 0), (1, 4), (4, 32)])
@pytest.mark.parametrize("builder", [1, 2])
def test_device_bvh_builder(crt, ctx, oracle, scene_name, max_leaf, radius, builder):
    """crt_bvh_params.builder = 1: the hierarchy built on the GPU (parallel locally-ordered clustering, csrc/bvh_ploc.cu).  The tree passes
    the library's own invariant check (every triangle in exactly one leaf, leaves <= max_leaf, boxes nested, 16-bit planes outside their
    boxes) and traversal returns the SAME hit records as with the host-built tree and as the oracle (the result is structure-independent, D:R10)."""
    scene = SCENES[scene_name]()
    bvh_d = ctx.crt_build_bvh(scene.verts, scene.mat_id, max_leaf=max_leaf, builder=builder, ploc_radius=radius)
    bvh_h = ctx.crt_build_bvh(scene.verts, scene.mat_id, max_leaf=max_leaf)
    assert bvh_d.check() == 0
    info_d, info_h = bvh_d.info(), bvh_h.info()
    assert info_d["builder"] == builder and info_h["builder"] == 0 and info_d["build_rounds"] > 3 and info_d["device_build_seconds"] > 0
    assert info_d["n_tris"] == scene.n_tris and info_d["max_leaf"] == max_leaf and 0 < info_d["depth"] <= 60
    assert np.array_equal(info_d["bounds"], info_h["bounds"]) and 100 <= info_d["q16_inflation_pct"] <= 130
    assert scene.n_tris / max_leaf <= (info_d["n_nodes"] + 1) / 2 <= scene.n_tris
    assert info_d["sah_cost"] < 1.6 * info_h["sah_cost"]                     # a comparable tree, not a degenerate one
    r = I.random_rays(6, 30000 + 11, info_h["bounds"][:3], info_h["bounds"][3:], inactive_frac=0.05)
    rd = ctx.upload(r)
    hd = hits_np(oracle, ctx.crt_trace(bvh_d, rd)); hh = hits_np(oracle, ctx.crt_trace(bvh_h, rd))
    assert hd.tobytes() == hh.tobytes()
    compare_hits(hd, oracle.Bvh(scene.verts).trace(r.view(oracle.RAY_DTYPE).reshape(-1)))


def test_device_bvh_builder_degenerate_inputs(crt, ctx, oracle):
    """one triangle, two triangles, many identical triangles (all centroids and boxes coincide), an empty scene; then the frame loop"""
    base = I.cornell().verts
    for v in (base[:1], base[:2], base[:5], np.repeat(base[:1], 37, axis=0), base[:0]):
        v = np.ascontiguousarray(v, np.float32)
        for builder in (1, 2):
            bvh = ctx.crt_build_bvh(v, np.zeros(len(v), np.int32), builder=builder)
            assert bvh.check() == 0
            r = I.random_rays(2, 500, [0, 0, 0], [1, 1, 1])
            h = hits_np(oracle, ctx.crt_trace(bvh, ctx.upload(r)))
            compare_hits(h, oracle.trace_brute(v, r.view(oracle.RAY_DTYPE).reshape(-1)))
    # the frame loop on a device-built tree: generation reads its triangle records and slot map
    import torch
    scene = _small_interior()
    imgs = []
    for builder in (0, 1):
        bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, builder=builder)
        mats_dev = ctx.upload(scene.materials); mats = ctx.scene_mats(mats_dev, len(scene.materials), scene.env)
        fr = crt.make_frame(96, 64, 1, 3, 2); order = crt.make_order("direct_reuse", 4, 4, 2)
        acc = torch.zeros((64, 96, 3), device=ctx.device)
        ctx.crt_render_frame(bvh, mats, crt.make_camera(scene.camera), fr, order, 2, acc, ctx.frame_workspace(fr, order))
        torch.cuda.synchronize(); imgs.append(acc.cpu().numpy())
    assert imgs[0].sum() > 0 and np.array_equal(imgs[0], imgs[1])


def test_trace_tolerance_only_triangle_test(crt, ctx, oracle):
    """Option trace_exact = 0 (fused multiply-adds + approximate reciprocal in the triangle test; measured 3-5 % faster, profiles/r02a):
    NOT the default, because it only meets part of north_star's bar: ids agree on >= 99.99 % of rays, but t of grazing hits can
    deviate by a few 1e-4 relative.  Checked here: ids >= 99.99 %, hit/miss decisions equal except at those, t within 1e-3."""
    scene = _small_interior()
    G = GpuScene(crt, scene, ctx)
    info = G.bvh.info()
    r = I.random_rays(5, 200000 + 13, info["bounds"][:3], info["bounds"][3:], inactive_frac=0.05)
    ho = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    ctx.crt_set_option("trace_exact", 0)
    try:
        h = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    finally:
        ctx.crt_set_option("trace_exact", 1)
    same = h["prim"] == ho["prim"]
    assert same.mean() >= 0.9999
    m = same & (ho["prim"] >= 0)
    assert np.all(np.abs(h["t"][m].astype(np.float64) - ho["t"][m]) <= 1e-3 * np.abs(ho["t"][m]))
    assert np.median(np.abs(h["t"][m].astype(np.float64) - ho["t"][m]) / np.abs(ho["t"][m])) < 1e-6


@pytest.mark.parametrize("scene_name", ["cornell", "interior_small", "landscape_small"])
@pytest.mark.parametrize("n", [20037, 900, 33])
def test_trace_tail_split_and_timeline(crt, ctx, oracle, scene_name, n):
    """Option trace_tail_split = 1 (idle lanes take over stack entries of their warp's busy lanes once the ray list is exhausted; measured no
    faster, profiles/r02i): the hit records are those of the default kernel and of the oracle, bit for bit.  Small n: the whole launch is tail.
    crt_trace_timeline: same records, and marks that are ordered in time."""
    import torch
    scene = SCENES[scene_name]()
    G = GpuScene(crt, scene, ctx)
    info = G.bvh.info()
    r = I.random_rays(11, n, info["bounds"][:3], info["bounds"][3:], inactive_frac=0.05)
    rd = ctx.upload(r)
    ho = oracle.Bvh(scene.verts).trace(r.view(oracle.RAY_DTYPE).reshape(-1))
    h0 = ctx.crt_trace(G.bvh, rd).clone()
    for split in (1, 0):
        ctx.crt_set_option("trace_tail_split", split)
        try:
            h1 = ctx.crt_trace(G.bvh, rd).clone()
            h2, marks = ctx.crt_trace_timeline(G.bvh, rd)
        finally:
            ctx.crt_set_option("trace_tail_split", 0)
        assert torch.equal(h0.view(torch.int32), h1.view(torch.int32))
        assert torch.equal(h0.view(torch.int32), h2.view(torch.int32))
        assert marks.shape[0] == min(148 * 8 * 4, (n + 127) // 128 * 4) and marks.shape[1] == 4
        assert np.all(marks[:, 0] > 0) and np.all(marks[:, 2] >= marks[:, 0])
        seen = marks[:, 1] > 0
        assert np.all(marks[seen, 1] >= marks[seen, 0]) and np.all(marks[seen, 1] <= marks[seen, 2])
    compare_hits(hits_np(oracle, h0), ho)


@pytest.mark.parametrize("scene_name", ["cornell", "interior_small", "landscape_small"])
def test_presplit_and_optimised_trees_return_the_same_hits(crt, ctx, oracle, scene_name):
    """Pre-splitting large triangles (crt_bvh_params.presplit, the default 1/16 and a much finer 1/128) and the insertion-based optimisation of the tree
    (crt_bvh_params.optimize: parallel re-insertion on the device for builder 0, the host's own for builder 3) change the tree, not the triangles: the hit
    records equal those of the unsplit tree and of the oracle bit for bit (D:R10: the result does not depend on the structure), also when a triangle
    sits in many leaves and is tested more than once; the device layouts pass their check."""
    import torch
    scene = SCENES[scene_name]()
    ref = None; r = None
    # builder 0: the optimisation step is the device's parallel re-insertion; builder 3: the host's own
    for ps, opt, builder in ((0.0, 0, 0), (1 / 16, 0, 0), (1 / 128, 0, 0), (0.0, 30, 0), (1 / 16, 100, 0), (1 / 16, 30, 3), (1 / 128, 7, 0)):
        bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, presplit=ps, optimize=opt, builder=builder)
        assert bvh.check() == 0
        info = bvh.info()
        if r is None:
            r = I.random_rays(13, 30000 + 5, info["bounds"][:3], info["bounds"][3:], inactive_frac=0.05)
        assert info["n_tris"] == scene.n_tris and (info["n_refs"] == info["n_tris"] if ps == 0 else info["n_refs"] >= info["n_tris"])
        assert ps < 1 / 16 or scene_name == "landscape_small" or info["n_refs"] > info["n_tris"]      # (the small terrain has no triangle that long)
        h = ctx.crt_trace(bvh, ctx.upload(r)).clone()
        if ref is None:
            ref = h
            compare_hits(hits_np(oracle, h), oracle.Bvh(scene.verts).trace(r.view(oracle.RAY_DTYPE).reshape(-1)))
        assert torch.equal(ref.view(torch.int32), h.view(torch.int32)), (ps, opt, builder)
        assert info["builder"] == builder and info["depth"] <= 60 and (info["optimize_iterations"] > 0 if (opt >= 30 and scene_name != "landscape_small") else info["optimize_iterations"] <= opt)
        bvh.destroy()


def test_trace_tiny_scene_against_brute_force(crt, ctx, oracle):
    scene = I.furnace_sphere(1)                       # 80 triangles
    G = GpuScene(crt, scene, ctx)
    r = I.random_rays(8, 3001, [-1, -1, -1], [1, 1, 1])
    h = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    hb = oracle.trace_brute(scene.verts, r.view(oracle.RAY_DTYPE).reshape(-1))
    compare_hits(h, hb)


def test_trace_edge_cases(crt, ctx, oracle):
    import torch
    scene = I.cornell()
    G = GpuScene(crt, scene, ctx)
    # empty batch
    assert ctx.crt_trace(G.bvh, ctx.empty((0, 8))).shape[0] == 0
    # all inactive
    r = I.random_rays(1, 100, [0, 0, 0], [1, 1, 1], inactive_frac=1.0)
    h = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    assert np.all(h["prim"] == -1) and np.all(h["t"] == -1.0)
    # a single triangle and an empty scene
    one = GpuScene(crt, I.Scene("one", scene.verts[:1], scene.mat_id[:1], scene.materials, scene.env, scene.camera), ctx)
    rr = I.random_rays(2, 500, [0, 0, 0], [1, 1, 1])
    compare_hits(hits_np(oracle, ctx.crt_trace(one.bvh, ctx.upload(rr))), oracle.trace_brute(scene.verts[:1], rr.view(oracle.RAY_DTYPE).reshape(-1)))
    empty = ctx.crt_build_bvh(np.zeros((0, 3, 3), np.float32), np.zeros(0, np.int32))
    he = hits_np(oracle, ctx.crt_trace(empty, ctx.upload(rr)))
    assert np.all(he["prim"] == -1)
    # tmin / tmax windows
    rw = rr.copy(); rw[:, 3] = 0.3; rw[:, 7] = 0.9
    compare_hits(hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(rw))), oracle.Bvh(scene.verts).trace(rw.view(oracle.RAY_DTYPE).reshape(-1)))
    # misaligned pointer is rejected
    buf = ctx.empty((101 * 8 + 1,))
    with pytest.raises(crt.CrtError) as e:
        ctx.crt_trace(G.bvh, buf[1:].view(-1)[: 100 * 8].view(100, 8))
    assert e.value.status == crt.api.CRT_ERR_INVALID_ARG
    torch.cuda.synchronize()


@pytest.mark.parametrize("kernel", [0, 1, 3, 4])
def test_trace_degenerate_directions_and_far_origins(crt, ctx, oracle, kernel):
    """The box test must stay conservative where its arithmetic degenerates: direction components that are exactly zero
    (1/d infinite, plane distances NaN), origins exactly on box planes of the axis-aligned Cornell walls, and origins far
    outside the scene (the 16-bit layout states 16 scene extents, include/crt.h).  Hits must equal the
    all-triangles definition."""
    scene = I.cornell()
    G = GpuScene(crt, scene, ctx)
    rng = np.random.default_rng(21)
    n = 6000
    r = np.zeros((n, 8), np.float32); r[:, 7] = 1e30
    o = rng.random((n, 3)).astype(np.float32)
    o[: n // 3] = np.round(o[: n // 3] * 4) / 4                       # grid points: on wall and tessellation planes
    d = rng.normal(size=(n, 3))
    d[0:2000:2, rng.integers(0, 3)] = 0.0                             # one zero component
    k = rng.integers(0, 3, n)
    ax = np.zeros((n, 3)); ax[np.arange(n), k] = rng.choice([-1.0, 1.0], n)
    d[1:2000:2] = ax[1:2000:2]                                        # axis-aligned: two zero components
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    far = slice(4000, n)                                              # origins 4-15 extents away, aimed at the box
    tgt = rng.random((n, 3))
    dirs = rng.normal(size=(n, 3)); dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    # kernel 4 (directed rounding + per-ray margin) is conservative for any origin: 30 to 3000 extents; the others inside their contract
    dist = np.exp(rng.uniform(np.log(30.0), np.log(3000.0), (n, 1))) if kernel == 4 else rng.uniform(4, 15, (n, 1))
    o64 = o.astype(np.float64); o64[far] = tgt[far] - dirs[far] * dist[far]; d[far] = dirs[far]
    r[:, 0:3] = o64; r[:, 4:7] = d
    ctx.crt_set_option("trace_kernel", kernel)
    try:
        h = hits_np(oracle, ctx.crt_trace(G.bvh, ctx.upload(r)))
    finally:
        ctx.crt_set_option("trace_kernel", 3)
    hb = oracle.trace_brute(scene.verts, r.view(oracle.RAY_DTYPE).reshape(-1))
    compare_hits(h, hb)
    assert (hb["prim"] >= 0).mean() > 0.5


def test_coarse_grid_falls_back_to_fp32_nodes(crt, ctx, oracle):
    """A scene whose detail is far below the 16-bit grid step (two small clusters of triangles 10^6 triangle sizes apart): the
    decoded boxes are reported as inflated (`q16_inflation_pct` > 200), the default kernel reads the fp32 nodes, and the hits
    equal the all-triangles definition either way (forcing the 16-bit nodes is slower, not wrong)."""
    rng = np.random.default_rng(5)
    def cluster(c):
        p = c + rng.random((200, 1, 3)) * 1e-2
        return (p + rng.random((200, 3, 3)) * 1e-3).astype(np.float32)
    verts = np.concatenate([cluster(np.zeros(3)), cluster(np.array([1000.0, 500.0, 250.0]))])
    bvh = ctx.crt_build_bvh(verts, np.zeros(len(verts), np.int32))
    info = bvh.info()
    assert bvh.check() == 0 and info["q16_inflation_pct"] > 200
    small = GpuScene(crt, I.cornell(), ctx).bvh.info()["q16_inflation_pct"]
    assert 100 <= small < 130
    n = 4000
    r = np.zeros((n, 8), np.float32); r[:, 7] = 1e30
    tgt = verts[rng.integers(0, len(verts), n)].mean(1) + rng.normal(size=(n, 3)) * 2e-4
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    r[:, 0:3] = tgt - d * rng.uniform(0.01, 5.0, (n, 1)); r[:, 4:7] = d
    hb = oracle.trace_brute(verts, r.view(oracle.RAY_DTYPE).reshape(-1))
    compare_hits(hits_np(oracle, ctx.crt_trace(bvh, ctx.upload(r))), hb)
    assert (hb["prim"] >= 0).mean() > 0.2


def test_trace_stats_counts(crt, ctx, oracle):
    scene = _small_interior()
    G = GpuScene(crt, scene, ctx)
    r = I.random_rays(5, 5000, [0, 0, 0], [40, 8, 40], inactive_frac=0.1)
    nn, nt, act = ctx.crt_trace_stats(G.bvh, ctx.upload(r))
    assert act == int((r[:, 7] >= 0).sum())
    assert nn > act and nt > 0
    # same order of magnitude as the oracle's own tree (different builder parameters, so not equal)
    cnt = np.zeros(2, np.int64)
    oracle.Bvh(scene.verts).trace(r.view(oracle.RAY_DTYPE).reshape(-1), cnt)
    assert 0.3 < nn / cnt[0] < 3.0 and 0.3 < nt / cnt[1] < 3.0


# ------------------------------------------------------------------ a1: primary rays
@pytest.mark.parametrize("mode,gw,gh,s", [("independent", 1, 1, 1), ("direct_reuse", 4, 4, 2), ("direct_reuse", 2, 4, 4), ("direct_reuse", 4, 4, 2 | (1 << 14)),
                                          ("direct_reuse", 8, 2, 2 | (4 << 16) | (1 << 14)),
                                          ("direct_reuse", 4, 4, 2 | (1 << 15)), ("direct_reuse", 8, 8, 8 | (1 << 15)), ("direct_reuse", 2, 1, 1 | (1 << 15)),   # LCG-sequence rule (D:R21)
                                          ("direct_reuse", 8, 1, 1 | (8 << 16) | (1 << 15))])
@pytest.mark.parametrize("w,h,spp", [(64, 64, 1), (50, 37, 2)])
def test_primary_matches_oracle(crt, ctx, oracle, mode, gw, gh, s, w, h, spp):
    scene = I.cornell(width=w, height=h)
    G = GpuScene(crt, scene, ctx)
    fr = crt.make_frame(w, h, spp, seed=0, frame=3)
    order = crt.make_order(mode, gw, gh, s)
    rays, hits, r2p = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    ofr = oracle.frame(w, h, spp, 0, 3)
    ro, ho, po = oracle.trace_primary(oracle.Bvh(scene.verts), scene.camera, ofr, MODES[mode], gw, gh, s)
    assert crt.crt_layout(fr, order)[1] == len(po)
    assert np.array_equal(r2p.cpu().numpy(), po)                       # partition: bit-exact
    rg = rays_np(oracle, rays)
    compare_rays(rg, ro)
    act = ro["tmax"] >= 0
    assert rg[act].tobytes() == ro[act].tobytes()                        # same fp32 operation sequence
    hg = hits_np(oracle, hits)
    compare_hits(hg[act], ho[act])


# ------------------------------------------------------------------ a2-a4: generation, stage-wise (oracle buffers in)
GEN_CASES = [
    ("cornell", "independent", 1, 1, 1, 64, 64, 1),
    ("cornell", "morton_reorder", 1, 1, 1, 64, 64, 1),
    ("cornell", "direct_reuse", 4, 4, 2, 64, 64, 1),          # BASELINE config 1
    ("interior_small", "independent", 1, 1, 1, 96, 64, 1),
    ("interior_small", "morton_reorder", 1, 1, 1, 96, 64, 2),
    ("interior_small", "sort_origin", 1, 1, 1, 96, 64, 1),     # the paper's other reordering keys (D:R19)
    ("interior_small", "sort_reis", 1, 1, 1, 96, 64, 2),
    ("interior_small", "sort_costa", 1, 1, 1, 96, 64, 1),
    ("interior_small", "sort_twopoint", 1, 1, 1, 96, 64, 2),
    ("landscape_small", "sort_twopoint", 1, 1, 1, 96, 64, 1),
    ("interior_small", "direct_reuse", 4, 4, 4, 96, 64, 1),   # config 2's grouping, partial tiles (96x64 vs 16x16: exact) ...
    ("interior_small", "direct_reuse", 2, 2, 8, 90, 61, 2),   # ... and ragged ones with 2 spp
    ("interior_small", "direct_reuse", 8, 8, 1, 96, 64, 1),   # stride 1: one group per tile, K = 64 (two warps per group)
    ("interior_small", "direct_reuse", 8, 8, 8, 96, 64, 1),   # largest tile: M = 4096
    ("checker", "direct_reuse", 4, 4, 2, 48, 40, 1),          # hybrid groups
    ("checker", "direct_reuse", 1, 1, 4, 48, 40, 1),          # K = 1
    ("interior_small", "direct_reuse", 4, 4, 4 | (1 << 14), 96, 64, 1),      # regular-lattice partition rule (D:R20)
    ("checker", "direct_reuse", 4, 2, 2 | (4 << 16) | (1 << 14), 50, 37, 2),  # lattice, unequal strides, ragged, 2 spp, hybrid groups
    ("interior_small", "direct_reuse", 4, 4, 4 | (1 << 15), 96, 64, 1),      # LCG-sequence partition rule (D:R21)
    ("checker", "direct_reuse", 4, 2, 2 | (4 << 16) | (1 << 15), 50, 37, 2),  # sequence rule, unequal strides, ragged, 2 spp, hybrid groups
    ("interior_small", "direct_reuse", 8, 1, 1 | (8 << 16), 96, 64, 1),     # the paper's own setting: tile 8x8, K = 8
    ("interior_small", "direct_reuse", 16, 1, 2 | (8 << 16), 90, 61, 2),    # tile 32x8, K = 16 (Table 3), ragged, 2 spp
    ("landscape_small", "direct_reuse", 4, 4, 4, 96, 64, 1),  # config 4's grouping on a reduced landscape (coordinates up to 192, sky misses)
    ("landscape_small", "morton_reorder", 1, 1, 1, 90, 61, 1),
    ("cornell", "world_reuse", 4, 4, 2, 64, 64, 1),           # world-space reuse (D:R18)
    ("interior_small", "world_reuse", 4, 4, 4, 96, 64, 1),
    ("interior_small", "world_reuse", 8, 8, 1, 90, 61, 2),    # K = 64, ragged image, 2 spp
    ("checker", "world_reuse", 4, 4, 2, 48, 40, 1),           # glossy and mirror members evaluate / ignore the shared direction
]


@pytest.mark.parametrize("scene_name,mode,gw,gh,s,w,h,spp", GEN_CASES)
def test_generate_stagewise_matches_oracle(crt, ctx, oracle, scene_name, mode, gw, gh, s, w, h, spp):
    scene = SCENES[scene_name]().with_camera(w, h)
    G = GpuScene(crt, scene, ctx)
    n_b = 2
    ofr = oracle.frame(w, h, spp, 7, 2)
    st = oracle_frame(oracle, scene, ofr, n_b, MODES[mode], gw, gh, s)
    fr = crt.make_frame(w, h, spp, 7, 2)
    order = crt.make_order(mode, gw, gh, s)
    saw_hybrid = False
    for b in range(1, n_b + 1):
        paths = G.paths_to_dev(st["paths_before_gen"][b - 1])
        out = ctx.crt_generate_secondary(G.bvh, G.mats, fr, b, order, G.rays_to_dev(st["rays"][b - 1]), G.hits_to_dev(st["hits"][b - 1]),
                                         ctx.upload(st["r2p"][b - 1]), paths)
        g = st["gen"][b]
        # integer outputs: bit-exact
        assert np.array_equal(out["ray_to_path"].cpu().numpy(), g["ray_to_path"])
        assert np.array_equal(out["dir_src"].cpu().numpy(), g["dir_src"])
        assert np.array_equal(out["group_id"].cpu().numpy(), g["group_id"])
        assert int(out["n_active"].cpu().numpy().view(np.uint32)[0]) == g["n_active"]
        if mode == "direct_reuse":
            assert np.array_equal(out["group_class"].cpu().numpy(), g["group_class"])
            saw_hybrid |= bool((g["group_class"] == 3).any())
        else:
            # per-path class, written by path id (the oracle writes it per group = per path as well)
            assert np.array_equal(out["group_class"].cpu().numpy(), g["group_class"])
        rg = rays_np(oracle, out["rays"])
        compare_rays(rg, g["rays"])
        assert rg.tobytes() == g["rays"].tobytes()                        # same fp32 operation sequence: bit-identical rays
        pg = paths_np(oracle, paths); po = st["paths_after_gen"][b - 1]
        assert np.array_equal(pg["flags"] & 1, po["flags"] & 1)
        assert np.allclose(pg["T"], po["T"], rtol=1e-6, atol=0)
    if scene_name == "checker" and gw * gh > 1 and mode == "direct_reuse":
        assert saw_hybrid


def test_ray_code_encode_bit_exact(crt, ctx, oracle):
    """Origin / Reis / Costa / TwoPoint keys (D:R19) against the oracle, bit for bit; rays reach outside the scene box so the
    clamps of origin and end point are exercised; code out of range is rejected."""
    scene = _small_interior()
    G = GpuScene(crt, scene, ctx)
    b = G.bvh.info()["bounds"]
    r = I.random_rays(17, 50021, b[:3], b[3:], inactive_frac=0.1)
    for name, code in crt.api.RAY_CODES.items():
        keys = ctx.crt_ray_code_encode(G.bvh, code, ctx.upload(r)).cpu().numpy().view(np.uint32)
        ko = oracle.ray_code_encode(oracle.RAY_CODES[name], r.view(oracle.RAY_DTYPE).reshape(-1), b)
        assert np.array_equal(keys, ko), name
    assert np.array_equal(ctx.crt_ray_code_encode(G.bvh, 0, ctx.upload(r)).cpu().numpy(), ctx.crt_morton_encode(G.bvh, ctx.upload(r)).cpu().numpy())
    with pytest.raises(crt.CrtError) as e:
        ctx.crt_ray_code_encode(G.bvh, 5, ctx.upload(r))
    assert e.value.status == crt.api.CRT_ERR_INVALID_ARG


def test_morton_encode_and_radix_sort_bit_exact(crt, ctx, oracle):
    import torch
    scene = _small_interior()
    G = GpuScene(crt, scene, ctx)
    b = G.bvh.info()["bounds"]
    for n in (0, 1, 255, 4096, 4097, 100003):
        r = I.random_rays(n + 1, n, b[:3], b[3:], inactive_frac=0.1)
        keys = ctx.crt_morton_encode(G.bvh, ctx.upload(r))
        ko = oracle.morton_encode(r.view(oracle.RAY_DTYPE).reshape(-1), b)
        assert np.array_equal(keys.cpu().numpy().view(np.uint32), ko)
        vals = torch.arange(n, dtype=torch.int32, device=ctx.device)
        if n == 0:
            continue
        ks, vs = ctx.crt_radix_sort_pairs(keys, vals)
        order = oracle.sort_keys(ko)
        assert np.array_equal(vs.cpu().numpy(), order)
        assert np.array_equal(ks.cpu().numpy().view(np.uint32), ko[order])
    # full-range 32-bit keys with many duplicates (all four passes matter, stability matters)
    rng = np.random.default_rng(0)
    k = rng.integers(0, 2 ** 32, 50000, dtype=np.uint64).astype(np.uint32); k[::3] = k[0]
    ks, vs = ctx.crt_radix_sort_pairs(ctx.upload(k.view(np.int32)), torch.arange(len(k), dtype=torch.int32, device=ctx.device))
    assert np.array_equal(vs.cpu().numpy(), np.argsort(k, kind="stable").astype(np.int32))


# ------------------------------------------------------------------ a6: shading, stage-wise
@pytest.mark.parametrize("scene_name,spp", [("cornell", 1), ("interior_small", 2)])
def test_shade_accumulate_stagewise(crt, ctx, oracle, scene_name, spp):
    import torch
    scene = SCENES[scene_name]()
    w, h = scene.width, scene.height
    G = GpuScene(crt, scene, ctx)
    ofr = oracle.frame(w, h, spp, 1, 0); fr = crt.make_frame(w, h, spp, 1, 0)
    st = oracle_frame(oracle, scene, ofr, 2, 2, 4, 4, 2)
    accum = torch.zeros((h, w, 3), device=ctx.device)
    paths = ctx.empty((spp * w * h, 8)); ctx.crt_paths_init(paths)
    assert paths_np(oracle, paths).tobytes() == oracle.paths_init(spp * w * h).tobytes()
    for b in range(0, 3):
        if b > 0:
            paths = G.paths_to_dev(st["paths_after_gen"][b - 1])
        ctx.crt_shade_accumulate(G.bvh, G.mats, fr, b, b == 2, G.rays_to_dev(st["rays"][b]), G.hits_to_dev(st["hits"][b]), ctx.upload(st["r2p"][b]),
                                 paths, accum)
        pg = paths_np(oracle, paths); po = st["paths_after_shade"][b]
        assert np.array_equal(pg["flags"] & 1, po["flags"] & 1)
        assert np.allclose(pg["L"], po["L"], rtol=1e-6, atol=1e-7)
    assert rmse(accum.cpu().numpy(), st["accum"]) <= 1e-5


# ------------------------------------------------------------------ end to end
@pytest.mark.parametrize("mode,gw,gh,s", [("independent", 1, 1, 1), ("morton_reorder", 1, 1, 1), ("direct_reuse", 4, 4, 2)])
def test_config1_end_to_end(crt, ctx, oracle, mode, gw, gh, s):
    """BASELINE config 1: Cornell 64x64, 1 spp, 1 secondary bounce, groups 4x4 stride 2, seed 0, all three modes."""
    import torch
    scene = I.cornell(seed=0)
    G = GpuScene(crt, scene, ctx)
    fr = crt.make_frame(64, 64, 1, 0, 0); order = crt.make_order(mode, gw, gh, s)
    st = oracle_frame(oracle, scene, oracle.frame(64, 64, 1, 0, 0), 1, MODES[mode], gw, gh, s)
    accum = torch.zeros((64, 64, 3), device=ctx.device)
    ws = ctx.frame_workspace(fr, order)
    nsec = torch.zeros((1,), dtype=torch.int32, device=ctx.device)
    ctx.crt_render_frame(G.bvh, G.mats, G.camera, fr, order, 1, accum, ws, n_secondary=nsec)
    assert int(nsec.cpu()[0]) == st["gen"][1]["n_active"]
    assert rmse(accum.cpu().numpy(), st["accum"]) <= 1e-3
    # the same frame call by call (free-running: GPU buffers feed GPU stages)
    rays, hits, r2p = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    paths = ctx.empty((64 * 64, 8)); ctx.crt_paths_init(paths)
    acc2 = torch.zeros_like(accum)
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 0, False, rays, hits, r2p, paths, acc2)
    out = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 1, order, rays, hits, r2p, paths)
    g = st["gen"][1]
    assert np.array_equal(out["ray_to_path"].cpu().numpy(), g["ray_to_path"])
    assert np.array_equal(out["dir_src"].cpu().numpy(), g["dir_src"])
    assert np.array_equal(out["group_id"].cpu().numpy(), g["group_id"])
    assert np.array_equal(out["group_class"].cpu().numpy(), g["group_class"])
    h2 = ctx.crt_trace(G.bvh, out["rays"])
    compare_hits(hits_np(oracle, h2), st["hits"][1])
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 1, True, out["rays"], h2, out["ray_to_path"], paths, acc2)
    assert torch.equal(acc2, accum)
    # host-buffer entry point gives the same image
    acc_h = np.zeros((64, 64, 3), np.float32); nsec_h = np.zeros(1, np.uint32)
    ws_h = ctx.frame_workspace(fr, order, host_materials=len(scene.materials))
    ctx.crt_render_frame_host(G.bvh, scene.materials, scene.env, G.camera, fr, order, 1, acc_h, nsec_h, ws_h)
    assert np.array_equal(acc_h, accum.cpu().numpy()) and nsec_h[0] == g["n_active"]
    # device-resident accumulation: two frames through either host entry point give the same sum; reset starts over
    fr2 = crt.make_frame(fr.w, fr.h, fr.spp, fr.seed, fr.frame + 1)
    ctx.crt_render_frame_host(G.bvh, scene.materials, scene.env, G.camera, fr2, order, 1, acc_h, nsec_h, ws_h)
    img_r = np.full((64, 64, 3), -1.0, np.float32); ws_r = ctx.frame_workspace(fr, order, host_materials=len(scene.materials))
    ctx.crt_render_frame_host_resident(G.bvh, scene.materials, scene.env, G.camera, fr, order, 1, True, img_r, nsec_h, ws_r)
    assert np.array_equal(img_r, accum.cpu().numpy())
    # the non-synchronising form: outputs valid after the stream has been synchronised
    img_a = torch.full((64, 64, 3), -1.0).pin_memory(); nsec_a = torch.zeros(1, dtype=torch.int32).pin_memory(); st = torch.cuda.Stream()
    ctx.crt_render_frame_host_resident(G.bvh, scene.materials, scene.env, G.camera, fr, order, 1, True, img_a, nsec_a, ws_r, stream=st, wait=False)
    st.synchronize()
    assert np.array_equal(img_a.numpy(), accum.cpu().numpy()) and int(nsec_a[0]) == g["n_active"]
    ctx.crt_render_frame_host_resident(G.bvh, scene.materials, scene.env, G.camera, fr2, order, 1, False, img_r, nsec_h, ws_r)
    assert np.array_equal(img_r, acc_h)
    ctx.crt_render_frame_host_resident(G.bvh, scene.materials, scene.env, G.camera, fr, order, 1, True, img_r, nsec_h, ws_r)
    assert np.array_equal(img_r, accum.cpu().numpy())


@pytest.mark.parametrize("mode,gw,gh,s", [("independent", 1, 1, 1), ("morton_reorder", 1, 1, 1), ("direct_reuse", 4, 4, 4), ("direct_reuse", 8, 8, 2), ("world_reuse", 4, 4, 4),
                                          ("sort_reis", 1, 1, 1), ("sort_twopoint", 1, 1, 1)])
def test_mixed_materials_two_bounces_end_to_end(crt, ctx, oracle, mode, gw, gh, s):
    import torch
    scene = _small_interior()
    w, h, spp = 96, 64, 2
    G = GpuScene(crt, scene, ctx)
    acc_o = np.zeros((h, w, 3), np.float32)
    accum = torch.zeros((h, w, 3), device=ctx.device)
    ob = oracle.Bvh(scene.verts)
    for f in range(2):                                # accumulation over frames
        fr = crt.make_frame(w, h, spp, 1, f); order = crt.make_order(mode, gw, gh, s)
        oracle.render_frame(ob, scene, oracle.frame(w, h, spp, 1, f), 2, MODES[mode], gw, gh, s, accum=acc_o)
        ctx.crt_render_frame(G.bvh, G.mats, G.camera, fr, order, 2, accum, ctx.frame_workspace(fr, order))
    assert rmse(accum.cpu().numpy() / 2, acc_o / 2) <= 1e-3


@pytest.mark.parametrize("mode,gw,gh,s", [("direct_reuse", 4, 4, 2), ("direct_reuse", 4, 2, 2 | (4 << 16) | (1 << 14)), ("direct_reuse", 4, 4, 2 | (1 << 15)), ("world_reuse", 8, 8, 1), ("independent", 1, 1, 1)])
def test_render_frame_on_a_ragged_image_matches_the_oracle(crt, ctx, oracle, mode, gw, gh, s):
    """crt_render_frame as bench.py runs it (shading fused into generation, path state by slot under grouped orders) on an image that is
    not a multiple of the tile (50x37, 2 spp, 3 bounces, partial tiles on two sides): the accumulated image equals the oracle's."""
    import torch
    scene = _small_interior().with_camera(50, 37)
    w, h, spp, nb = 50, 37, 2, 3
    G = GpuScene(crt, scene, ctx)
    ob = oracle.Bvh(scene.verts)
    acc_o = np.zeros((h, w, 3), np.float32); accum = torch.zeros((h, w, 3), device=ctx.device)
    order = crt.make_order(mode, gw, gh, s)
    ws = ctx.frame_workspace(crt.make_frame(w, h, spp), order)
    for f in range(2):
        oracle.render_frame(ob, scene, oracle.frame(w, h, spp, 4, f), nb, MODES[mode], gw, gh, s, accum=acc_o)
        ctx.crt_render_frame(G.bvh, G.mats, G.camera, crt.make_frame(w, h, spp, 4, f), order, nb, accum, ws)
    assert rmse(accum.cpu().numpy() / 2, acc_o / 2) <= 1e-3
    assert acc_o.sum() > 0


@pytest.mark.parametrize("mode,gw,gh,s", [("independent", 1, 1, 1), ("morton_reorder", 1, 1, 1), ("direct_reuse", 4, 4, 2)])
def test_white_furnace_is_one(crt, ctx, mode, gw, gh, s):
    """Closed form: a convex white Lambert sphere under uniform radiance 1 renders to exactly 1 (north_star)."""
    import torch
    scene = I.furnace_sphere(2)
    G = GpuScene(crt, scene, ctx)
    fr = crt.make_frame(32, 32, 1, 0, 0); order = crt.make_order(mode, gw, gh, s)
    accum = torch.zeros((32, 32, 3), device=ctx.device)
    ctx.crt_render_frame(G.bvh, G.mats, G.camera, fr, order, 2, accum, ctx.frame_workspace(fr, order))
    assert torch.all(accum == 1.0)


def test_two_contexts_render_concurrently_without_interfering(crt, ctx):
    """bench.py keeps several frames in flight: one context + stream + workspace per frame (a crt_ctx serialises its own calls: its ray
    counter and event pool are per context).  Frames rendered concurrently on two contexts equal the same frames rendered alone."""
    import torch
    scene = _small_interior()
    w, h, spp, nb = 192, 128, 1, 2
    G = GpuScene(crt, scene.with_camera(w, h), ctx)
    ctx2 = crt.Context(0)
    mats2_dev = ctx2.upload(scene.materials); mats2 = ctx2.scene_mats(mats2_dev, len(scene.materials), scene.env)
    order = crt.make_order("direct_reuse", 4, 4, 4); fr0 = crt.make_frame(w, h, spp)
    lanes = [(ctx, G.mats, torch.cuda.Stream()), (ctx2, mats2, torch.cuda.Stream())]
    ws = [c.frame_workspace(fr0, order) for c, _, _ in lanes]
    alone = []
    for f in range(8):
        a = torch.zeros((h, w, 3), device=ctx.device)
        ctx.crt_render_frame(G.bvh, G.mats, G.camera, crt.make_frame(w, h, spp, 1, f), order, nb, a, ws[0])
        alone.append(a)
    torch.cuda.synchronize()
    acc = [torch.zeros((h, w, 3), device=ctx.device) for _ in range(8)]
    for f in range(8):
        c, m, st = lanes[f % 2]
        c.crt_render_frame(G.bvh, m, G.camera, crt.make_frame(w, h, spp, 1, f), order, nb, acc[f], ws[f % 2], stream=st)
    torch.cuda.synchronize()
    for f in range(8):
        assert torch.equal(acc[f], alone[f]), f


@pytest.mark.parametrize("mode,gw,gh,s", [("direct_reuse", 4, 4, 4), ("direct_reuse", 8, 8, 8 | (1 << 15)), ("independent", 1, 1, 1), ("world_reuse", 4, 4, 2 | (1 << 14))])
def test_frame_in_bands_gives_the_identical_image(crt, ctx, mode, gw, gh, s):
    """crt_set_option("frame_bands", n): a frame is cut into n bands of whole tiles, each running its whole sequence on its own stream so that one band's
    traversal tail is filled by the others' work (default 1 = off; only for frames of at least n * 262144 slots).  Same kernels on the same slots: the image and
    the live-ray counts must not change, bit for bit (1 spp: every pixel is written by exactly one thread)."""
    import torch
    scene = _small_interior().with_camera(1100, 779)                  # ragged against every tile size; 857 k paths
    G = GpuScene(crt, scene, ctx)
    order = crt.make_order(mode, gw, gh, s)
    fr = crt.make_frame(1100, 779, 1, 5, 2)
    assert crt.crt_layout(fr, order)[1] >= 3 * 262144
    ws = ctx.frame_workspace(fr, order)
    out = {}
    for bands in (1, 2, 3, 4):
        ctx.crt_set_option("frame_bands", bands)
        try:
            acc = torch.zeros((779, 1100, 3), device=ctx.device)
            nsec = torch.zeros(3, dtype=torch.int32, device=ctx.device)
            for f in range(2):
                ctx.crt_render_frame(G.bvh, G.mats, G.camera, crt.make_frame(1100, 779, 1, 5, f), order, 3, acc, ws, n_secondary=nsec)
            torch.cuda.synchronize()
            out[bands] = (acc.cpu().numpy(), nsec.cpu().numpy())
        finally:
            ctx.crt_set_option("frame_bands", 1)
    assert out[1][0].sum() > 0 and out[1][1].min() > 100000
    for bands in (2, 3, 4):
        assert np.array_equal(out[bands][0], out[1][0]) and np.array_equal(out[bands][1], out[1][1]), bands


def test_local_direction_reuse_is_unbiased_and_world_reuse_is_not(crt, ctx):
    """A statistical check of the method itself that does not go through the oracle: on an all-Lambert scene every group is a DIFFUSE group; each member
    uses the leader's LOCAL direction in its own tangent frame, so marginally its direction is cosine-distributed about its own normal and the pixel estimate is
    unbiased: the long-run mean image must agree with independent sampling's to within the noise floor (two independent means over disjoint frame ranges).  Sharing
    the WORLD direction (the paper's first variant, mode world_reuse) skews each member's distribution: its mean image must NOT agree (bench.py --sweep bias at full
    size: 1.00x the floor against 1.32x, profiles/r02j)."""
    import torch
    scene = I.cornell().with_camera(128, 128)
    G = GpuScene(crt, scene, ctx)
    F = 4096

    def mean_image(mode, g, s, first):
        order = crt.make_order(mode, g, g, s)
        ws = ctx.frame_workspace(crt.make_frame(128, 128), order)
        acc = torch.zeros((128, 128, 3), device=ctx.device)
        for f in range(F):
            ctx.crt_render_frame(G.bvh, G.mats, G.camera, crt.make_frame(128, 128, 1, 9, first + f), order, 2, acc, ws)
        torch.cuda.synchronize()
        return (acc / F).double()

    rm = lambda a, b: float(torch.sqrt(torch.mean((a - b) ** 2)).item())
    ind_a, ind_b = mean_image("independent", 1, 1, 0), mean_image("independent", 1, 1, 100000)
    floor = rm(ind_a, ind_b)
    assert 0.005 < floor < 0.1
    reuse = rm(mean_image("direct_reuse", 4, 4, 200000), ind_b)
    world = rm(mean_image("world_reuse", 4, 4, 200000), ind_b)
    print(f"noise floor {floor:.5f}, direct_reuse {reuse / floor:.3f}x, world_reuse {world / floor:.3f}x")
    assert reuse < 1.06 * floor, (reuse, floor)
    assert world > 1.15 * floor, (world, floor)


def test_argument_errors(crt, ctx):
    import torch
    scene = I.cornell()
    G = GpuScene(crt, scene, ctx)
    fr = crt.make_frame(64, 64)
    with pytest.raises(crt.CrtError) as e:
        crt.crt_layout(fr, crt.make_order("direct_reuse", 3, 4, 2))
    assert e.value.status == crt.api.CRT_ERR_UNSUPPORTED
    with pytest.raises(crt.CrtError) as e:
        crt.crt_layout(fr, crt.make_order("direct_reuse", 16, 16, 8))
    assert e.value.status == crt.api.CRT_ERR_UNSUPPORTED
    with pytest.raises(crt.CrtError) as e:
        crt.crt_layout(fr, crt.make_order(8))
    assert e.value.status == crt.api.CRT_ERR_INVALID_ARG
    order = crt.make_order("independent")
    rays, hits, r2p = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    paths = ctx.empty((64 * 64, 8)); ctx.crt_paths_init(paths)
    with pytest.raises(crt.CrtError) as e:
        ctx.crt_generate_secondary(G.bvh, G.mats, fr, 0, order, rays, hits, r2p, paths)     # bounce < 1
    assert e.value.status == crt.api.CRT_ERR_INVALID_ARG
    with pytest.raises(crt.CrtError):
        ctx.crt_set_option("no_such_option", 1)
    torch.cuda.synchronize()


def test_fused_shading_option_gives_the_identical_image(crt, ctx):
    """crt_set_option("fuse_shade", 0 / 1 (default)): same arithmetic inside the generation kernel; the image must not change."""
    import torch
    scene = _small_interior().with_camera(90, 61)
    G = GpuScene(crt, scene, ctx)
    imgs = []
    for mode, gw, gh, s in (("direct_reuse", 4, 4, 2), ("independent", 1, 1, 1), ("morton_reorder", 1, 1, 1), ("world_reuse", 4, 4, 2)):
        for fuse in (0, 1):
            ctx.crt_set_option("fuse_shade", fuse)
            try:
                order = crt.make_order(mode, gw, gh, s)
                fr = crt.make_frame(90, 61, 2, 5, 1)
                ws = ctx.frame_workspace(fr, order)
                acc = torch.zeros((61, 90, 3), device=ctx.device)
                ctx.crt_render_frame(G.bvh, G.mats, G.camera, fr, order, 3, acc, ws)
                torch.cuda.synchronize()
                imgs.append(acc.cpu().numpy())
            finally:
                ctx.crt_set_option("fuse_shade", 1)           # the default
        # 2 spp: the two samples of a pixel are added with atomicAdd in either order, so allow one rounding of difference
        assert imgs[-1].sum() > 0 and np.allclose(imgs[-2], imgs[-1], rtol=1e-6, atol=0)


def test_full_size_config4_sampled(crt, ctx, oracle):
    """BASELINE config 4 at full size (10,300,418 triangles, coordinates up to 2048): ALL hits of the primary segment and of both
    bounces of the direct_reuse frame equal the oracle's, a sample of them the all-triangles definition; the partition is the oracle's."""
    scene = I.landscape(seed=2).with_camera(1920, 1080)
    assert scene.n_tris == 10300418
    G = GpuScene(crt, scene, ctx)
    assert G.bvh.check() == 0
    w, h, spp, gw, gh, s = 1920, 1080, 1, 4, 4, 4
    fr = crt.make_frame(w, h, spp, 2, 1); ofr = oracle.frame(w, h, spp, 2, 1)
    order = crt.make_order("direct_reuse", gw, gh, s)
    rays0, hits0, r2p0 = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    assert np.array_equal(r2p0.cpu().numpy(), oracle.partition(ofr, 2, gw, gh, s))
    import torch
    n_paths = crt.crt_layout(fr, order)[0]
    paths = ctx.empty((n_paths, 8)); ctx.crt_paths_init(paths)
    accum = torch.zeros((h, w, 3), device=ctx.device)
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 0, False, rays0, hits0, r2p0, paths, accum)
    out = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 1, order, rays0, hits0, r2p0, paths)
    hits1 = ctx.crt_trace(G.bvh, out["rays"])
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 1, False, out["rays"], hits1, out["ray_to_path"], paths, accum)
    out2 = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 2, order, out["rays"], hits1, out["ray_to_path"], paths)
    hits2 = ctx.crt_trace(G.bvh, out2["rays"])
    # EVERY hit of the three segments against the oracle's BVH (10.3 M triangles; the 16-bit grid is coarsest here: 3 cm steps);
    # the oracle's BVH against the all-triangles definition on a sample
    ob = oracle.Bvh(scene.verts)
    rng = np.random.default_rng(12)
    for rays_dev, hits_dev, n_s in ((rays0, hits0, 40), (out["rays"], hits1, 80), (out2["rays"], hits2, 40)):
        r = rays_np(oracle, rays_dev); hh = hits_np(oracle, hits_dev)
        ho = ob.trace(r)
        assert compare_hits(hh, ho) >= 0.9999
        act = np.flatnonzero(r["tmax"] >= 0)
        pick = rng.choice(act, n_s, replace=False)
        ref = oracle.trace_brute(scene.verts, r[pick])
        assert np.array_equal(ho[pick], ref)
        compare_hits(hh[pick], ref)
        if n_s == 80:
            assert (ref["prim"] >= 0).any() and (ref["prim"] < 0).any()               # the secondary sample has terrain hits and sky misses


def test_full_size_config3_point_stagewise(crt, ctx, oracle):
    """BASELINE config 3 at its stated size, one sweep point: 3840x2160, 4 spp (33,177,600 paths), direct_reuse 8x8 stride 8
    (tile 64x64 = 4096 slots, the largest tile; 2160 is not a multiple of 64: partial tiles).  Partition == the oracle's and an
    exact cover; generation of bounce 1 fed the GPU's own primary hits == the oracle's on the same buffers (integer maps bit-exact,
    rays byte-identical); sampled primary and secondary hits == the oracle's BVH (== all-triangles definition on a subsample)."""
    import torch
    scene = I.interior(seed=1).with_camera(3840, 2160)
    G = GpuScene(crt, scene, ctx)
    w, h, spp, gw, gh, s = 3840, 2160, 4, 8, 8, 8
    fr = crt.make_frame(w, h, spp, 1, 0); ofr = oracle.frame(w, h, spp, 1, 0)
    order = crt.make_order("direct_reuse", gw, gh, s)
    n_paths, n_slots, n_groups = crt.crt_layout(fr, order)
    assert n_paths == 33177600 and n_slots == 4 * 60 * 34 * 4096 and n_groups * 64 == n_slots
    rays0, hits0, r2p0 = ctx.crt_trace_primary(G.bvh, G.camera, fr, order)
    r2p = r2p0.cpu().numpy()
    assert np.array_equal(r2p, oracle.partition(ofr, 2, gw, gh, s))
    live = r2p[r2p >= 0]
    assert len(live) == n_paths and np.array_equal(np.bincount(live, minlength=n_paths), np.ones(n_paths, np.int64))    # exact cover
    del live
    paths = ctx.empty((n_paths, 8)); ctx.crt_paths_init(paths)
    accum = torch.zeros((h, w, 3), device=ctx.device)
    ctx.crt_shade_accumulate(G.bvh, G.mats, fr, 0, False, rays0, hits0, r2p0, paths, accum)
    paths_before = paths_np(oracle, paths).copy()
    out = ctx.crt_generate_secondary(G.bvh, G.mats, fr, 1, order, rays0, hits0, r2p0, paths)
    bounds = np.asarray(G.bvh.info()["bounds"], np.float32)
    r0 = rays_np(oracle, rays0); h0 = hits_np(oracle, hits0)
    g = oracle.generate_secondary(scene, ofr, 1, 2, gw, gh, s, bounds, r0, h0, r2p, paths_before)
    for k in ("ray_to_path", "group_id", "dir_src", "group_class"):
        assert np.array_equal(out[k].cpu().numpy(), g[k]), k
    assert int(out["n_active"].cpu().numpy().view(np.uint32)[0]) == g["n_active"] > 20000000
    r1 = rays_np(oracle, out["rays"])
    assert r1.tobytes() == g["rays"].tobytes()
    pg = paths_np(oracle, paths)
    assert np.array_equal(pg["flags"] & 1, paths_before["flags"] & 1) and np.array_equal(pg["T"], paths_before["T"])
    del g, pg
    hits1 = ctx.crt_trace(G.bvh, out["rays"])
    h1 = hits_np(oracle, hits1)
    ob = oracle.Bvh(scene.verts)
    rng = np.random.default_rng(13)
    for r, hh in ((r0, h0), (r1, h1)):
        act = np.flatnonzero(r["tmax"] >= 0)
        pick = rng.choice(act, 200000, replace=False)
        ho = ob.trace(r[pick])
        compare_hits(hh[pick], ho)
        assert np.array_equal(ho[:100], oracle.trace_brute(scene.verts, r[pick[:100]]))
        assert np.all(hh["prim"][r["tmax"] < 0] == -1)
