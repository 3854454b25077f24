"""CPU-only checks of the C-ABI boundary: libcrt.so builds for sm_100a, loads, exports every symbol include/crt.h
declares, fails loudly without a CUDA device (no CPU fallback), and its host-side logic (layout arithmetic, BVH
builder invariants) is right.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import crt_inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2310_07182_b200 import build
    return C.CDLL(build.build())


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "crt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(crt_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert len(names) >= 24
    for n in names:
        assert hasattr(lib, n), f"libcrt.so does not export {n}"
    from paper_2310_07182_b200 import api
    assert sorted(api.EXPORTS) == names


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    st = lib.crt_create(C.c_int32(0), C.byref(h))
    assert st == 3 and not h.value                     # CRT_ERR_CUDA
    lib.crt_last_error.restype = C.c_char_p
    assert b"no CPU fallback" in lib.crt_last_error(None)
    import paper_2310_07182_b200 as crt
    with pytest.raises(crt.CrtError):
        crt.Context(0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2310_07182_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower().replace("no cpu fallback", ""), f"{f} mentions the oracle"


@pytest.mark.parametrize("w,h,spp,mode,gw,gh,s", [(64, 64, 1, 2, 4, 4, 2), (1920, 1080, 1, 2, 4, 4, 4), (3840, 2160, 4, 2, 8, 8, 8),
                                                  (50, 37, 2, 2, 2, 4, 4), (50, 37, 2, 3, 4, 4, 2), (1920, 1080, 1, 0, 1, 1, 1), (7, 5, 3, 1, 1, 1, 1), (7, 5, 3, 5, 1, 1, 1), (0, 0, 1, 2, 2, 2, 2),
                                                  (50, 37, 2, 2, 4, 4, 2 | (1 << 14))])            # lattice partition rule (D:R20)
def test_layout_matches_the_paper_parametrisation(lib, oracle, w, h, spp, mode, gw, gh, s):
    """tiles of W x H pixels, WH/K groups of K; K = gw*gh, W = gw*s, H = gh*s (reading R3)."""
    import paper_2310_07182_b200 as crt
    n_paths, n_slots, n_groups = crt.crt_layout(crt.make_frame(w, h, spp), crt.make_order(mode, gw, gh, s))
    assert n_paths == spp * w * h
    if mode in (2, 3):            # direct_reuse and world_reuse share the grouped slot space
        W, H = gw * (s & 0x3fff), gh * ((s >> 16) or (s & 0x3fff))
        tiles = -(-w // W) * -(-h // H)
        assert n_slots == spp * tiles * W * H and n_groups * gw * gh == n_slots
    else:
        assert n_slots == n_paths == n_groups
    ofr = oracle.frame(w, h, spp)
    assert n_slots == oracle.n_slots(ofr, mode, gw, gh, s) and n_groups == oracle.n_groups(ofr, mode, gw, gh, s)


def test_host_bvh_builder_invariants(lib):
    """ctx == NULL builds the host tree only: every triangle in exactly one leaf, leaves <= max_leaf, boxes nested."""
    from paper_2310_07182_b200 import api
    for scene, max_leaf in ((I.cornell(), 4), (I.interior(n_boxes=80, n_spheres=10, subdiv=2), 2), (I.landscape(n=96, n_trees=40), 8),
                            (I.cornell(), 1), (I.interior(n_boxes=80, n_spheres=10, subdiv=2), 1), (I.landscape(n=96, n_trees=40), 1)):
        v = np.ascontiguousarray(scene.verts, np.float32); m = np.ascontiguousarray(scene.mat_id, np.int32)
        pr = api.BvhParams(max_leaf, 16, 1.0, 1.0, 2)
        h = C.c_void_p()
        assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), C.c_void_p(m.ctypes.data), C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 0
        bad = C.c_int32(-1)
        assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and bad.value == 0
        info = api.BvhInfo()
        assert lib.crt_bvh_get_info(h, C.byref(info)) == 0
        assert info.n_tris == len(v) and info.max_leaf == max_leaf and 0 < info.depth <= 60
        assert len(v) / max_leaf <= (info.n_nodes + 1) / 2 <= len(v)
        assert np.array_equal(np.array(list(info.bounds), np.float32), np.concatenate([v.reshape(-1, 3).min(0), v.reshape(-1, 3).max(0)]))
        assert info.device_bytes == 0
        # 16-bit node layout: every plane at least one grid step outside its fp32 box (check bit 16 clear) and the decoded boxes
        # only slightly larger than the fp32 ones on scenes of this kind
        assert 100 <= info.q16_inflation_pct <= 125
        # the 8-wide compressed layout exists exactly when every leaf holds one triangle; crt_bvh_check covers its soundness too
        assert (info.n_wide_nodes > 0) == (max_leaf == 1)
        if max_leaf == 1:
            assert len(v) / 8 <= info.n_wide_nodes <= len(v) and 0 < info.wide_depth <= info.depth
        lib.crt_bvh_destroy(h)
    # degenerate inputs: no triangles, one triangle, many identical triangles (centroids coincide)
    for v in (np.zeros((0, 3, 3), np.float32), I.cornell().verts[:1], np.repeat(I.cornell().verts[:1], 37, axis=0)):
        v = np.ascontiguousarray(v)
        h = C.c_void_p()
        assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), None, C.byref(h)) == 0
        bad = C.c_int32(-1)
        assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and bad.value == 0
        lib.crt_bvh_destroy(h)
    # a unit-extent scene far from the origin (gmin is a float; its rounding must not eat the grid's margin): the 16-bit
    # layout still passes its own check, or -- when fp32 itself has too few bits left at that offset -- the check says so and the
    # kernel falls back to the fp32 nodes (launch_trace reads q_violations)
    rng = np.random.default_rng(3)
    tri = (rng.random((2000, 1, 3)) + 0.02 * rng.standard_normal((2000, 3, 3))).astype(np.float64)
    for offset in (0.0, 5e3, 1e4, 1e5, 3e6):
        v = np.ascontiguousarray(tri + offset, np.float32)
        h = C.c_void_p()
        assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), None, C.byref(h)) == 0
        bad = C.c_int32(-1)
        assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and (bad.value & 0xffff) == 0
        if offset <= 1e5:
            assert bad.value == 0, (offset, hex(bad.value))
        lib.crt_bvh_destroy(h)
    # rejected: NaN vertex, bad max_leaf, negative material id
    v = I.cornell().verts; m = np.zeros(len(v), np.int32); m[5] = -1
    h = C.c_void_p()
    assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), C.c_void_p(m.ctypes.data), C.c_int64(len(v)), None, C.byref(h)) == 1
    v = I.cornell().verts.copy(); v[3, 1, 2] = np.nan
    h = C.c_void_p()
    assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), None, C.byref(h)) == 1
    pr = api.BvhParams(9, 16, 1.0, 1.0, 1)
    v = I.cornell().verts
    assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 1


def test_scratch_size_queries(lib):
    import paper_2310_07182_b200 as crt
    lib.crt_radix_sort_scratch_bytes.restype = C.c_size_t
    lib.crt_frame_workspace_bytes.restype = C.c_size_t
    lib.crt_generate_secondary_scratch_bytes.restype = C.c_size_t
    assert lib.crt_radix_sort_scratch_bytes(C.c_int64(0)) >= 0
    n = 2073600
    assert lib.crt_radix_sort_scratch_bytes(C.c_int64(n)) >= 8 * n
    fr = crt.make_frame(1920, 1080)
    for mode, lo in (("independent", 0), ("morton_reorder", 32 + 5 * 4 + 8), ("direct_reuse", 0)):
        order = crt.make_order(mode, 4, 4, 4)
        assert lib.crt_generate_secondary_scratch_bytes(C.byref(fr), C.byref(order)) >= lo * n
        # rays x2, hits, 4 int maps, path state
        assert lib.crt_frame_workspace_bytes(C.byref(fr), C.byref(order)) >= (32 * 2 + 16 + 16 + 32) * n
    bad = crt.make_order("direct_reuse", 3, 3, 3)
    assert lib.crt_frame_workspace_bytes(C.byref(fr), C.byref(bad)) == 0


def test_native_tile_shapes_and_layout_errors(lib, oracle):
    """The paper's (W, H, K) through crt_order.stride_y; what the kernels do not implement is refused."""
    import paper_2310_07182_b200 as crt
    from paper_2310_07182_b200 import api
    fr = crt.make_frame(1920, 1080, 1)
    for tw, th, k in ((8, 8, 8), (16, 8, 16), (16, 16, 32), (32, 8, 64), (8, 8, 64), (4, 4, 1)):
        o = crt.order_for_tile("direct_reuse", tw, th, k)
        assert o.group_w * o.stride == tw and o.group_h * (o.stride_y or o.stride) == th and o.group_w * o.group_h == k
        n_paths, n_slots, n_groups = crt.crt_layout(fr, o)
        tiles = -(-1920 // tw) * -(-1080 // th)
        assert n_slots == tiles * tw * th and n_groups * k == n_slots
        assert n_slots == oracle.n_slots(oracle.frame(1920, 1080, 1), 2, o.group_w, o.group_h, o.stride | ((o.stride_y or 0) << 16))
    for bad in (crt.make_order("direct_reuse", 3, 4, 2), crt.make_order("direct_reuse", 4, 4, 2, 3), crt.make_order("direct_reuse", 64, 64, 2),
                crt.make_order("direct_reuse", 4, 4, 0)):
        n = C.c_int64()
        assert lib.crt_layout(C.byref(fr), C.byref(bad), C.byref(n), None, None) == api.CRT_ERR_UNSUPPORTED
    for bad_mode in (-1, 8):
        o = api.Order(bad_mode, 1, 1, 1, 0, 0); n = C.c_int64()
        assert lib.crt_layout(C.byref(fr), C.byref(o), C.byref(n), None, None) == api.CRT_ERR_INVALID_ARG


def test_presplit_builds_a_tree_over_references(lib):
    """crt_bvh_params.presplit: a triangle whose box is longer than presplit x the scene diagonal gets several references (one per cell of a midpoint
    split of its box, each with the box of the part of the triangle inside the cell).  Host-only builds: more references than triangles, the tree passes
    its check (every triangle referenced; the boxes of a multiply referenced triangle's leaves together cover it; leaves <= max_leaf; boxes nested), the
    bounds stay the vertices' exact min / max, and one-triangle-per-leaf builds (which feed the 8-wide layout) are never split."""
    from paper_2310_07182_b200 import api
    one_big = np.array([[[0, 0, 0], [100, 0, 0], [0, 100, 3]]], np.float32)                   # a single triangle: 1 -> many references
    sliver = np.concatenate([one_big, np.array([[[5, 5, 5], [5.1, 5, 5], [5, 5.1, 5]]], np.float32)])
    for verts, max_leaf, ps, split in ((I.cornell().verts, 3, 1 / 16, True), (I.cornell().verts, 3, 0.0, False), (I.cornell().verts, 1, 1 / 16, False),
                                       (I.interior(n_boxes=80, n_spheres=10, subdiv=2).verts, 2, 1 / 16, True), (I.landscape(n=96, n_trees=40).verts, 4, 1 / 64, True),
                                       (one_big, 3, 1 / 16, True), (sliver, 2, 1 / 32, True), (I.cornell().verts + np.float32(3e5), 3, 1 / 16, True)):
        v = np.ascontiguousarray(verts, np.float32)
        pr = api.BvhParams(max_leaf, 64, 1.0, 1.0, 2, 0, 0, ps)
        h = C.c_void_p()
        assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 0
        bad = C.c_int32(-1)
        assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and bad.value == 0, (len(v), max_leaf, ps, bad.value)
        info = api.BvhInfo()
        assert lib.crt_bvh_get_info(h, C.byref(info)) == 0
        assert info.n_tris == len(v) and (info.n_refs > info.n_tris) == split and info.n_refs <= info.n_tris + max(info.n_tris // 4, 4096)
        assert np.array_equal(np.array(list(info.bounds), np.float32), np.concatenate([v.reshape(-1, 3).min(0), v.reshape(-1, 3).max(0)]))
        lib.crt_bvh_destroy(h)
    for ps in (-0.1, 1.5, float("nan")):
        pr = api.BvhParams(3, 64, 1.0, 1.0, 1, 0, 0, ps); h = C.c_void_p()
        assert lib.crt_build_bvh(None, C.c_void_p(one_big.ctypes.data), None, C.c_int64(1), C.byref(pr), C.byref(h)) == 1


def test_tree_optimisation_keeps_the_invariants_and_lowers_the_cost(lib):
    """crt_bvh_params.optimize: insertion-based optimisation of the built tree.  Host-only builds: the same number of nodes and references, the check still
    passes (every triangle in one leaf, leaves <= max_leaf, boxes nested: the restructured tree is a valid BVH over the same leaves), the SAH cost does not rise
    (on the cornell and interior scenes it falls by 2-8 %), the depth stays inside the traversal stack."""
    from paper_2310_07182_b200 import api
    for scene, max_leaf, ps in ((I.cornell(), 3, 0.0), (I.interior(n_boxes=80, n_spheres=10, subdiv=2), 3, 1 / 16), (I.landscape(n=96, n_trees=40), 4, 0.0), (I.interior(n_boxes=40, n_spheres=5, subdiv=1), 1, 0.0)):
        v = np.ascontiguousarray(scene.verts, np.float32)
        got = {}
        for opt in (0, 3, 40):
            pr = api.BvhParams(max_leaf, 64, 1.0, 1.0, 1, 0, 0, ps, opt)          # one thread: the unoptimised tree is the same in the three builds
            h = C.c_void_p()
            assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 0
            bad = C.c_int32(-1)
            assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and bad.value == 0, (scene.name, opt, bad.value)
            info = api.BvhInfo(); assert lib.crt_bvh_get_info(h, C.byref(info)) == 0
            got[opt] = (info.n_nodes, info.n_refs, info.sah_cost, info.depth)
            lib.crt_bvh_destroy(h)
        assert got[0][:2] == got[3][:2] == got[40][:2]
        assert got[40][2] <= got[3][2] * 1.0001 and got[3][2] <= got[0][2] * 1.0001, got
        assert scene.name == "landscape" or got[40][2] < got[0][2] * 0.995, got          # (a terrain grid gains next to nothing and the optimisation stops early)
        assert got[40][3] <= 60
    pr = api.BvhParams(3, 64, 1.0, 1.0, 1, 0, 0, 0.0, -1); h = C.c_void_p()
    v = np.ascontiguousarray(I.cornell().verts, np.float32)
    assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 1


def test_builder_steps_on_degenerate_inputs(lib):
    """Pre-splitting and tree optimisation on inputs that could break them: point and collinear triangles, hundreds of identical triangles (identical boxes can
    be chained into a list: the optimisation must not deepen the tree beyond the traversal stack), slivers, one giant triangle among tiny ones, coordinates
    far from the origin.  Every build succeeds and passes its check."""
    from paper_2310_07182_b200 import api
    rng = np.random.default_rng(7)
    cases = {
        "points": np.repeat(rng.random((500, 1, 3)), 3, axis=1),
        "identical": np.tile(rng.random((1, 3, 3)), (300, 1, 1)),
        "identical big": np.tile(rng.random((1, 3, 3)) * 100, (2000, 1, 1)),
        "slivers": np.stack([rng.random((200, 3)) * 100, rng.random((200, 3)) * 100, rng.random((200, 3)) * 100], 1) * np.array([1, 1e-6, 1e-6]),
        "giant+tiny": np.concatenate([np.array([[[-1e4, 0, -1e4], [1e4, 0, -1e4], [0, 0, 1e4]]]), rng.random((3000, 3, 3)) * 0.01 + rng.random((3000, 1, 3)) * 10]),
        "collinear": np.stack([np.zeros((50, 3)), np.ones((50, 3)), 2 * np.ones((50, 3))], 1) * rng.random((50, 1, 1)) * 50,
        "offset": rng.random((1000, 3, 3)) + 4e6,
        "two": rng.random((2, 3, 3)) * 1000,
    }
    for name, verts in cases.items():
        v = np.ascontiguousarray(verts, np.float32)
        for max_leaf in (1, 3, 8):
            for ps, opt in ((1 / 16, 20), (1 / 256, 50), (0.0, 200)):
                pr = api.BvhParams(max_leaf, 64, 1.0, 1.0, 2, 0, 0, ps, opt); h = C.c_void_p()
                assert lib.crt_build_bvh(None, C.c_void_p(v.ctypes.data), None, C.c_int64(len(v)), C.byref(pr), C.byref(h)) == 0, (name, max_leaf, ps, opt)
                bad = C.c_int32(-1)
                assert lib.crt_bvh_check(h, C.byref(bad)) == 0 and bad.value == 0, (name, max_leaf, ps, opt, bad.value)
                info = api.BvhInfo(); assert lib.crt_bvh_get_info(h, C.byref(info)) == 0 and info.depth <= 60
                lib.crt_bvh_destroy(h)


def test_q16_box_test_error_budget():
    """The 16-bit-node box test evaluates a plane distance as t = (2^23 + q) * s + c in fp32 (csrc/trace.cu: QRay).  Re-enacting
    that arithmetic in numpy against the exact (q - o') * s shows the budget the kernel's comment states: the error, in grid steps
    of position, stays below the ONE step by which crt_bvh_quantise pads the planes for ray origins within 16 scene extents (the contract
    of include/crt.h) — dominated by the half step of rounding c inside the scene — and passes one step somewhere beyond 20 extents,
    which is why the contract exists."""
    rng = np.random.default_rng(3)
    f32 = np.float32
    n = 200000
    fma = lambda a, b, c: (a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64)).astype(f32)
    seen = {}
    for reach, bound in ((1.0, 0.53), (16.0, 0.92), (60.0, None)):
        gmin = f32(rng.uniform(-50, 50)); ext = rng.uniform(1, 2000)
        scale = f32((65535.0 - 16.0) / ext); inv_scale = f32(1.0 / np.float64(scale))
        o = (np.float64(gmin) + rng.uniform(-reach, reach + 1, n) * ext).astype(f32)
        d = (rng.choice([-1.0, 1.0], n) * np.exp(rng.uniform(np.log(1e-6), 0.0, n))).astype(f32)
        q = rng.integers(0, 65536, n)
        idx = (f32(1.0) / d).astype(f32)
        s = (idx * inv_scale).astype(f32)
        p = ((o - gmin).astype(f32) * scale).astype(f32)
        c = fma(np.full(n, -8388608.0, f32), s, -(p * s).astype(f32))
        t = fma((8388608.0 + q).astype(f32), s, c)
        # exact: the grid and the ray as given (fp32 values taken as exact reals)
        o_steps = (o.astype(np.float64) - np.float64(gmin)) * np.float64(scale)
        t_exact = (q - o_steps) / (d.astype(np.float64) * np.float64(scale))
        err_steps = np.abs(t.astype(np.float64) - t_exact) * np.abs(d.astype(np.float64)) * np.float64(scale)
        seen[reach] = err_steps.max()
        if bound is not None:
            assert err_steps.max() <= bound, (reach, err_steps.max())
        assert err_steps.max() > 0.3                       # the half step of rounding c is real: the padding is needed
    assert seen[60.0] > 1.0                                # beyond the contract the one step of padding is not enough
