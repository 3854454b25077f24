"""Pins for the oracle functions that the round-1 review found unpinned ("What's weak" 1): the Smith G1 /
Schlick factors of the GGX weight, ggx_weight of a given direction, the pinhole camera and the shading point's position.
Nothing here re-types the oracle's code: the checks are fp64 quadrature of the textbook microfacet integral, analytic
pinhole geometry and the ray equation o + t d on axis-aligned walls (CPU only).

Each pin was checked to FAIL under the mutation it is there for (alpha*alpha*tan2 -> alpha*tan2; Schlick exponent 5 -> 4 in
sample_ggx and in ggx_weight; sy = 1 - 2 fy -> 2 fy - 1; u and v swapped in the hit position)."""
import math

import numpy as np
import pytest

import crt_inputs as I

M_IND, M_REUSE, M_WORLD = 0, 2, 3


# ------------------------------------------------------------------ GGX weight: Smith G1 and Schlick F ("glossy"; D:R9)
def _ggx_terms(wo, alpha, f0, WI):
    """Textbook single-scattering GGX terms for exit directions WI[..., 3] (fp64): D(h), G1(wo), G1(wi), Schlick F(wo.h)."""
    H = wo + WI
    H = H / np.linalg.norm(H, axis=-1, keepdims=True)
    D = alpha**2 / (math.pi * ((H[..., 2] ** 2) * (alpha**2 - 1) + 1) ** 2)

    def g1(w):
        tan2 = (w[..., 0] ** 2 + w[..., 1] ** 2) / np.maximum(w[..., 2] ** 2, 1e-300)
        return 2 / (1 + np.sqrt(1 + alpha**2 * tan2))
    woh = np.clip((H * wo).sum(-1), 0, 1)
    F = f0 + (1 - f0) * (1 - woh) ** 5
    return D, g1(wo[None, None, :])[0, 0], g1(WI), F


def _hemisphere_grid(nt, nph):
    ct = (np.arange(nt) + 0.5) / nt
    ph = (np.arange(nph) + 0.5) / nph * 2 * math.pi
    CT, PH = np.meshgrid(ct, ph, indexing="ij"); ST = np.sqrt(1 - CT**2)
    return np.stack([ST * np.cos(PH), ST * np.sin(PH), CT], -1), 2 * math.pi / (nt * nph)


@pytest.mark.parametrize("alpha,theta", [(0.5, 0.3), (0.2, 1.0), (0.35, 1.35)])
def test_ggx_weight_integrates_to_the_directional_albedo(oracle, alpha, theta):
    """E_samples[weight] (invalid samples count 0) == int F(wo.h) D(h) G1(wo) G1(wi) / (4 wo.z) dwi over the upper hemisphere,
    the single-scattering directional albedo of the separable-Smith GGX BRDF, by fp64 quadrature; for F0 = 1 (F == 1: Smith G1
    alone) and for a coloured F0 (Schlick).  Also P(valid sample) == int D(h) G1(wo) / (4 wo.z) dwi (the VNDF pdf of wi)."""
    wo = np.array([math.sin(theta) * 0.8, math.sin(theta) * 0.6, math.cos(theta)])
    WI, dw = _hemisphere_grid(3000, 1440)
    n = 192
    u = (np.arange(n) + 0.5) / n
    f0s = ((1.0, 1.0, 1.0), (0.3, 0.04, 0.8))
    for f0 in f0s:
        got = np.zeros(3); n_valid = 0
        for a in u:
            for b in u:
                ok, wi, wt = oracle.sample_ggx_f0(wo, alpha, f0, float(a), float(b))
                if ok:
                    got += wt; n_valid += 1
        got /= n * n
        for k in range(3):
            D, g1o, g1i, F = _ggx_terms(wo, alpha, f0[k], WI)
            exp = (F * D * g1o * g1i).sum() * dw / (4 * wo[2])
            assert abs(got[k] - exp) < 4e-3, (f0, k, got[k], exp)
        p_valid = (D * g1o).sum() * dw / (4 * wo[2])
        assert abs(n_valid / (n * n) - p_valid) < 4e-3


def test_ggx_weight_of_a_given_direction_equals_the_sampled_weight(oracle):
    """ggx_weight(wo, wi) (world-space reuse, D:R18: "calculating the probability based on the direction and their respective
    materials") is the weight sample_ggx returns when it samples that same wi: F(wo.h) G1(wi) with h = normalize(wo + wi)."""
    rng = np.random.default_rng(5)
    f0 = (0.3, 0.6, 0.9)
    n = 0
    for _ in range(400):
        th = rng.uniform(0.05, 1.45); ph = rng.uniform(0, 2 * math.pi); alpha = rng.uniform(0.1, 0.6)
        wo = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)], np.float32)
        ok, wi, wt = oracle.sample_ggx_f0(wo, alpha, f0, rng.random(), rng.random())
        if not ok:
            continue
        ok2, wt2 = oracle.ggx_weight(wo, wi, alpha, f0)
        assert ok2 and np.allclose(wt2, wt, rtol=2e-5, atol=2e-6), (wo, wi, wt, wt2)
        # and against the textbook terms in fp64
        for k in range(3):
            D, g1o, g1i, F = _ggx_terms(wo.astype(np.float64), alpha, f0[k], wi.astype(np.float64)[None, None, :])
            assert abs(wt2[k] - F[0, 0] * g1i[0, 0]) < 1e-4 * max(1.0, wt2[k]) + 1e-5
        n += 1
    assert n > 300
    # opposite directions: wo + wi vanishes -> no weight
    ok3, _ = oracle.ggx_weight((0, 0, 1), (0, 0, -1), 0.3, f0)
    assert not ok3


# ------------------------------------------------------------------ pinhole camera (D:R6)
def test_camera_ray_is_the_analytic_pinhole(oracle):
    """Pixel (x, y) looks through screen point (sx, sy) in its own pixel cell, sx growing to the RIGHT of the view and sy UP:
    solve d ~ W + sx U + sy V for (sx, sy) in fp64 and locate it in the cell; the position inside the cell is the Philox CAMERA
    jitter.  Image of a target plane: the top-left pixel sees the up-left corner region, the centre pixel the look-at point."""
    w, h = 40, 24
    eye = np.array([0.3, 1.2, 5.0]); target = np.array([0.1, 0.9, 0.0])
    cam = I.make_camera(eye, target, (0, 1, 0), 50.0, w / h)
    # a big wall z = 0 facing the camera
    wall = np.array([[[-50, -50, 0], [50, -50, 0], [50, 50, 0]], [[-50, -50, 0], [50, 50, 0], [-50, 50, 0]]], np.float32)
    b = oracle.Bvh(wall)
    for seed, frame, spp in ((0, 0, 1), (7, 3, 2)):
        fr = oracle.frame(w, h, spp, seed, frame)
        rays, hits, r2p = oracle.trace_primary(b, cam, fr, M_IND)
        assert np.array_equal(r2p, np.arange(spp * w * h)) and np.all(hits["prim"] >= 0)
        assert np.all(rays["o"] == cam[:3]) and np.all(rays["tmin"] == 0) and np.all(rays["tmax"] == np.float32(1e30))
        d = rays["d"].astype(np.float64)
        assert np.allclose(np.linalg.norm(d, axis=1), 1, atol=2e-7)
        U, V, W = (cam[3:6].astype(np.float64), cam[6:9].astype(np.float64), cam[9:12].astype(np.float64))
        # d * lam = W + sx U + sy V  ->  [U V -d] (sx sy lam)^T = -W
        A = np.stack([np.broadcast_to(U, d.shape), np.broadcast_to(V, d.shape), -d], axis=2)
        sol = np.linalg.solve(A, np.broadcast_to(-W, d.shape)[..., None])[..., 0]
        sx, sy, lam = sol[:, 0], sol[:, 1], sol[:, 2]
        assert np.all(lam > 0)
        p = np.arange(spp * w * h); x = p % w; y = (p // w) % h; sg = p // (w * h)
        fx = (sx + 1) / 2 * w - x; fy = (1 - sy) / 2 * h - y             # position inside the pixel cell, y DOWN the image
        assert np.all(fx > -1e-4) and np.all(fx < 1 + 1e-4) and np.all(fy > -1e-4) and np.all(fy < 1 + 1e-4)
        # the jitter is the CAMERA stream of the pixel: counter (pixel, sample, 0, purpose 0), key (seed, frame)  (D:R2, R6)
        for i in (0, 1, w, w * h - 1, spp * w * h - 1, 333):
            r = oracle.philox(int(y[i] * w + x[i]), int(sg[i]), 0, 0, seed, frame)
            assert abs(fx[i] - oracle.u01(r[0])) < 2e-4 and abs(fy[i] - oracle.u01(r[1])) < 2e-4
        assert 0.4 < fx.mean() < 0.6 and 0.4 < fy.mean() < 0.6 and fx.std() > 0.25 and fy.std() > 0.25
        # where the rays land on the wall z = 0
        hit = eye + hits["t"].astype(np.float64)[:, None] * d
        assert np.allclose(hit[:, 2], 0, atol=1e-5)
        img = hit.reshape(spp, h, w, 3)[0]
        assert np.all(img[:, 1:, 0] > img[:, :-1, 0] - 0.05 * abs(img[0, 1, 0] - img[0, 0, 0]))     # x grows to the right ...
        assert img[:, -1, 0].min() > img[:, 0, 0].max()
        assert img[0, :, 1].min() > img[-1, :, 1].max()                    # ... and row 0 is the TOP of the view (world y up)
        c = 0.25 * (img[h // 2 - 1, w // 2 - 1] + img[h // 2, w // 2 - 1] + img[h // 2 - 1, w // 2] + img[h // 2, w // 2])
        cell = abs(img[h // 2, w // 2, 0] - img[h // 2, w // 2 - 1, 0])
        assert np.all(np.abs(c[:2] - target[:2]) < cell)                  # the image centre looks at the target
        # corner pixels against normalize(W -/+ U +/- V) within one pixel's angle
        pix_angle = 2 * np.linalg.norm(U) / w + 2 * np.linalg.norm(V) / h
        for (px, py, su, sv) in ((0, 0, -1, 1), (w - 1, 0, 1, 1), (0, h - 1, -1, -1), (w - 1, h - 1, 1, -1)):
            e = W + su * U + sv * V; e /= np.linalg.norm(e)
            assert np.linalg.norm(d[py * w + px] - e) < pix_angle


# ------------------------------------------------------------------ shading point position and offset (D:R7)
@pytest.mark.parametrize("mode", [M_IND, M_REUSE, M_WORLD])
def test_secondary_origin_is_the_hit_point_offset_along_the_wall_normal(oracle, mode):
    """On Cornell's axis-aligned walls the next ray starts at o_prev + t d_prev (ray equation, fp64) moved by
    2^-15 (1 + max|p_i|) along the wall's normal toward the side the ray came from; all three components."""
    sc = I.cornell()
    fr = oracle.frame(sc.width, sc.height, 1, 0, 0)
    b = oracle.Bvh(sc.verts)
    rays, hits, r2p = oracle.trace_primary(b, sc.camera, fr, mode, 4, 4, 2)
    paths = oracle.paths_init(sc.width * sc.height)
    accum = np.zeros((sc.height, sc.width, 3), np.float32)
    oracle.shade_accumulate(sc, fr, 0, False, rays, hits, r2p, paths, accum)
    g = oracle.generate_secondary(sc, fr, 1, mode, 4, 4, 2, b.info()["bounds"], rays, hits, r2p, paths)
    # previous slot of every path
    prev_slot = np.full(sc.width * sc.height, -1, np.int64); ok = r2p >= 0; prev_slot[r2p[ok]] = np.nonzero(ok)[0]
    act = g["rays"]["tmax"] >= 0
    ps = prev_slot[g["ray_to_path"][act]]
    o_prev = rays["o"][ps].astype(np.float64); d_prev = rays["d"][ps].astype(np.float64); t = hits["t"][ps].astype(np.float64)
    p = o_prev + t[:, None] * d_prev
    tri = sc.verts[hits["prim"][ps]].astype(np.float64)
    n = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0]); n /= np.linalg.norm(n, axis=1, keepdims=True)
    axis_aligned = np.isclose(np.abs(n).max(1), 1.0, atol=1e-12)
    assert axis_aligned.sum() > 1000                                      # floor, ceiling, back, left, right (+ tops of the boxes)
    n[(n * d_prev).sum(1) > 0] *= -1                                       # toward the incoming side
    kappa = 2.0 ** -15
    exp = p + n * (kappa * (1 + np.abs(p).max(1)))[:, None]
    got = g["rays"]["o"][act].astype(np.float64)
    assert np.all(np.abs(got - exp)[axis_aligned] < 1e-5)
    # everywhere (tilted boxes too): the origin lies on the hit triangle's plane lifted by the offset, and at the ray equation's point
    lift = ((got - tri[:, 0]) * n).sum(1)
    assert np.allclose(lift, kappa * (1 + np.abs(p).max(1)), atol=2e-6)
    assert np.all(np.abs(got - exp) < 2e-5)
    # the hit position in barycentric form (P:L69 shading point = first hit): v0 + u (v1 - v0) + v (v2 - v0), independent of the ray
    u = hits["u"][ps].astype(np.float64); v = hits["v"][ps].astype(np.float64)
    pb = tri[:, 0] + u[:, None] * (tri[:, 1] - tri[:, 0]) + v[:, None] * (tri[:, 2] - tri[:, 0])
    assert np.all(np.abs(pb - p) < 5e-6)


# ------------------------------------------------------------------ pins added after a second mutation sweep (leader rule, tile constants, hybrid with one glossy sample,
#                                                                    BSDF stream per bounce, group ids)
def _first_bounce(oracle, scene, mode, gw=4, gh=4, s=2, frame=0, spp=1, seed=0):
    fr = oracle.frame(scene.width, scene.height, spp, seed, frame)
    b = oracle.Bvh(scene.verts)
    rays, hits, r2p = oracle.trace_primary(b, scene.camera, fr, mode, gw, gh, s)
    paths = oracle.paths_init(spp * scene.width * scene.height)
    accum = np.zeros((scene.height, scene.width, 3), np.float32)
    oracle.shade_accumulate(scene, fr, 0, False, rays, hits, r2p, paths, accum)
    out = oracle.generate_secondary(scene, fr, 1, mode, gw, gh, s, b.info()["bounds"], rays, hits, r2p, paths)
    out.update(prev_rays=rays, prev_hits=hits, prev_r2p=r2p, paths=paths, fr=fr, bvh=b, accum=accum)
    return out


def _member_types(sc, g):
    """material type of the primary hit of every slot's path (-1: no path / miss)"""
    ok = g["prev_r2p"] >= 0
    prim_of_path = np.full(sc.width * sc.height, -1); prim_of_path[g["prev_r2p"][ok]] = g["prev_hits"]["prim"][ok]
    p = g["ray_to_path"]
    pr = np.where(p >= 0, prim_of_path[np.maximum(p, 0)], -1)
    return np.where(pr >= 0, sc.materials["type"][sc.mat_id[np.maximum(pr, 0)]], -1)


@pytest.mark.parametrize("mode", [M_REUSE, M_WORLD])
def test_leader_is_the_first_eligible_member_in_cyclic_order_from_the_leader_stream(oracle, mode):
    """"Randomly selects one pixel" (D:R8, R18): start slot j0 = Philox(group, sample, bounce, LEADER).r0 mod K, then the first live DIFFUSE member in
    cyclic slot order (tangent-space reuse) / the first live member of ANY material (world-space reuse).  Expected leaders are recomputed here from the pinned
    Philox and the members' materials."""
    # world mode: Lambert, GGX and mirror cells, so leaders of every material occur; tangent mode: mostly-Lambert floor, so many all-diffuse groups
    sc = I.checker_floor() if mode == M_WORLD else I.checker_floor(p_diffuse=0.97)
    K = 16
    g = _first_bounce(oracle, sc, mode)
    mt = _member_types(sc, g).reshape(-1, K); p = g["ray_to_path"].reshape(-1, K); src = g["dir_src"].reshape(-1, K)
    act = g["rays"]["tmax"].reshape(-1, K) >= 0
    n_checked = n_glossy_leader = 0
    for gi in range(len(p)):
        live = (mt[gi] >= 0) & (mt[gi] != I.MAT_EMISSIVE)
        elig = live & (mt[gi] == I.MAT_DIFFUSE) if mode == M_REUSE else live
        if mode == M_REUSE and ((mt[gi] == I.MAT_GLOSSY) | (mt[gi] == I.MAT_SPECULAR)).any():
            continue                                      # hybrid groups take the glossy mean instead (separate test)
        if not elig.any():
            continue
        j0 = oracle.philox(gi, 0, 1, 3, 0, 0)[0] % K
        lead_slot = next(j % K for j in range(j0, j0 + K) if elig[j % K])
        reusers = act[gi] & (src[gi] != p[gi]) if mode == M_WORLD else act[gi] & elig
        if reusers.any():
            assert np.all(src[gi][reusers] == p[gi][lead_slot]), (gi, j0, lead_slot)
            n_checked += 1
            n_glossy_leader += int(mt[gi][lead_slot] != I.MAT_DIFFUSE)
    assert n_checked > (20 if mode == M_REUSE else 50) and (mode == M_REUSE or n_glossy_leader > 5)


def test_tile_shuffle_constants_come_from_the_tile_stream(oracle):
    """D:R3: m = (a n + c) mod M with a = (r0 mod M) | 1, c = r1 mod M, (r0, r1) = Philox(tile, sample, 0, TILE; seed, frame)."""
    fr = oracle.frame(64, 48, 2, seed=9, frame=4)
    for gw, gh, s in ((4, 4, 2), (2, 2, 4), (8, 4, 1)):
        W, H = gw * s, gh * s; M = W * H
        pos = oracle.partition(fr, M_REUSE, gw, gh, s)
        tiles_x, tiles_y = 64 // W, 48 // H
        for sample in (0, 1):
            for tile in (0, 3, tiles_x * tiles_y - 1):
                blk = pos[(sample * tiles_x * tiles_y + tile) * M:][:M]
                tx, ty = tile % tiles_x, tile // tiles_x
                pix = blk % (64 * 48)
                n_of_m = ((pix // 64) - ty * H) * W + ((pix % 64) - tx * W)
                r = oracle.philox(tile, sample, 0, 2, 9, 4)
                a, c = (r[0] % M) | 1, r[1] % M
                assert np.array_equal((a * n_of_m + c) % M, np.arange(M))
                assert np.all(blk // (64 * 48) == sample)


def test_hybrid_group_with_a_single_glossy_sample_and_group_ids(oracle):
    """the diffuse members of a hybrid group take the mean glossy direction also when ONE glossy member produced it; group_id = slot / K in the grouped
    modes and the path id otherwise."""
    sc = I.checker_floor(p_diffuse=0.85)                 # mostly Lambert: many groups with exactly one glossy / mirror member
    K = 16
    g = _first_bounce(oracle, sc, M_REUSE)
    mt = _member_types(sc, g).reshape(-1, K); src = g["dir_src"].reshape(-1, K); p = g["ray_to_path"].reshape(-1, K)
    act = g["rays"]["tmax"].reshape(-1, K) >= 0
    loc = g["local_dir"].reshape(-1, K, 3)
    n_single = 0
    for gi in np.nonzero(g["group_class"] == oracle.CLASS_HYBRID)[0]:
        gl = (mt[gi] == I.MAT_GLOSSY) | (mt[gi] == I.MAT_SPECULAR)
        valid = gl & act[gi]
        dif = mt[gi] == I.MAT_DIFFUSE
        if valid.sum() >= 1:
            assert np.all(src[gi][dif & act[gi]] == -2 - gi) and (dif & act[gi]).sum() == dif.sum()
        if valid.sum() == 1:
            assert np.allclose(loc[gi][dif], loc[gi][valid][0], atol=1e-6)
            n_single += 1
    assert n_single >= 10
    assert np.array_equal(g["group_id"], np.arange(len(g["ray_to_path"])) // K)
    gi_ = _first_bounce(oracle, sc, M_IND)
    assert np.array_equal(gi_["group_id"], gi_["ray_to_path"])
    gm = _first_bounce(oracle, sc, 1)
    assert np.array_equal(gm["group_id"], gm["ray_to_path"])


def test_bsdf_stream_is_keyed_by_pixel_sample_and_bounce(oracle):
    """north_star: "Philox keyed by pixel, sample and bounce" (D:R2): a Lambert path's local direction at bounce b is sample_cosine of the first two floats of
    Philox(pixel, sample, b, BSDF; seed, frame) — checked at bounce 1 and bounce 2 (so consecutive bounces draw different numbers), 2 spp."""
    sc = I.emissive_box(albedo=0.8)                      # closed Lambert cube: every path lives on
    w, h, spp, seed, frame = sc.width, sc.height, 2, 6, 2
    fr = oracle.frame(w, h, spp, seed, frame)
    b = oracle.Bvh(sc.verts)
    rays, hits, r2p = oracle.trace_primary(b, sc.camera, fr, M_IND)
    paths = oracle.paths_init(spp * w * h)
    for bounce in (1, 2):
        g = oracle.generate_secondary(sc, fr, bounce, M_IND, 1, 1, 1, b.info()["bounds"], rays, hits, r2p, paths)
        for path in (0, 7, w * h - 1, w * h + 5, 2 * w * h - 1):
            r = oracle.philox(path % (w * h), path // (w * h), bounce, 1, seed, frame)
            exp = oracle.sample_cosine(oracle.u01(r[0]), oracle.u01(r[1]))
            assert np.array_equal(g["local_dir"][path], exp.astype(np.float32)), (bounce, path)
        rays, r2p = g["rays"], g["ray_to_path"]
        hits = b.trace(rays)
