"""Pins for the oracle's partition, classification, reuse rules, sampling, Morton code,
sort and shading (CPU only).  Nothing here re-types the oracle's formulas: the checks are
invariants the paper states, closed forms, library routines and fp64 quadrature."""
import math

import numpy as np
import pytest

import crt_inputs as I

M_IND, M_MOR, M_REUSE, M_WORLD = 0, 1, 2, 3


# ------------------------------------------------------------------ partition
def _tile(tw, th, k):
    """the paper's native (W, H, K) as (gw, gh, s) with the vertical stride in the high half of s"""
    gw = min(k, tw); gh = k // gw
    return gw, gh, (tw // gw) | ((th // gh) << 16)


@pytest.mark.parametrize("gw,gh,s", [(2, 2, 1), (2, 2, 8), (4, 4, 2), (4, 4, 4), (8, 8, 1), (8, 8, 8), (4, 2, 2), (1, 1, 4),
                                     _tile(8, 8, 8), _tile(16, 8, 16), _tile(32, 8, 64), _tile(16, 16, 32)])      # Table 3's shapes
@pytest.mark.parametrize("w,h,spp", [(64, 64, 1), (50, 37, 2)])
def test_partition_is_exact_cover(oracle, gw, gh, s, w, h, spp):
    fr = oracle.frame(w, h, spp, seed=3, frame=5)
    pos = oracle.partition(fr, M_REUSE, gw, gh, s)
    W, H = gw * (s & 0xffff), gh * ((s >> 16) or (s & 0xffff))
    M, K = W * H, gw * gh
    tiles_x, tiles_y = -(-w // W), -(-h // H)
    assert len(pos) == spp * tiles_x * tiles_y * M == oracle.n_slots(fr, M_REUSE, gw, gh, s)
    assert oracle.n_groups(fr, M_REUSE, gw, gh, s) * K == len(pos)
    live = pos[pos >= 0]
    # covers every path exactly once
    assert np.array_equal(np.sort(live), np.arange(spp * w * h))
    # every slot block holds exactly the pixels of its tile and sample plane
    slot = np.nonzero(pos >= 0)[0]
    tile_of_slot = (slot // M) % (tiles_x * tiles_y)
    samp_of_slot = slot // (M * tiles_x * tiles_y)
    x = live % w; y = (live // w) % h; sg = live // (w * h)
    assert np.array_equal(tile_of_slot, (y // H) * tiles_x + (x // W))
    assert np.array_equal(samp_of_slot, sg)
    # full tiles: the map n -> m is an affine bijection m = a*n + c mod M with a odd
    blk = pos[:M]
    if w >= W and h >= H:
        assert np.all(blk >= 0)
        n_of_m = (blk // w) * W + (blk % w)           # tile 0, sample 0: y*W + x
        m_of_n = np.empty(M, np.int64); m_of_n[n_of_m] = np.arange(M)
        c = m_of_n[0]
        a = (m_of_n[1] - c) % M if M > 1 else 1
        assert a % 2 == 1
        assert np.array_equal(m_of_n, (a * np.arange(M) + c) % M)
        # groups: K members each, quotient rule
        assert np.all(np.bincount(m_of_n // K, minlength=M // K) == K)


LATTICE = 1 << 14       # partition rule bit in the packed stride (D:R20)


@pytest.mark.parametrize("gw,gh,sx,sy", [(4, 4, 2, 2), (4, 4, 4, 4), (2, 2, 8, 8), (8, 8, 1, 1), (8, 1, 1, 8), (4, 2, 2, 4)])
@pytest.mark.parametrize("w,h,spp", [(64, 64, 1), (50, 37, 2)])
def test_lattice_partition_is_an_interleaved_exact_cover(oracle, gw, gh, sx, sy, w, h, spp):
    """Alternative partition rule (D:R20; S:8c A-3): a regular lattice.  Exact cover as for the shuffled rule; inside a full tile
    the members of a group are the pixels congruent modulo (sx, sy) after the tile's cyclic shift — gw x gh pixels lying sx
    apart horizontally and sy apart vertically (cyclically) — and member order inside the group is row-major over that grid;
    the shift differs between tiles and frames; stride 1 makes the whole tile one group."""
    s = sx | (sy << 16) | LATTICE
    fr = oracle.frame(w, h, spp, seed=3, frame=5)
    pos = oracle.partition(fr, M_REUSE, gw, gh, s)
    W, H = gw * sx, gh * sy
    M, K = W * H, gw * gh
    tiles_x, tiles_y = -(-w // W), -(-h // H)
    assert len(pos) == spp * tiles_x * tiles_y * M == oracle.n_slots(fr, M_REUSE, gw, gh, s)
    live = pos[pos >= 0]
    assert np.array_equal(np.sort(live), np.arange(spp * w * h))
    slot = np.nonzero(pos >= 0)[0]
    x = live % w; y = (live // w) % h
    assert np.array_equal((slot // M) % (tiles_x * tiles_y), (y // H) * tiles_x + (x // W))
    if w >= W and h >= H:
        blk = pos[:M].reshape(M // K, K)               # tile 0: groups x members
        lx, ly = blk % w, blk // w
        for g in range(M // K):
            # all members congruent modulo the strides, up to the tile's cyclic shift
            dx = (lx[g] - lx[g][0]) % W; dy = (ly[g] - ly[g][0]) % H
            assert np.all(dx % sx == 0) and np.all(dy % sy == 0)
            assert len(set(zip(dx.tolist(), dy.tolist()))) == K
        # different groups are different residue classes: the first members of the G groups are pairwise incongruent
        firsts = {(int(lx[g][0]) % sx, int(ly[g][0]) % sy) for g in range(M // K)}
        assert len(firsts) == M // K == sx * sy
        # member order inside a group is row-major over its gw x gh grid (after the shift): consecutive members step by sx
        if gw > 1:
            assert np.all((lx[:, 1] - lx[:, 0]) % W == sx) and np.all(ly[:, 1] == ly[:, 0])
    if sx == 1 and sy == 1:
        assert oracle.n_groups(fr, M_REUSE, gw, gh, s) == spp * tiles_x * tiles_y


def test_lattice_partition_shift_varies_per_tile_and_frame(oracle):
    s = 2 | LATTICE
    p0 = oracle.partition(oracle.frame(64, 64, 1, 0, 0), M_REUSE, 4, 4, s).reshape(-1, 64)
    p1 = oracle.partition(oracle.frame(64, 64, 1, 0, 1), M_REUSE, 4, 4, s).reshape(-1, 64)
    first = lambda p: [(int(b[0]) % 64 % 8, int(b[0]) // 64 % 8) for b in p]       # in-tile position of every tile's slot 0
    assert len(set(first(p0))) > 8 and first(p0) != first(p1)
    # against the definition, written out for one tile: slot m = g*K + j with g = (py % 2)*2 + px % 2, j = (py // 2)*4 + px // 2
    fr = oracle.frame(64, 64, 1, 0, 0)
    r = oracle.philox(9, 0, 0, 2, 0, 0)                                       # tile 9, sample 0, purpose TILE; key (seed 0, frame 0)
    ox, oy = int(r[0]) % 8, int(r[1]) % 8
    tx, ty = 9 % 8, 9 // 8
    exp = np.empty(64, np.int64)
    for ly in range(8):
        for lx in range(8):
            px, py = (lx + ox) % 8, (ly + oy) % 8
            exp[((py % 2) * 2 + px % 2) * 16 + (py // 2) * 4 + px // 2] = (ty * 8 + ly) * 64 + tx * 8 + lx
    assert np.array_equal(p0[9], exp)


def test_partition_varies_per_tile_and_frame_not_per_bounce(oracle):
    fr0 = oracle.frame(64, 64, 1, 0, 0); fr1 = oracle.frame(64, 64, 1, 0, 1); fs = oracle.frame(64, 64, 1, 1, 0)
    p0 = oracle.partition(fr0, M_REUSE, 4, 4, 2).reshape(-1, 64)
    p1 = oracle.partition(fr1, M_REUSE, 4, 4, 2).reshape(-1, 64)
    ps = oracle.partition(fs, M_REUSE, 4, 4, 2).reshape(-1, 64)
    assert not np.array_equal(p0, p1) and not np.array_equal(p0, ps)
    # within a frame, different tiles use different shuffles (compare local pixel numbering)
    loc = lambda p: ((p // 64) % 8) * 8 + (p % 64) % 8
    assert len({tuple(loc(row)) for row in p0}) > 32
    assert np.array_equal(p0, oracle.partition(fr0, M_REUSE, 4, 4, 2).reshape(-1, 64))     # deterministic


def test_stride_one_is_one_group_per_tile_and_other_modes_are_row_major(oracle):
    fr = oracle.frame(32, 32, 1, 0, 0)
    assert oracle.n_groups(fr, M_REUSE, 4, 4, 1) == 64
    assert np.array_equal(oracle.partition(fr, M_IND), np.arange(1024))
    assert np.array_equal(oracle.partition(fr, M_MOR), np.arange(1024))


# ------------------------------------------------------------------ helpers
def _first_bounce(oracle, scene, mode, gw=4, gh=4, s=2, frame=0, spp=1, seed=0, fp64=False):
    fr = oracle.frame(scene.width, scene.height, spp, seed, frame)
    b = oracle.Bvh(scene.verts)
    rays, hits, r2p = oracle.trace_primary(b, scene.camera, fr, mode, gw, gh, s)
    paths = oracle.paths_init(spp * scene.width * scene.height)
    accum = np.zeros((scene.height, scene.width, 3), np.float32)
    oracle.shade_accumulate(scene, fr, 0, False, rays, hits, r2p, paths, accum)
    out = oracle.generate_secondary(scene, fr, 1, mode, gw, gh, s, b.info()["bounds"], rays, hits, r2p, paths, fp64=fp64)
    out.update(prev_rays=rays, prev_hits=hits, prev_r2p=r2p, paths=paths, fr=fr, bvh=b)
    return out


def _normals(scene, prims, d_prev):
    tri = scene.verts[prims].astype(np.float64)
    n = np.cross(tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0])
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    flip = (n * d_prev).sum(1) > 0
    n[flip] *= -1
    return n


# ------------------------------------------------------------------ classification
def test_classification_constructed_scenes(oracle):
    g = _first_bounce(oracle, I.cornell(), M_REUSE)
    cls = g["group_class"]
    assert set(np.unique(cls)) <= {oracle.CLASS_EMPTY, oracle.CLASS_DIFFUSE} and (cls == oracle.CLASS_DIFFUSE).mean() > 0.5
    g = _first_bounce(oracle, I.floor_plane(I.MAT_SPECULAR), M_REUSE)
    assert np.all(g["group_class"] == oracle.CLASS_GLOSSY)
    g = _first_bounce(oracle, I.floor_plane(I.MAT_GLOSSY), M_REUSE)
    assert np.all(g["group_class"] == oracle.CLASS_GLOSSY)
    sc = I.checker_floor()
    g = _first_bounce(oracle, sc, M_REUSE)
    assert (g["group_class"] == oracle.CLASS_HYBRID).mean() > 0.9
    # recount from scratch: material type of the primary hit of every member
    K = 16
    p = g["ray_to_path"].reshape(-1, K)
    prim_of_path = np.full(sc.width * sc.height, -1); prim_of_path[g["prev_r2p"][g["prev_r2p"] >= 0]] = g["prev_hits"]["prim"][g["prev_r2p"] >= 0]
    mt = np.where(prim_of_path >= 0, sc.materials["type"][sc.mat_id[np.maximum(prim_of_path, 0)]], -1)
    mt_slot = np.where(p >= 0, mt[np.maximum(p, 0)], -1)
    nd = (mt_slot == 0).sum(1); ngl = ((mt_slot == 1) | (mt_slot == 2)).sum(1)
    exp = np.where(nd + ngl == 0, 0, np.where(ngl == 0, 1, np.where(nd == 0, 2, 3)))
    assert np.array_equal(g["group_class"], exp)


# ------------------------------------------------------------------ reuse rules
@pytest.mark.parametrize("s", [2, 2 | (1 << 14)])          # shuffled rule, lattice rule (D:R20)
def test_diffuse_group_shares_one_tangent_space_direction(oracle, s):
    sc = I.cornell()
    g = _first_bounce(oracle, sc, M_REUSE, s=s)
    gi = _first_bounce(oracle, sc, M_IND)
    K = 16
    loc = g["local_dir"].reshape(-1, K, 3); src = g["dir_src"].reshape(-1, K); p = g["ray_to_path"].reshape(-1, K)
    act = g["rays"]["tmax"].reshape(-1, K) >= 0
    n_checked = 0
    for gidx in np.nonzero(g["group_class"] == oracle.CLASS_DIFFUSE)[0]:
        a = act[gidx]
        assert a.any()
        d = loc[gidx][a]
        assert np.all(d == d[0])                                   # bit-identical local direction
        leader = src[gidx][a]
        assert np.all(leader == leader[0]) and leader[0] in p[gidx][a]        # one leader, a live member
        # the leader's direction is the one it samples independently
        assert np.array_equal(gi["local_dir"][leader[0]], d[0])
        n_checked += 1
    assert n_checked > 100
    # leaders are spread over member slots ("randomly selects one pixel")
    lead_slot = np.array([np.nonzero(p[i] == src[i][act[i]][0])[0][0] for i in np.nonzero(g["group_class"] == 1)[0]])
    assert len(np.unique(lead_slot)) == K
    assert abs(lead_slot.mean() - (K - 1) / 2) < 1.5


def test_world_direction_identical_on_a_plane_and_upper_hemisphere_everywhere(oracle):
    g = _first_bounce(oracle, I.floor_plane(I.MAT_DIFFUSE), M_REUSE)
    act = g["rays"]["tmax"] >= 0
    d = g["rays"]["d"].reshape(-1, 16, 3); a = act.reshape(-1, 16)
    for i in range(len(d)):
        if a[i].any():
            assert np.all(d[i][a[i]] == d[i][a[i]][0])             # parallel planes -> same world direction
    for sc in (I.cornell(), I.checker_floor(), I.interior(n_boxes=40, n_spheres=10, subdiv=2, width=48, height=32)):
        for mode in (M_IND, M_REUSE):
            g = _first_bounce(oracle, sc, mode)
            act = g["rays"]["tmax"] >= 0
            prev_slot_of_path = np.empty(sc.width * sc.height, np.int64)
            ok = g["prev_r2p"] >= 0
            prev_slot_of_path[g["prev_r2p"][ok]] = np.nonzero(ok)[0]
            ps = prev_slot_of_path[g["ray_to_path"][act]]
            n = _normals(sc, g["prev_hits"]["prim"][ps], g["prev_rays"]["d"][ps].astype(np.float64))
            cosw = (g["rays"]["d"][act].astype(np.float64) * n).sum(1)
            assert np.all(cosw > 0)                                 # never the lower hemisphere
            assert np.all(g["local_dir"][act][:, 2] > 0)
            assert np.allclose(np.linalg.norm(g["rays"]["d"][act].astype(np.float64), axis=1), 1, atol=2e-6)
            # local z equals the cosine with the face-forwarded geometric normal
            assert np.allclose(cosw, g["local_dir"][act][:, 2], atol=3e-6)
            assert g["n_active"] == act.sum()


def test_hybrid_group_diffuse_members_take_mean_glossy_direction(oracle):
    sc = I.checker_floor()
    g = _first_bounce(oracle, sc, M_REUSE)
    gi = _first_bounce(oracle, sc, M_IND)
    K = 16
    loc = g["local_dir"].astype(np.float64).reshape(-1, K, 3); src = g["dir_src"].reshape(-1, K)
    p = g["ray_to_path"].reshape(-1, K); act = g["rays"]["tmax"].reshape(-1, K) >= 0
    n = 0
    for gidx in np.nonzero(g["group_class"] == oracle.CLASS_HYBRID)[0]:
        own = act[gidx] & (src[gidx] == p[gidx])                   # glossy / specular members: own sample
        shared = act[gidx] & (src[gidx] == -2 - gidx)
        if not shared.any() or not own.any():
            continue
        # glossy members are untouched: same direction as independent sampling
        assert np.array_equal(g["local_dir"].reshape(-1, K, 3)[gidx][own], gi["local_dir"][p[gidx][own]])
        mean = loc[gidx][own].sum(0); mean /= np.linalg.norm(mean)
        assert np.allclose(loc[gidx][shared], mean, atol=1e-6)
        n += 1
    assert n > 30
    # weight of a diffuse member is its own albedo whatever the direction (own material's pdf)
    ok = g["prev_r2p"] >= 0
    prim_of_path = np.full(sc.width * sc.height, -1); prim_of_path[g["prev_r2p"][ok]] = g["prev_hits"]["prim"][ok]
    act1 = g["rays"]["tmax"] >= 0
    pp = g["ray_to_path"][act1]
    mats = sc.materials[sc.mat_id[prim_of_path[pp]]]
    dm = mats["type"] == I.MAT_DIFFUSE
    assert np.array_equal(g["paths"]["T"][pp][dm], mats["albedo"][dm])
    sm = mats["type"] == I.MAT_SPECULAR
    assert np.array_equal(g["paths"]["T"][pp][sm], mats["albedo"][sm])
    gm = mats["type"] == I.MAT_GLOSSY
    assert np.all(g["paths"]["T"][pp][gm] <= 1.0) and np.all(g["paths"]["T"][pp][gm] > 0)


def test_all_glossy_scene_reuse_equals_independent_ray_set(oracle):
    sc = I.floor_plane(I.MAT_GLOSSY, roughness=0.3)
    g = _first_bounce(oracle, sc, M_REUSE); gi = _first_bounce(oracle, sc, M_IND)
    a = g["rays"]["tmax"] >= 0
    by_path = np.zeros(sc.width * sc.height, oracle.RAY_DTYPE); by_path["tmax"] = -1
    by_path[g["ray_to_path"][a]] = g["rays"][a]
    assert np.array_equal(by_path, gi["rays"])
    assert np.array_equal(g["paths"], gi["paths"])


def test_group_of_one_equals_independent(oracle):
    sc = I.cornell()
    g = _first_bounce(oracle, sc, M_REUSE, gw=1, gh=1, s=4); gi = _first_bounce(oracle, sc, M_IND)
    a = g["ray_to_path"] >= 0
    by_path = np.zeros(sc.width * sc.height, oracle.RAY_DTYPE)
    by_path[g["ray_to_path"][a]] = g["rays"][a]
    assert np.array_equal(by_path, gi["rays"])


def test_specular_rule_is_mirror_reflection(oracle):
    sc = I.floor_plane(I.MAT_SPECULAR, albedo=0.6)
    g = _first_bounce(oracle, sc, M_IND)
    a = g["rays"]["tmax"] >= 0
    din = g["prev_rays"]["d"][a].astype(np.float64)
    exp = din * np.array([1, -1, 1])
    assert np.allclose(g["rays"]["d"][a], exp, atol=3e-7)
    # origin sits on the floor, lifted along +y by the self-intersection offset
    o = g["rays"]["o"][a]
    assert np.all(o[:, 1] > 0) and np.all(o[:, 1] < 1e-2)


# ------------------------------------------------------------------ sampling distributions
def test_cosine_sampling_moments_and_chi_square(oracle):
    n = 256
    u = (np.arange(n) + 0.5) / n
    w = np.array([oracle.sample_cosine(float(a), float(b)) for a in u for b in u])
    assert np.allclose(np.linalg.norm(w, axis=1), 1, atol=1e-6)
    assert abs(w[:, 2].mean() - 2 / 3) < 1e-4                       # E[cos] = 2/3 for pdf cos/pi
    assert abs((w[:, 2] ** 2).mean() - 0.5) < 1e-4                  # E[cos^2] = 1/2
    assert abs(w[:, 0].mean()) < 1e-4 and abs(w[:, 1].mean()) < 1e-4
    # chi-square on a (cos^2 theta, phi) grid: cos^2 is uniform under the cosine pdf
    hist, _, _ = np.histogram2d(w[:, 2] ** 2, np.arctan2(w[:, 1], w[:, 0]), bins=(8, 16), range=((0, 1), (-math.pi, math.pi)))
    e = len(w) / hist.size
    assert ((hist - e) ** 2 / e).sum() < 250


def _ggx_vndf_pdf_h(wo, alpha, h):
    """Textbook density of visible normals: G1(wo) max(0, wo.h) D(h) / wo.z  (per solid angle of h)."""
    D = alpha**2 / (math.pi * ((h[..., 2] ** 2) * (alpha**2 - 1) + 1) ** 2)
    tan2 = (wo[0] ** 2 + wo[1] ** 2) / wo[2] ** 2
    G1 = 2 / (1 + math.sqrt(1 + alpha**2 * tan2))
    return G1 * np.maximum(0, h @ wo) * D / wo[2]


@pytest.mark.parametrize("alpha,theta", [(0.5, 0.3), (0.2, 1.0), (0.35, 1.35)])
def test_ggx_half_vectors_follow_the_visible_normal_distribution(oracle, alpha, theta):
    """Moments of the sampled half-vector against fp64 quadrature of the textbook VNDF density."""
    wo = np.array([math.sin(theta) * 0.8, math.sin(theta) * 0.6, math.cos(theta)])
    n = 192
    u = (np.arange(n) + 0.5) / n
    hs, wts = [], []
    for a in u:
        for b in u:
            ok, wi, wt = oracle.sample_ggx(wo, alpha, float(a), float(b))
            h = wo + wi.astype(np.float64)
            # reflect(wo, h) = wi  =>  h parallel to wo + wi (also when wi is below the horizon)
            hs.append(h / np.linalg.norm(h)); wts.append(wt if ok else 0.0)
            if ok:
                assert 0 < wt <= 1.0 + 1e-6 and wi[2] > 0
            assert abs(np.linalg.norm(wi) - 1) < 2e-5
    hs = np.array(hs)
    # quadrature over the hemisphere of h
    nt, nph = 2000, 720
    ct = (np.arange(nt) + 0.5) / nt                                  # cos(theta_h) uniform
    ph = (np.arange(nph) + 0.5) / nph * 2 * math.pi
    CT, PH = np.meshgrid(ct, ph, indexing="ij"); ST = np.sqrt(1 - CT**2)
    H = np.stack([ST * np.cos(PH), ST * np.sin(PH), CT], -1)
    pdf = _ggx_vndf_pdf_h(wo, alpha, H) * (2 * math.pi / (nt * nph))
    assert abs(pdf.sum() - 1) < 2e-3                                 # VNDF is normalised
    for f in (lambda h: h[..., 0], lambda h: h[..., 1], lambda h: h[..., 2], lambda h: h[..., 2] ** 2, lambda h: h[..., 0] * h[..., 1]):
        assert abs(f(hs).mean() - (f(H) * pdf).sum()) < 4e-3
    assert np.mean(wts) <= 1.0                                       # white furnace: energy never gained


# ------------------------------------------------------------------ world-space reuse (section 3.1; DESIGN.md D:R18)
def test_world_space_reuse_rules(oracle):
    """The paper's first variant: the group shares one WORLD direction.  On a plane it coincides with tangent-space reuse;
    on curved / mixed geometry the shared direction is bit-identical across the reusing members, equals the selected
    pixel's own (independent) ray, never leaves a member's upper hemisphere (such members end), and mirrors are untouched."""
    flat_t = _first_bounce(oracle, I.floor_plane(I.MAT_DIFFUSE), M_REUSE)
    flat_w = _first_bounce(oracle, I.floor_plane(I.MAT_DIFFUSE), M_WORLD)
    assert flat_w["rays"].tobytes() == flat_t["rays"].tobytes() and np.array_equal(flat_w["dir_src"], flat_t["dir_src"])
    n_dead_total = 0
    for sc in (I.cornell(), I.interior(n_boxes=40, n_spheres=10, subdiv=2, width=48, height=32), I.checker_floor()):
        g = _first_bounce(oracle, sc, M_WORLD); gi = _first_bounce(oracle, sc, M_IND); gt = _first_bounce(oracle, sc, M_REUSE)
        K = 16
        assert np.array_equal(g["ray_to_path"], gt["ray_to_path"]) and np.array_equal(g["group_class"], gt["group_class"])   # same partition and census
        act = g["rays"]["tmax"] >= 0
        p = g["ray_to_path"]; src = g["dir_src"]
        prev_slot_of_path = np.full(sc.width * sc.height, -1, np.int64); ok = g["prev_r2p"] >= 0
        prev_slot_of_path[g["prev_r2p"][ok]] = np.nonzero(ok)[0]
        ps = prev_slot_of_path[np.maximum(p, 0)]
        mtype = np.where(p >= 0, sc.materials["type"][sc.mat_id[np.maximum(g["prev_hits"]["prim"][ps], 0)]], -1)
        # upper hemisphere for every emitted ray
        n = _normals(sc, g["prev_hits"]["prim"][ps[act]], g["prev_rays"]["d"][ps[act]].astype(np.float64))
        assert np.all((g["rays"]["d"][act].astype(np.float64) * n).sum(1) > 0)
        reuse = act & (src != p)
        assert reuse.sum() > 100
        # a reusing member's direction is bit-identical to its leader's independent-mode ray direction
        assert np.array_equal(g["rays"]["d"][reuse], gi["rays"]["d"][src[reuse]])
        assert np.all(mtype[reuse] != I.MAT_SPECULAR)
        # own-sampling members (leaders, mirrors): exactly their independent ray
        own = act & (src == p)
        assert np.array_equal(g["rays"][own], gi["rays"][p[own]])
        spec = act & (mtype == I.MAT_SPECULAR)
        assert np.all(src[spec] == p[spec])
        # one leader per group among the reusing members
        for gidx in np.unique(np.nonzero(reuse)[0] // K)[:200]:
            sl = slice(gidx * K, (gidx + 1) * K)
            leaders = np.unique(src[sl][reuse[sl]])
            assert len(leaders) == 1 and leaders[0] in p[sl]
        # paths that were alive with a hit but emitted no ray: ended because the shared direction was below their horizon
        alive_before = (g["prev_hits"]["prim"][ps] >= 0) & (p >= 0)
        n_dead_total += int((alive_before & ~act).sum()) - int(((gi["rays"]["tmax"] < 0)[np.maximum(p, 0)] & alive_before).sum())
    assert n_dead_total > 50            # the artifact of Fig. 1 exists on non-planar scenes ...
    assert flat_w["n_active"] == flat_t["n_active"]          # ... and not on a plane


def test_world_space_reuse_is_biased_on_curved_geometry_but_exact_on_a_plane(oracle):
    """Furnace: white Lambert under uniform light.  On a floor every direction is valid for every member -> exactly 1;
    on a sphere members whose normal faces away from the shared direction end -> darker than 1."""
    def image(sc, mode):
        fr = oracle.frame(sc.width, sc.height, 1, 0, 0)
        acc, _, _ = oracle.render_frame(oracle.Bvh(sc.verts), sc, fr, 1, mode, 4, 4, 8)      # tile 32x32: members all over the sphere
        return acc
    floor = I.floor_plane(I.MAT_DIFFUSE, albedo=1.0)
    assert np.all(image(floor, M_WORLD) == 1.0)
    sph = I.furnace_sphere()
    hit = image(sph, M_REUSE)
    assert np.all(hit == 1.0)
    w = image(sph, M_WORLD)
    assert w.max() == 1.0 and 0.5 < w.mean() < 0.99 and set(np.unique(w)) == {0.0, 1.0}


# ------------------------------------------------------------------ Morton code + sort
def _spread6(v):
    """table-driven spread of a 5-bit value to every 6th bit (the oracle uses a bit-by-bit loop)"""
    lut = np.array([sum(((i >> l) & 1) << (6 * l) for l in range(5)) for i in range(32)], np.uint64)
    return lut[v]


def test_morton_code_and_sort(oracle):
    sc = I.cornell()
    bounds = np.array([0, 0, 0, 1, 1, 1], np.float32)
    rays = I.random_rays(4, 5000, [0, 0, 0], [1, 1, 1], inactive_frac=0.1).view(oracle.RAY_DTYPE).reshape(-1)
    rays["o"] = np.clip(rays["o"], -0.05, 1.05)
    keys = oracle.morton_encode(rays, bounds)
    act = rays["tmax"] >= 0
    assert np.all(keys[~act] == 0xFFFFFFFF) and np.all(keys[act] < 2**30)
    qo = np.clip(np.floor(rays["o"].astype(np.float64) * 32), 0, 31).astype(np.int64)
    qd = np.clip(np.floor((rays["d"].astype(np.float64) + 1) * 16), 0, 31).astype(np.int64)
    exp = (_spread6(qo[:, 0]) << 5) | (_spread6(qo[:, 1]) << 4) | (_spread6(qo[:, 2]) << 3) | \
          (_spread6(qd[:, 0]) << 2) | (_spread6(qd[:, 1]) << 1) | _spread6(qd[:, 2])
    # fp32 quantisation may differ from fp64 only when a coordinate sits within an ulp of a cell edge
    assert (keys[act] == exp[act]).mean() > 0.999
    order = oracle.sort_keys(keys)
    assert np.array_equal(order, np.argsort(keys, kind="stable"))
    assert np.array_equal(np.sort(order), np.arange(len(keys)))      # permutation
    k = keys[order]
    assert np.all(k[1:] >= k[:-1])
    eq = k[1:] == k[:-1]
    assert np.all(order[1:][eq] > order[:-1][eq])                    # equal keys keep input order


def test_morton_golden(oracle):
    """Hand-derived codes (tests/golden/morton_codes.txt): quantised cells and bit patterns written out per level."""
    import os
    rows = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "morton_codes.txt")) if not l.startswith("#")]
    assert len(rows) >= 6
    rays = np.zeros(len(rows), oracle.RAY_DTYPE)
    exp = []
    for i, l in enumerate(rows):
        vals, q, levels, code = [p.strip() for p in l.split("|")]
        v = [float(x) for x in vals.split()]
        rays["o"][i] = v[:3]; rays["d"][i] = v[3:]; rays["tmax"][i] = 1e30
        bits = "".join(levels.split())
        assert len(bits) == 30 and int(bits, 2) == int(code, 16)          # the fixture is self-consistent
        qs = [int(x) for x in q.split()]
        assert bits == "".join(str((qs[k] >> lv) & 1) for lv in (4, 3, 2, 1, 0) for k in range(6))
        exp.append(int(code, 16))
    keys = oracle.morton_encode(rays, np.array([0, 0, 0, 1, 1, 1], np.float32))
    assert [int(k) for k in keys] == exp


def test_morton_mode_is_a_sorted_permutation_of_independent_rays(oracle):
    sc = I.interior(n_boxes=40, n_spheres=10, subdiv=2, width=48, height=32)
    gm = _first_bounce(oracle, sc, M_MOR); gi = _first_bounce(oracle, sc, M_IND)
    perm = gm["ray_to_path"]
    assert np.array_equal(np.sort(perm), np.arange(sc.width * sc.height))
    assert np.array_equal(gm["rays"], gi["rays"][perm])
    assert np.array_equal(gm["dir_src"], gi["dir_src"][perm])
    keys = oracle.morton_encode(gm["rays"], gm["bvh"].info()["bounds"])
    assert np.all(keys[1:] >= keys[:-1])
    assert gm["n_active"] == (keys != 0xFFFFFFFF).sum() == gi["n_active"]
    assert np.array_equal(gm["paths"], gi["paths"])


# ------------------------------------------------------------------ further reordering keys (D:R19)
def _m3(a, b, c, bits):
    """3D Morton code by table lookup per byte-free shifts (the oracle loops over bits)"""
    out = np.zeros(len(a), np.int64)
    for l in range(bits):
        out |= (((a >> l) & 1) << (3 * l + 2)) | (((b >> l) & 1) << (3 * l + 1)) | (((c >> l) & 1) << (3 * l))
    return out


def test_ray_codes_against_definitions_and_relations(oracle):
    """Origin / Reis / Costa / TwoPoint keys: an independent numpy encoder, and the relations the definitions imply:
    Reis and Costa hold the same two 15-bit halves swapped; the top 5 levels of Origin are the origin half of Reis;
    TwoPoint is AilaCompact's layout with the clamped end point o + 0.25*maxext*d in place of the direction, so a ray
    of zero length direction (end = origin) repeats every origin bit."""
    bounds = np.array([-1, 0, 2, 3, 1, 10], np.float32)              # extents 4, 1, 8: largest 8 -> length 2
    lo, ext = bounds[:3].astype(np.float64), (bounds[3:] - bounds[:3]).astype(np.float64)
    rays = I.random_rays(9, 4000, bounds[:3], bounds[3:], inactive_frac=0.1).view(oracle.RAY_DTYPE).reshape(-1)
    act = rays["tmax"] >= 0
    o, d = rays["o"].astype(np.float64), rays["d"].astype(np.float64)
    q5 = np.clip(np.floor((o - lo) * (32 / ext)), 0, 31).astype(np.int64)
    q10 = np.clip(np.floor((o - lo) * (1024 / ext)), 0, 1023).astype(np.int64)
    qd = np.clip(np.floor((d + 1) * 16), 0, 31).astype(np.int64)
    qe = np.clip(np.floor((o + 0.25 * ext.max() * d - lo) * (32 / ext)), 0, 31).astype(np.int64)
    k = {n: oracle.ray_code_encode(c, rays, bounds).astype(np.int64) for n, c in oracle.RAY_CODES.items()}
    for n in k:
        assert np.all(k[n][~act] == 0xFFFFFFFF) and np.all(k[n][act] < 2**30)
    assert np.array_equal(k["aila_compact"], oracle.morton_encode(rays, bounds))
    mo, md = _m3(q5[:, 0], q5[:, 1], q5[:, 2], 5), _m3(qd[:, 0], qd[:, 1], qd[:, 2], 5)
    exp = {"origin": _m3(q10[:, 0], q10[:, 1], q10[:, 2], 10), "reis": (mo << 15) | md, "costa": (md << 15) | mo,
           "twopoint": (_spread6(q5[:, 0]) << 5) | (_spread6(q5[:, 1]) << 4) | (_spread6(q5[:, 2]) << 3)
                       | (_spread6(qe[:, 0]) << 2) | (_spread6(qe[:, 1]) << 1) | _spread6(qe[:, 2])}
    for n, e in exp.items():      # fp32 quantisation differs from fp64 only within an ulp of a cell edge
        assert (k[n][act] == np.asarray(e, np.int64)[act]).mean() > 0.998, n
    a = act
    assert np.array_equal(k["reis"][a] >> 15, k["costa"][a] & 0x7FFF) and np.array_equal(k["reis"][a] & 0x7FFF, k["costa"][a] >> 15)
    assert np.array_equal(k["origin"][a] >> 15, k["reis"][a] >> 15)
    # origin bits of TwoPoint and AilaCompact sit at the same positions
    omask = sum(0b111000 << (6 * l) for l in range(5))
    assert np.array_equal(k["twopoint"][a] & omask, k["aila_compact"][a] & omask)
    z = rays.copy(); z["d"] = 0
    kz = oracle.ray_code_encode(4, z, bounds).astype(np.int64)[a]
    assert np.array_equal((kz & omask) >> 3, kz & (omask >> 3))


def test_ray_codes_golden(oracle):
    """Hand-derived keys (tests/golden/ray_codes.txt)."""
    import os
    rows = [l for l in open(os.path.join(os.path.dirname(__file__), "golden", "ray_codes.txt")) if not l.startswith("#") and l.strip()]
    assert len(rows) >= 8
    for l in rows:
        name, vals, bits, code = [p.strip() for p in l.split("|")]
        v = [float(x) for x in vals.split()]
        r = np.zeros(1, oracle.RAY_DTYPE); r["o"][0] = v[:3]; r["d"][0] = v[3:]; r["tmax"][0] = 1e30
        b = "".join(bits.split())
        assert len(b) == 30 and int(b, 2) == int(code, 16)                     # the fixture is self-consistent
        got = int(oracle.ray_code_encode(oracle.RAY_CODES[name], r, np.array([0, 0, 0, 1, 1, 1], np.float32))[0])
        assert got == int(code, 16), (name, l)


@pytest.mark.parametrize("mode_name,code", [("sort_origin", 1), ("sort_reis", 2), ("sort_costa", 3), ("sort_twopoint", 4)])
def test_sort_modes_are_sorted_permutations_of_independent_rays(oracle, mode_name, code):
    sc = I.interior(n_boxes=40, n_spheres=10, subdiv=2, width=48, height=32)
    gm = _first_bounce(oracle, sc, oracle.MODES[mode_name]); gi = _first_bounce(oracle, sc, M_IND)
    perm = gm["ray_to_path"]
    assert np.array_equal(np.sort(perm), np.arange(sc.width * sc.height))
    assert np.array_equal(gm["rays"], gi["rays"][perm])
    keys_by_path = oracle.ray_code_encode(code, gi["rays"], gm["bvh"].info()["bounds"])
    assert np.array_equal(perm, np.argsort(keys_by_path, kind="stable"))       # stable ascending sort of the mode's own key
    assert gm["n_active"] == gi["n_active"] and np.array_equal(gm["paths"], gi["paths"])


# ------------------------------------------------------------------ shading / accumulation
@pytest.mark.parametrize("mode", [M_IND, M_MOR, M_REUSE])
@pytest.mark.parametrize("mat", [I.MAT_DIFFUSE, I.MAT_SPECULAR])
def test_white_furnace_is_exactly_one(oracle, mode, mat):
    """Convex white sphere under uniform radiance 1: every pixel is exactly 1 (north_star's furnace test)."""
    sc = I.furnace_sphere(2, albedo=1.0, mat_type=mat)
    b = oracle.Bvh(sc.verts)
    for nb in (1, 3):
        img, _, cnt = oracle.render_frame(b, sc, oracle.frame(sc.width, sc.height, 2, 0, 1), nb, mode, 4, 4, 2)
        assert np.all(img == 1.0)
        assert cnt[0] > 0


def test_white_furnace_is_exactly_one_with_the_lattice_partition(oracle):
    sc = I.furnace_sphere(2, albedo=1.0, mat_type=I.MAT_DIFFUSE)
    b = oracle.Bvh(sc.verts)
    img, _, cnt = oracle.render_frame(b, sc, oracle.frame(sc.width, sc.height, 2, 0, 1), 2, M_REUSE, 4, 4, 2 | (1 << 14))
    assert np.all(img == 1.0) and cnt[0] > 0


@pytest.mark.parametrize("mode", [M_IND, M_REUSE])
def test_albedo_furnace_closed_form(oracle, mode):
    """Convex sphere of albedo rho: pixel = rho where the primary ray hits, 1 where it misses."""
    rho = np.float32(0.37)
    sc = I.furnace_sphere(2, albedo=rho)
    b = oracle.Bvh(sc.verts)
    fr = oracle.frame(sc.width, sc.height, 1, 0, 0)
    img, _, _ = oracle.render_frame(b, sc, fr, 2, mode, 4, 4, 2)
    _, hits, r2p = oracle.trace_primary(b, sc.camera, fr, M_IND)
    hit = (hits["prim"] >= 0).reshape(sc.height, sc.width)
    assert np.all(img[hit] == rho) and np.all(img[~hit] == 1.0) and 0.1 < hit.mean() < 0.9


def test_mirror_floor_under_sky_closed_form(oracle):
    """Mirror floor, env = vertical gradient: pixel = albedo * env(reflect(d))."""
    sc = I.floor_plane(I.MAT_SPECULAR, albedo=0.6)
    sc.env[:] = (1, 1, 1, 0.2, 0.4, 1.0)
    b = oracle.Bvh(sc.verts)
    fr = oracle.frame(sc.width, sc.height, 1, 0, 0)
    img, _, _ = oracle.render_frame(b, sc, fr, 1, M_REUSE, 4, 4, 2)
    rays, hits, _ = oracle.trace_primary(b, sc.camera, fr, M_IND)
    assert np.all(hits["prim"] >= 0)
    dy = -rays["d"][:, 1].astype(np.float64)
    wgt = 0.5 * (dy + 1)
    exp = 0.6 * (sc.env[:3][None] + (sc.env[3:] - sc.env[:3])[None] * wgt[:, None])
    assert np.allclose(img.reshape(-1, 3), exp, atol=2e-6)


def test_emission_and_accumulation_over_frames_and_spp(oracle):
    sc = I.cornell(width=32, height=32)
    b = oracle.Bvh(sc.verts)
    acc = np.zeros((32, 32, 3), np.float32)
    n_frames = 24
    for f in range(n_frames):
        oracle.render_frame(b, sc, oracle.frame(32, 32, 2, 0, f), 1, M_REUSE, 4, 4, 2, accum=acc)
    img_r = acc / n_frames
    acc = np.zeros((32, 32, 3), np.float32)
    for f in range(n_frames):
        oracle.render_frame(b, sc, oracle.frame(32, 32, 2, 0, f), 1, M_IND, accum=acc)
    img_i = acc / n_frames
    # pixels that see the light directly are Le = 15 in both
    assert (img_r.max() == 15.0) and (img_i.max() == 15.0)
    # all-diffuse scene: reuse is unbiased -- image means agree within Monte-Carlo noise
    m_r, m_i = img_r[img_r < 15].mean(), img_i[img_i < 15].mean()
    assert abs(m_r - m_i) / m_i < 0.15
    assert 0.02 < m_i < 2.0


def test_unbiasedness_rmse_shrinks_with_frames(oracle):
    """floor under a sky gradient with a diffuse floor: E[pixel] = albedo * E_cos[env]; reuse and independent agree
    and their RMSE falls roughly like 1/sqrt(frames)."""
    sc = I.floor_plane(I.MAT_DIFFUSE, albedo=0.5, width=16, height=16)
    sc.env[:] = (0, 0, 0, 2, 2, 2)                      # L(d) = (d.y + 1): E over cosine lobe about +y = 1 + 2/3
    b = oracle.Bvh(sc.verts)
    exact = 0.5 * (1 + 2 / 3)
    err = {}
    for mode in (M_IND, M_REUSE):
        acc = np.zeros((16, 16, 3), np.float32)
        for f in range(64):
            oracle.render_frame(b, sc, oracle.frame(16, 16, 1, 0, f), 1, mode, 4, 4, 2, accum=acc)
            if f + 1 in (4, 64):
                err[(mode, f + 1)] = math.sqrt(((acc / (f + 1) - exact) ** 2).mean())
    for mode in (M_IND, M_REUSE):
        assert err[(mode, 64)] < 0.45 * err[(mode, 4)]
        assert err[(mode, 64)] < 0.05


# ------------------------------------------------------------------ third partition rule: LCG sequence (S:8c A-1; D:R21)
SEQUENCE = 1 << 15      # partition rule bit in the packed stride


@pytest.mark.parametrize("gw,gh,s", [(4, 4, 2), (4, 4, 4), (2, 2, 8), (8, 8, 8), (8, 1, 1 | (8 << 16)), (1, 1, 4), (1, 1, 1), (2, 1, 1)])
@pytest.mark.parametrize("w,h,spp", [(64, 64, 1), (50, 37, 2)])
def test_lcg_sequence_partition_is_a_full_period_sequence(oracle, gw, gh, s, w, h, spp):
    """"Shuffled using a linear congruence method" read as a SEQUENCE: the shuffled number of pixel n is the n-th term of
    x_{n+1} = (A x_n + C) mod M.  Exact cover as for the other rules; inside a full tile consecutive pixel numbers satisfy the
    recurrence with ONE pair (A, C), A = 1 mod 4 and C odd (Hull-Dobell: full period for M a power of two, so the terms are a
    permutation); the terms follow from the tile's Philox TILE stream by plain iteration (brute force here)."""
    fr = oracle.frame(w, h, spp, seed=3, frame=5)
    pos = oracle.partition(fr, M_REUSE, gw, gh, s | SEQUENCE)
    W, H = gw * (s & 0x3fff), gh * ((s >> 16) or (s & 0x3fff))
    M, K = W * H, gw * gh
    tiles_x, tiles_y = -(-w // W), -(-h // H)
    assert len(pos) == spp * tiles_x * tiles_y * M == oracle.n_slots(fr, M_REUSE, gw, gh, s | SEQUENCE)
    live = pos[pos >= 0]
    assert np.array_equal(np.sort(live), np.arange(spp * w * h))                 # every path exactly once
    slot = np.nonzero(pos >= 0)[0]
    x = live % w; y = (live // w) % h
    assert np.array_equal((slot // M) % (tiles_x * tiles_y), (y // H) * tiles_x + (x // W))
    if w >= W and h >= H:
        for tile in (0, tiles_x + 1 if tiles_x > 1 and tiles_y > 1 else 0):
            blk = pos[tile * M:(tile + 1) * M]
            assert np.all(blk >= 0)
            tx, ty = tile % tiles_x, tile // tiles_x
            n_of_m = ((blk // w) - ty * H) * W + ((blk % w) - tx * W)
            m_of_n = np.empty(M, np.int64); m_of_n[n_of_m] = np.arange(M)
            # brute force from the definition: A, C, x0 from the TILE stream (counter (tile, sample 0, 0, purpose 2), key (seed, frame))
            r = oracle.philox(tile, 0, 0, 2, 3, 5)
            A, C, x0 = ((r[0] % M) & ~3) | 1, (r[1] % M) | 1, r[2] % M
            assert A % 4 == 1 and C % 2 == 1
            xs, xv = [], x0
            for _ in range(M):
                xs.append(xv); xv = (A * xv + C) % M
            assert np.array_equal(m_of_n, np.array(xs))
            assert sorted(xs) == list(range(M))                                   # full period
            assert np.all(np.bincount(m_of_n // K, minlength=M // K) == K)        # K members per group (quotient rule)


def test_lcg_sequence_differs_from_the_affine_map_and_varies(oracle):
    fr0 = oracle.frame(64, 64, 1, 0, 0); fr1 = oracle.frame(64, 64, 1, 0, 1)
    ps = oracle.partition(fr0, M_REUSE, 4, 4, 2 | SEQUENCE).reshape(-1, 64)
    pa = oracle.partition(fr0, M_REUSE, 4, 4, 2).reshape(-1, 64)
    assert not np.array_equal(ps, pa)
    assert not np.array_equal(ps, oracle.partition(fr1, M_REUSE, 4, 4, 2 | SEQUENCE).reshape(-1, 64))
    loc = lambda p: ((p // 64) % 8) * 8 + (p % 64) % 8
    assert len({tuple(loc(row)) for row in ps}) > 32                               # different tiles, different sequences
    # an affine map of n has constant second differences 0 mod M; a sequence with A != 1 does not
    n_nonaffine = 0
    for row in ps:
        m_of_n = np.empty(64, np.int64); m_of_n[loc(row)] = np.arange(64)
        d2 = (m_of_n[2:] - 2 * m_of_n[1:-1] + m_of_n[:-2]) % 64
        n_nonaffine += int(np.any(d2 != 0))
    assert n_nonaffine > len(ps) // 2


def test_lcg_sequence_rule_keeps_the_reuse_invariants_and_the_furnace(oracle):
    sc = I.cornell()
    g = _first_bounce(oracle, sc, M_REUSE, s=2 | SEQUENCE)
    gi = _first_bounce(oracle, sc, M_IND)
    K = 16
    loc = g["local_dir"].reshape(-1, K, 3); src = g["dir_src"].reshape(-1, K); act = g["rays"]["tmax"].reshape(-1, K) >= 0
    n = 0
    for gidx in np.nonzero(g["group_class"] == oracle.CLASS_DIFFUSE)[0]:
        a = act[gidx]; d = loc[gidx][a]
        assert np.all(d == d[0]) and np.array_equal(gi["local_dir"][src[gidx][a][0]], d[0])
        n += 1
    assert n > 100
    sph = I.furnace_sphere(2, albedo=1.0)
    img, _, cnt = oracle.render_frame(oracle.Bvh(sph.verts), sph, oracle.frame(sph.width, sph.height, 2, 0, 1), 2, M_REUSE, 4, 4, 2 | SEQUENCE)
    assert np.all(img == 1.0) and cnt[0] > 0
