"""Procedural scenes standing in for the paper's third-party test scenes.

The paper measures on Breakfast / Salle de Bain / Living room / Sibenik /
Vokselia; those assets are not available, so the
synthetic scenes below take their scale and character (BASELINE.json configs,
SURVEY.md §8d).  Everything is a pure function of the seed via
numpy.random.default_rng, with a fixed draw order.

A scene is: verts float32[n,3,3], mat_id int32[n], materials (structured array,
32 bytes each: albedo[3], roughness, emission[3], type), env float32[6]
(radiance on miss = lerp(env[0:3], env[3:6], 0.5*(d.y+1))), and a camera.
"""
from __future__ import annotations

import dataclasses
import numpy as np

MAT_DIFFUSE, MAT_GLOSSY, MAT_SPECULAR, MAT_EMISSIVE = 0, 1, 2, 3

MATERIAL_DTYPE = np.dtype([("albedo", "<f4", 3), ("roughness", "<f4"),
                           ("emission", "<f4", 3), ("type", "<i4")])
assert MATERIAL_DTYPE.itemsize == 32


@dataclasses.dataclass
class Scene:
    name: str
    verts: np.ndarray       # float32 [n,3,3]
    mat_id: np.ndarray      # int32 [n]
    materials: np.ndarray   # MATERIAL_DTYPE [n_mat]
    env: np.ndarray         # float32 [6]
    camera: np.ndarray      # float32 [12]: eye, U, V, W  (see make_camera)
    width: int = 64
    height: int = 64

    @property
    def n_tris(self) -> int:
        return int(self.verts.shape[0])

    def with_camera(self, width, height, eye=None, target=None, vfov_deg=None, up=(0, 1, 0)):
        cam = self.camera
        if eye is not None:
            cam = make_camera(eye, target, up, vfov_deg, width / height)
        else:
            # rescale U for the new aspect ratio, keeping V (vertical fov)
            cam = cam.copy()
            u = cam[3:6].astype(np.float64)
            v = cam[6:9].astype(np.float64)
            un = u / np.linalg.norm(u)
            cam[3:6] = (un * np.linalg.norm(v) * (width / height)).astype(np.float32)
        return dataclasses.replace(self, camera=cam, width=width, height=height)


def make_camera(eye, target, up, vfov_deg, aspect) -> np.ndarray:
    """Pinhole camera as 12 floats: eye, U, V, W.  A pixel at normalised screen
    position (sx, sy) in [-1,1]^2 (sy up) looks along W + sx*U + sy*V."""
    eye = np.asarray(eye, np.float64)
    target = np.asarray(target, np.float64)
    w = target - eye
    w /= np.linalg.norm(w)
    r = np.cross(w, np.asarray(up, np.float64))
    r /= np.linalg.norm(r)
    u = np.cross(r, w)
    th = np.tan(np.radians(vfov_deg) * 0.5)
    return np.concatenate([eye, r * th * aspect, u * th, w]).astype(np.float32)


def _materials(n):
    m = np.zeros(n, MATERIAL_DTYPE)
    m["roughness"] = 1.0
    return m


# --------------------------------------------------------------------------
# mesh helpers
# --------------------------------------------------------------------------
def _quad(p0, eu, ev, nu=4, nv=4):
    """Parallelogram p0 + a*eu + b*ev tessellated nu x nv cells, 2 tris per cell.
    Normal (right-handed) = eu x ev."""
    p0, eu, ev = (np.asarray(a, np.float64) for a in (p0, eu, ev))
    a = np.arange(nu + 1) / nu
    b = np.arange(nv + 1) / nv
    P = p0[None, None, :] + a[:, None, None] * eu[None, None, :] + b[None, :, None] * ev[None, None, :]
    p00, p10, p01, p11 = P[:-1, :-1], P[1:, :-1], P[:-1, 1:], P[1:, 1:]
    t0 = np.stack([p00, p10, p11], axis=2)
    t1 = np.stack([p00, p11, p01], axis=2)
    return np.concatenate([t0.reshape(-1, 3, 3), t1.reshape(-1, 3, 3)], axis=0)


_BOX_FACES = [  # (origin corner signs, u axis, v axis) with outward normal = u x v
    ((-1, -1, 1), 0, 1), ((1, -1, -1), (0, -1), 1),
    ((1, -1, 1), (2, -1), 1), ((-1, -1, -1), 2, 1),
    ((-1, 1, 1), 0, (2, -1)), ((-1, -1, -1), 0, 2),
]


def _unit_box(nu=4):
    """Axis-aligned box [-1,1]^3, 6 faces, each nu x nu cells x 2 tris, outward normals."""
    tris = []
    for corner, ua, va in _BOX_FACES:
        def axis(a):
            e = np.zeros(3)
            if isinstance(a, tuple):
                e[a[0]] = 2.0 * a[1]
            else:
                e[a] = 2.0
            return e
        tris.append(_quad(np.asarray(corner, np.float64), axis(ua), axis(va), nu, nu))
    return np.concatenate(tris, axis=0)


def _icosphere(subdiv):
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0], [0, -1, t], [0, 1, t],
                  [0, -1, -t], [0, 1, -t], [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11], [1, 5, 9], [5, 11, 4],
                  [11, 10, 2], [10, 7, 6], [7, 1, 8], [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8],
                  [3, 8, 9], [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]])
    tri = v[f]                                         # [20,3,3]
    for _ in range(subdiv):
        a, b, c = tri[:, 0], tri[:, 1], tri[:, 2]
        ab, bc, ca = (a + b), (b + c), (c + a)
        ab /= np.linalg.norm(ab, axis=1, keepdims=True)
        bc /= np.linalg.norm(bc, axis=1, keepdims=True)
        ca /= np.linalg.norm(ca, axis=1, keepdims=True)
        tri = np.concatenate([np.stack([a, ab, ca], 1), np.stack([b, bc, ab], 1),
                              np.stack([c, ca, bc], 1), np.stack([ab, bc, ca], 1)], axis=0)
    return tri


def _rot_y(deg):
    c, s = np.cos(np.radians(deg)), np.sin(np.radians(deg))
    return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]])


def _quat_to_mat(q):
    """q: [n,4] (x,y,z,w) unit -> [n,3,3]."""
    x, y, z, w = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    return np.stack([
        np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)], -1),
        np.stack([2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)], -1),
        np.stack([2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)], -1)], 1)


def _random_rotations(rng, n):
    u = rng.random((n, 3))
    q = np.stack([np.sqrt(1 - u[:, 0]) * np.sin(2 * np.pi * u[:, 1]),
                  np.sqrt(1 - u[:, 0]) * np.cos(2 * np.pi * u[:, 1]),
                  np.sqrt(u[:, 0]) * np.sin(2 * np.pi * u[:, 2]),
                  np.sqrt(u[:, 0]) * np.cos(2 * np.pi * u[:, 2])], -1)
    return _quat_to_mat(q)


# --------------------------------------------------------------------------
# config 1: tiny Cornell box
# --------------------------------------------------------------------------
def cornell(seed=0, width=64, height=64, tess=4) -> Scene:
    """Unit box [0,1]^3 open toward +z, two boxes, one emissive quad under the
    ceiling.  18 quads x (tess*tess*2) tris = 576 triangles at tess=4
    (BASELINE.json config 1 says "about 1k"; order of magnitude only)."""
    rng = np.random.default_rng(seed)
    quads = [  # inward-facing
        ((0, 0, 0), (0, 0, 1), (1, 0, 0)),   # floor, normal +y
        ((0, 1, 0), (1, 0, 0), (0, 0, 1)),   # ceiling, normal -y
        ((0, 0, 0), (1, 0, 0), (0, 1, 0)),   # back, normal +z
        ((0, 0, 0), (0, 1, 0), (0, 0, 1)),   # left, normal +x
        ((1, 0, 0), (0, 0, 1), (0, 1, 0)),   # right, normal -x
    ]
    tris, mids = [], []
    mats = _materials(5 + 12 + 1)
    k = 0
    for p0, eu, ev in quads:
        q = _quad(p0, eu, ev, tess, tess)
        tris.append(q); mids.append(np.full(len(q), k)); k += 1
    for half, yaw, centre in (((0.15, 0.15, 0.15), -17.0, (0.68, 0.15, 0.62)),
                              ((0.15, 0.30, 0.15), 17.0, (0.33, 0.30, 0.33))):
        box = _unit_box(tess) * np.asarray(half)
        box = box @ _rot_y(yaw).T + np.asarray(centre)
        per_face = len(box) // 6
        for f in range(6):
            tris.append(box[f * per_face:(f + 1) * per_face]); mids.append(np.full(per_face, k)); k += 1
    light = _quad((0.375, 0.995, 0.375), (0.25, 0, 0), (0, 0, 0.25), tess, tess)
    tris.append(light); mids.append(np.full(len(light), k))
    mats["type"][:k] = MAT_DIFFUSE
    mats["albedo"][:k] = rng.uniform(0.2, 0.8, (k, 3))
    mats["type"][k] = MAT_EMISSIVE
    mats["emission"][k] = 15.0
    cam = make_camera((0.5, 0.5, 2.4), (0.5, 0.5, 0.0), (0, 1, 0), 40.0, width / height)
    return Scene("cornell", np.concatenate(tris).astype(np.float32), np.concatenate(mids).astype(np.int32),
                 mats, np.zeros(6, np.float32), cam, width, height)


# --------------------------------------------------------------------------
# config 2: interior
# --------------------------------------------------------------------------
def interior(seed=1, width=1920, height=1080, n_boxes=2000, n_spheres=500, subdiv=3) -> Scene:
    """Room 40 x 8 x 40 with n_boxes rotated boxes (192 tris each) and n_spheres
    icospheres (20*4^subdiv tris each); 60 % Lambert / 25 % GGX roughness
    U(0.1,0.5) / 15 % mirror per object; 16 emissive ceiling panels (Le = 8).
    Full size: about 1.02 M triangles (BASELINE.json config 2)."""
    rng = np.random.default_rng(seed)
    X, Y, Z = 40.0, 8.0, 40.0
    eye = np.array([3.0, 4.0, 3.0])
    tris, mids = [], []
    shell = [((0, 0, 0), (0, 0, Z), (X, 0, 0)), ((0, Y, 0), (X, 0, 0), (0, 0, Z)),
             ((0, 0, 0), (X, 0, 0), (0, Y, 0)), ((0, 0, Z), (0, Y, 0), (X, 0, 0)),
             ((0, 0, 0), (0, Y, 0), (0, 0, Z)), ((X, 0, 0), (0, 0, Z), (0, Y, 0))]
    for p0, eu, ev in shell:
        q = _quad(p0, eu, ev, 4, 4); tris.append(q); mids.append(np.full(len(q), 0))
    for i in range(4):
        for j in range(4):
            q = _quad((2.5 + 10 * i, Y - 0.01, 2.5 + 10 * j), (5, 0, 0), (0, 0, 5), 4, 4)
            tris.append(q); mids.append(np.full(len(q), 1))
    n_obj = n_boxes + n_spheres
    mats = _materials(2 + n_obj)
    mats["type"][0] = MAT_DIFFUSE; mats["albedo"][0] = 0.7
    mats["type"][1] = MAT_EMISSIVE; mats["emission"][1] = 8.0

    def place(n, radius_of):
        """draw centres until n objects clear a radius-1.5 sphere round the camera"""
        out_c, out_p = [], []
        need = n
        while need > 0:
            c = np.stack([rng.uniform(1, X - 1, need), rng.uniform(1, Y - 1, need), rng.uniform(1, Z - 1, need)], -1)
            p = radius_of(need)
            r = p[1]
            ok = np.linalg.norm(c - eye, axis=1) > 1.5 + r
            out_c.append(c[ok]); out_p.append(p[0][ok])
            need -= int(ok.sum())
        return np.concatenate(out_c), np.concatenate(out_p)

    def box_params(n):
        he = rng.uniform(0.1, 0.6, (n, 3))
        return he, np.linalg.norm(he, axis=1)

    def sph_params(n):
        r = rng.uniform(0.2, 0.8, n)
        return r, r

    bc, bhe = place(n_boxes, box_params)
    R = _random_rotations(rng, n_boxes)
    ub = _unit_box(4)                                     # [192,3,3]
    b = ub[None] * bhe[:, None, None, :]                  # [n,192,3,3]
    b = np.einsum("ntvk,njk->ntvj", b, R) + bc[:, None, None, :]
    tris.append(b.reshape(-1, 3, 3)); mids.append(np.repeat(2 + np.arange(n_boxes), len(ub)))
    sc, sr = place(n_spheres, sph_params)
    ico = _icosphere(subdiv)
    s = ico[None] * sr[:, None, None, None] + sc[:, None, None, :]
    tris.append(s.reshape(-1, 3, 3)); mids.append(np.repeat(2 + n_boxes + np.arange(n_spheres), len(ico)))
    kind = rng.random(n_obj)
    typ = np.where(kind < 0.60, MAT_DIFFUSE, np.where(kind < 0.85, MAT_GLOSSY, MAT_SPECULAR))
    mats["type"][2:] = typ
    mats["albedo"][2:] = rng.uniform(0.2, 0.8, (n_obj, 3))
    mats["roughness"][2:] = rng.uniform(0.1, 0.5, n_obj)
    cam = make_camera(eye, (X / 2, Y / 2, Z / 2), (0, 1, 0), 55.0, width / height)
    return Scene("interior", np.concatenate(tris).astype(np.float32), np.concatenate(mids).astype(np.int32),
                 mats, np.zeros(6, np.float32), cam, width, height)


# --------------------------------------------------------------------------
# config 4: landscape
# --------------------------------------------------------------------------
def _fbm_heights(rng, n, octaves=8, base_period=512.0, gain=0.5):
    """Value-noise fBm on an n x n grid: per octave a random lattice, quintic fade,
    bilinear blend; normalised to [0,1]."""
    x = np.arange(n, dtype=np.float64)
    h = np.zeros((n, n), np.float64)
    amp, period, total = 1.0, base_period, 0.0
    for _ in range(octaves):
        cells = int(np.ceil(n / period)) + 2
        lat = rng.random((cells, cells))
        f = x / period
        i = np.floor(f).astype(np.int64)
        t = f - i
        t = t * t * t * (t * (t * 6 - 15) + 10)
        a = lat[np.ix_(i, i)]; b = lat[np.ix_(i + 1, i)]
        c = lat[np.ix_(i, i + 1)]; d = lat[np.ix_(i + 1, i + 1)]
        tx = t[:, None]; tz = t[None, :]
        h += amp * ((a * (1 - tx) + b * tx) * (1 - tz) + (c * (1 - tx) + d * tx) * tz)
        total += amp
        amp *= gain
        period *= 0.5
    h /= total
    h -= h.min()
    h /= max(h.max(), 1e-12)
    return h


def _cone_cyl(sides=16):
    """Unit tree proxy: trunk cylinder radius 1, y in [0,1] (sides*4 tris: side quads
    split + caps), cone radius 1 base at y=0, apex y=1 (sides*2 tris: side + base)."""
    a = np.arange(sides) * (2 * np.pi / sides)
    a2 = np.roll(a, -1)
    c0 = np.stack([np.cos(a), np.zeros(sides), np.sin(a)], -1)
    c1 = np.stack([np.cos(a2), np.zeros(sides), np.sin(a2)], -1)
    up = np.array([0.0, 1.0, 0.0])
    o = np.zeros((sides, 3))
    cyl = np.concatenate([np.stack([c0, c0 + up, c1 + up], 1), np.stack([c0, c1 + up, c1], 1),
                          np.stack([o + up, c1 + up, c0 + up], 1), np.stack([o, c0, c1], 1)], 0)
    cone = np.concatenate([np.stack([c0, o + up, c1], 1), np.stack([o, c0, c1], 1)], 0)
    return cyl, cone


def landscape(seed=2, width=1920, height=1080, n=2048, n_trees=20000, amplitude=200.0) -> Scene:
    """n x n fBm heightfield (1-unit spacing, (n-1)^2*2 tris) plus n_trees tree proxies
    of 96 tris each; full size 8,380,418 + 1,920,000 = 10,300,418 triangles
    (BASELINE.json config 4).  Camera at a grazing angle over the terrain."""
    rng = np.random.default_rng(seed)
    hts = _fbm_heights(rng, n, base_period=512.0 * n / 2048.0) * amplitude * (n / 2048.0)
    xs = np.arange(n, dtype=np.float32)
    P = np.empty((n, n, 3), np.float32)
    P[..., 0] = xs[:, None]; P[..., 1] = hts.astype(np.float32); P[..., 2] = xs[None, :]
    p00, p10, p01, p11 = P[:-1, :-1], P[1:, :-1], P[:-1, 1:], P[1:, 1:]
    terr = np.empty(((n - 1), (n - 1), 2, 3, 3), np.float32)
    terr[:, :, 0, 0], terr[:, :, 0, 1], terr[:, :, 0, 2] = p00, p01, p11   # normal +y
    terr[:, :, 1, 0], terr[:, :, 1, 1], terr[:, :, 1, 2] = p00, p11, p10
    terr = terr.reshape(-1, 3, 3)
    lo, hi = int(10 * n / 2048), int(2037 * n / 2048)
    gx = rng.integers(lo, hi + 1, n_trees); gz = rng.integers(lo, hi + 1, n_trees)
    tr_r = rng.uniform(0.3, 0.5, n_trees); tr_h = rng.uniform(2, 4, n_trees)
    co_r = rng.uniform(1.5, 3.0, n_trees); co_h = rng.uniform(5, 10, n_trees)
    glossy = rng.random(n_trees) < 0.10
    alb = rng.uniform(0.2, 0.8, (n_trees, 3)); rough = rng.uniform(0.1, 0.5, n_trees)
    base = np.stack([gx, hts[gx, gz] - 0.2, gz], -1).astype(np.float64)
    cyl, cone = _cone_cyl(16)
    tc = cyl[None] * np.stack([tr_r, tr_h + 0.2, tr_r], -1)[:, None, None, :] + base[:, None, None, :]
    cbase = base + np.stack([np.zeros(n_trees), tr_h + 0.2, np.zeros(n_trees)], -1)
    cc = cone[None] * np.stack([co_r, co_h, co_r], -1)[:, None, None, :] + cbase[:, None, None, :]
    trees = np.concatenate([tc, cc], axis=1).reshape(-1, 3, 3).astype(np.float32)
    mats = _materials(1 + n_trees)
    mats["type"][0] = MAT_DIFFUSE; mats["albedo"][0] = (0.4, 0.5, 0.3)
    mats["type"][1:] = np.where(glossy, MAT_GLOSSY, MAT_DIFFUSE)
    mats["albedo"][1:] = alb; mats["roughness"][1:] = rough
    mid = np.concatenate([np.zeros(len(terr), np.int32),
                          np.repeat(1 + np.arange(n_trees, dtype=np.int32), cyl.shape[0] + cone.shape[0])])
    cx, cz = n // 2, int(200 * n / 2048)
    eye = np.array([cx, hts[cx, cz] + 15.0 * max(n / 2048.0, 0.25), cz], np.float64)
    fwd = np.array([0.0, -np.sin(np.radians(5.0)), np.cos(np.radians(5.0))])
    cam = make_camera(eye, eye + fwd, (0, 1, 0), 45.0, width / height)
    env = np.array([1, 1, 1, 0.5, 0.7, 1.0], np.float32)
    return Scene("landscape", np.concatenate([terr, trees]), mid, mats, env, cam, width, height)


# --------------------------------------------------------------------------
# small analytic scenes used to pin the oracle
# --------------------------------------------------------------------------
def furnace_sphere(subdiv=2, albedo=1.0, mat_type=MAT_DIFFUSE, roughness=0.3, width=32, height=32) -> Scene:
    """Convex icosphere of the given albedo under uniform environment radiance 1."""
    tri = _icosphere(subdiv).astype(np.float32)
    mats = _materials(1)
    mats["type"][0] = mat_type; mats["albedo"][0] = albedo; mats["roughness"][0] = roughness
    cam = make_camera((0, 0, 3.0), (0, 0, 0), (0, 1, 0), 50.0, width / height)
    return Scene("furnace_sphere", tri, np.zeros(len(tri), np.int32), mats, np.ones(6, np.float32), cam, width, height)


def emissive_box(seed=0, albedo=0.5, emission=1.0, width=16, height=16) -> Scene:      # (name kept from the survey; see docstring)
    """Closed unit cube seen from inside.  The method has no surface that both emits
    and reflects, so this returns a plain Lambert cube under NO light; tests use
    it for occlusion invariants (every ray from inside hits, image stays 0)."""
    box = (_unit_box(2) * 0.5 + 0.5).astype(np.float32)
    mats = _materials(1)
    mats["type"][0] = MAT_DIFFUSE; mats["albedo"][0] = albedo
    cam = make_camera((0.5, 0.5, 0.9), (0.5, 0.45, 0.0), (0, 1, 0), 70.0, width / height)
    return Scene("closed_box", box, np.zeros(len(box), np.int32), mats, np.zeros(6, np.float32), cam, width, height)


def floor_plane(mat_type=MAT_DIFFUSE, albedo=0.5, roughness=0.3, width=32, height=32, tess=8) -> Scene:
    """One big horizontal floor (normal +y) filling the view, uniform env 1."""
    q = _quad((-50, 0, -50), (0, 0, 100), (100, 0, 0), tess, tess).astype(np.float32)
    mats = _materials(1)
    mats["type"][0] = mat_type; mats["albedo"][0] = albedo; mats["roughness"][0] = roughness
    cam = make_camera((0, 3.0, 0), (0.3, 0.0, 0.2), (0, 0, 1), 60.0, width / height)
    return Scene("floor", q, np.zeros(len(q), np.int32), mats, np.ones(6, np.float32), cam, width, height)


def checker_floor(seed=0, width=32, height=32, tess=64, p_diffuse=0.5) -> Scene:
    """Floor whose cells alternate randomly between Lambert, GGX and mirror: every
    reuse group of a few pixels is HYBRID with high probability."""
    rng = np.random.default_rng(seed)
    q = _quad((-4, 0, -4), (0, 0, 8), (8, 0, 0), tess, tess).astype(np.float32)
    ncell = tess * tess
    kind = rng.random(ncell)
    typ = np.where(kind < p_diffuse, MAT_DIFFUSE, np.where(kind < 0.5 + p_diffuse / 2, MAT_GLOSSY, MAT_SPECULAR))
    mats = _materials(ncell)
    mats["type"] = typ; mats["albedo"] = rng.uniform(0.2, 0.8, (ncell, 3)); mats["roughness"] = rng.uniform(0.1, 0.5, ncell)
    mid = np.concatenate([np.arange(ncell), np.arange(ncell)]).astype(np.int32)
    cam = make_camera((0, 3.0, 0), (0.2, 0.0, 0.1), (0, 0, 1), 60.0, width / height)
    return Scene("checker_floor", q, mid, mats, np.ones(6, np.float32), cam, width, height)


def random_rays(seed, n, bmin, bmax, inactive_frac=0.0):
    """n rays (float32[n,8]: o, tmin, d, tmax) with origins uniform in the box
    [bmin,bmax] grown by 10 % and uniform directions; a fraction marked inactive
    (tmax = -1)."""
    rng = np.random.default_rng(seed)
    bmin = np.asarray(bmin, np.float64); bmax = np.asarray(bmax, np.float64)
    ext = bmax - bmin
    o = bmin - 0.1 * ext + rng.random((n, 3)) * 1.2 * ext
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    r = np.zeros((n, 8), np.float32)
    r[:, 0:3] = o; r[:, 4:7] = d; r[:, 7] = 1e30
    if inactive_frac > 0:
        r[rng.random(n) < inactive_frac, 7] = -1.0
    return r


def by_name(name, **kw) -> Scene:
    return {"cornell": cornell, "interior": interior, "landscape": landscape}[name](**kw)
