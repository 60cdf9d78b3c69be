"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds NO arithmetic of the method (no RNG streams, no path map, no sampler):
only triangle soups, materials, cameras and seeded test points.  The scenes stand in for
the paper's seven public scenes, which are third-party datasets that
are not available here; they take the paper's shapes: image-sized chain counts, diffuse /
dielectric / conductor materials plus one diffuse area light, no textures (L775-L780).
BASELINE.json `configs` fixes what each scene contains; the placements that it leaves
open are fixed here from a seed (marked "parity unpinned").
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

MAT_LAMBERT, MAT_DIELECTRIC, MAT_GGX, MAT_EMITTER = 0, 1, 2, 3


@dataclass
class SceneDesc:
    vertices: np.ndarray          # float32 [nv, 3]
    indices: np.ndarray           # uint32  [nt, 3]
    tri_material: np.ndarray      # uint32  [nt]
    materials: np.ndarray         # float32 [nm, 9]: kind, a0, a1, a2, ior, roughness, Le0, Le1, Le2
    env_radiance: tuple = (0.0, 0.0, 0.0)
    cam_pos: tuple = (0.0, 0.0, 0.0)
    cam_look: tuple = (0.0, 0.0, 1.0)
    cam_up: tuple = (0.0, 1.0, 0.0)
    vfov_deg: float = 40.0
    width: int = 64
    height: int = 64
    max_path_len: int = 4
    name: str = ""
    meta: dict = field(default_factory=dict)
    nee: bool = False             # next-event estimation + MIS (Q21): four PSS coordinates per vertex

    @property
    def dim(self) -> int:
        return (4 if self.nee else 2) * self.max_path_len

    @property
    def n_tris(self) -> int:
        return int(self.indices.shape[0])


@dataclass
class Analytic2DDesc:
    weights: np.ndarray   # float32 [k]
    means: np.ndarray     # float32 [k, 2]
    stddevs: np.ndarray   # float32 [k]
    width: int = 32
    height: int = 32
    name: str = "analytic2d"

    @property
    def dim(self) -> int:
        return 2


def material(kind, a=(0, 0, 0), ior=1.0, rough=0.0, le=(0, 0, 0)):
    return np.array([kind, a[0], a[1], a[2], ior, rough, le[0], le[1], le[2]], dtype=np.float32)


class _Mesh:
    def __init__(self):
        self.v, self.i, self.m = [], [], []
        self.nv = 0

    def add(self, verts, tris, mat):
        verts = np.asarray(verts, dtype=np.float64).reshape(-1, 3)
        tris = np.asarray(tris, dtype=np.int64).reshape(-1, 3)
        self.v.append(verts)
        self.i.append(tris + self.nv)
        self.m.append(np.full(len(tris), mat, dtype=np.uint32))
        self.nv += len(verts)

    def quad(self, p0, p1, p2, p3, mat, div=1):
        """Quad p0,p1,p2,p3 (counter-clockwise seen from its front), div x div cells."""
        p0, p1, p2, p3 = (np.asarray(p, dtype=np.float64) for p in (p0, p1, p2, p3))
        s = np.linspace(0.0, 1.0, div + 1)
        grid = np.array([[(1 - a) * (1 - b) * p0 + a * (1 - b) * p1 + a * b * p2 + (1 - a) * b * p3 for a in s] for b in s])
        verts = grid.reshape(-1, 3)
        tris = []
        for b in range(div):
            for a in range(div):
                i00 = b * (div + 1) + a
                i10, i01, i11 = i00 + 1, i00 + div + 1, i00 + div + 2
                tris += [(i00, i10, i11), (i00, i11, i01)]
        self.add(verts, tris, mat)

    def finish(self):
        return (np.concatenate(self.v).astype(np.float32), np.concatenate(self.i).astype(np.uint32),
                np.concatenate(self.m).astype(np.uint32))


def icosphere(level: int):
    """Unit icosphere, outward-facing triangles: 20 * 4**level faces."""
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t),
         (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    v = [np.array(p, dtype=np.float64) / np.linalg.norm(p) for p in v]
    f = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6),
         (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10),
         (8, 6, 7), (9, 8, 1)]
    for _ in range(level):
        cache, nf = {}, []

        def mid(a, b):
            key = (min(a, b), max(a, b))
            if key not in cache:
                p = v[a] + v[b]
                v.append(p / np.linalg.norm(p))
                cache[key] = len(v) - 1
            return cache[key]

        for a, b, c in f:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        f = nf
    return np.array(v), np.array(f, dtype=np.int64)


def _box_faces(mesh: _Mesh, c, h, rot, mat, div=1, skip_bottom=False):
    """Axis box of half-extents h, rotated by matrix rot about centre c; outward faces."""
    c, h = np.asarray(c, dtype=np.float64), np.asarray(h, dtype=np.float64)
    corner = lambda sx, sy, sz: c + rot @ (np.array([sx, sy, sz]) * h)
    faces = [
        ((+1, -1, -1), (+1, +1, -1), (+1, +1, +1), (+1, -1, +1)),  # +x
        ((-1, -1, +1), (-1, +1, +1), (-1, +1, -1), (-1, -1, -1)),  # -x
        ((-1, +1, -1), (-1, +1, +1), (+1, +1, +1), (+1, +1, -1)),  # +y
        ((-1, -1, +1), (-1, -1, -1), (+1, -1, -1), (+1, -1, +1)),  # -y
        ((+1, -1, +1), (+1, +1, +1), (-1, +1, +1), (-1, -1, +1)),  # +z
        ((-1, -1, -1), (-1, +1, -1), (+1, +1, -1), (+1, -1, -1)),  # -z
    ]
    for k, fc in enumerate(faces):
        if skip_bottom and k == 3:
            continue
        mesh.quad(*[corner(*p) for p in fc], mat, div)


def _prism(mesh: _Mesh, profile, c, hy, rot, mat, centre_fan):
    """Extrude a closed 2-D profile (x,z; clockwise seen from +y) along y in [-hy, hy]; outward faces."""
    n = len(profile)
    top = np.array([[p[0], hy, p[1]] for p in profile])
    bot = np.array([[p[0], -hy, p[1]] for p in profile])
    verts = np.concatenate([top, bot, [[0, hy, 0], [0, -hy, 0]]])
    tris = []
    for k in range(n):
        k2 = (k + 1) % n
        tris += [(k, k2, n + k2), (k, n + k2, n + k)]      # side
    if centre_fan:
        for k in range(n):
            k2 = (k + 1) % n
            tris += [(2 * n, k2, k), (2 * n + 1, n + k, n + k2)]
    else:
        for k in range(1, n - 1):
            tris += [(0, k + 1, k), (n, n + k, n + k + 1)]
    verts = (rot @ verts.T).T + np.asarray(c, dtype=np.float64)
    mesh.add(verts, [(a, c_, b) for a, b, c_ in tris], mat)   # outward-facing


def _rot_y(deg):
    a = np.deg2rad(deg)
    return np.array([[np.cos(a), 0, np.sin(a)], [0, 1, 0], [-np.sin(a), 0, np.cos(a)]])


def _rot_quat(q):
    w, x, y, z = q / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


# --------------------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------------------

def furnace(width=64, height=64, level=4, max_path_len=4) -> SceneDesc:
    """configs[0]: white furnace.  Lambert sphere r=1, albedo 0.5, environment radiance 1."""
    v, f = icosphere(level)
    mesh = _Mesh()
    mesh.add(v, f, 0)
    verts, idx, tm = mesh.finish()
    mats = np.stack([material(MAT_LAMBERT, (0.5, 0.5, 0.5))])
    return SceneDesc(verts, idx, tm, mats, env_radiance=(1.0, 1.0, 1.0), cam_pos=(0, 0, 4), cam_look=(0, 0, 0),
                     cam_up=(0, 1, 0), vfov_deg=40.0, width=width, height=height, max_path_len=max_path_len, name="furnace")


def cornell(seed=2, width=256, height=256, max_path_len=8) -> SceneDesc:
    """configs[1]: procedural Cornell box, 32 triangles, all Lambertian, one ceiling quad light."""
    rng = np.random.default_rng(seed)
    ang_tall, ang_short = rng.uniform(-30.0, 30.0, size=2)
    mesh = _Mesh()
    WHITE, RED, GREEN, LIGHT = 0, 1, 2, 3
    mesh.quad((0, 0, 0), (1, 0, 0), (1, 0, 1), (0, 0, 1), WHITE)          # floor
    mesh.quad((0, 1, 1), (1, 1, 1), (1, 1, 0), (0, 1, 0), WHITE)          # ceiling
    mesh.quad((0, 0, 1), (1, 0, 1), (1, 1, 1), (0, 1, 1), WHITE)          # back wall z=1
    mesh.quad((0, 0, 0), (0, 0, 1), (0, 1, 1), (0, 1, 0), RED)            # left wall x=0
    mesh.quad((1, 0, 1), (1, 0, 0), (1, 1, 0), (1, 1, 1), GREEN)          # right wall x=1
    _box_faces(mesh, (0.33, 0.3, 0.67), (0.15, 0.3, 0.15), _rot_y(ang_tall), WHITE, skip_bottom=True)
    _box_faces(mesh, (0.68, 0.15, 0.33), (0.15, 0.15, 0.15), _rot_y(ang_short), WHITE, skip_bottom=True)
    a, b, y = 0.5 - 0.125, 0.5 + 0.125, 0.999
    mesh.quad((a, y, a), (b, y, a), (b, y, b), (a, y, b), LIGHT)           # light, normal -y
    verts, idx, tm = mesh.finish()
    mats = np.stack([material(MAT_LAMBERT, (0.73, 0.73, 0.73)), material(MAT_LAMBERT, (0.65, 0.05, 0.05)),
                     material(MAT_LAMBERT, (0.12, 0.45, 0.15)), material(MAT_EMITTER, le=(17, 17, 17))])
    return SceneDesc(verts, idx, tm, mats, cam_pos=(0.5, 0.5, -1.37), cam_look=(0.5, 0.5, 0.0), vfov_deg=40.0,
                     width=width, height=height, max_path_len=max_path_len, name="cornell",
                     meta={"angles": (float(ang_tall), float(ang_short))})


def caustic(width=512, height=512, level=5, max_path_len=12) -> SceneDesc:
    """configs[2]: dielectric icosphere (IOR 1.5) over a Lambert ground, small quad light above."""
    mesh = _Mesh()
    GROUND, GLASS, LIGHT = 0, 1, 2
    mesh.quad((-5, 0, -5), (-5, 0, 5), (5, 0, 5), (5, 0, -5), GROUND)
    v, f = icosphere(level)
    mesh.add(v + np.array([0.0, 1.5, 0.0]), f, GLASS)
    a, y = 0.05, 2.7
    mesh.quad((-a, y, -a), (a, y, -a), (a, y, a), (-a, y, a), LIGHT)       # normal -y, area 0.01
    verts, idx, tm = mesh.finish()
    mats = np.stack([material(MAT_LAMBERT, (0.8, 0.8, 0.8)), material(MAT_DIELECTRIC, ior=1.5),
                     material(MAT_EMITTER, le=(500, 500, 500))])
    return SceneDesc(verts, idx, tm, mats, cam_pos=(0, 3.5, -7), cam_look=(0, 0.8, 0), vfov_deg=35.0, width=width,
                     height=height, max_path_len=max_path_len, name="caustic")


def machines(seed=4, n_objects=2000, room=10.0, width=1024, height=576, max_path_len=16, box_div=5, cyl_seg=64,
             gear_teeth=16, scale_lo=0.05, scale_hi=1.0, light_size=1.0, light_le=50.0) -> SceneDesc:
    """configs[3]: procedural 'transparent machines': boxes, cylinders and gear prisms in a closed room.

    `scale` (log-uniform in [scale_lo, scale_hi]) is an object's edge length / diameter.  An
    object whose bounding sphere would contain the camera or touch the light is redrawn.
    """
    rng = np.random.default_rng(seed)
    R = room
    mesh = _Mesh()
    WALL, LIGHT = 0, 1
    mats = [material(MAT_LAMBERT, (0.7, 0.7, 0.7)), material(MAT_EMITTER, le=(light_le,) * 3)]
    _q = mesh.quad
    _q((0, 0, 0), (0, 0, R), (R, 0, R), (R, 0, 0), WALL)      # floor
    _q((0, R, 0), (R, R, 0), (R, R, R), (0, R, R), WALL)      # ceiling
    _q((0, 0, 0), (R, 0, 0), (R, R, 0), (0, R, 0), WALL)      # z=0
    _q((0, 0, R), (0, R, R), (R, R, R), (R, 0, R), WALL)      # z=R
    _q((0, 0, 0), (0, R, 0), (0, R, R), (0, 0, R), WALL)      # x=0
    _q((R, 0, 0), (R, 0, R), (R, R, R), (R, R, 0), WALL)      # x=R
    a, b, y = R / 2 - light_size / 2, R / 2 + light_size / 2, R - 0.01 * R / 10.0
    _q((a, y, a), (b, y, a), (b, y, b), (a, y, b), LIGHT)     # normal -y
    cam_pos = np.array([0.07 * R, 0.5 * R, 0.07 * R])
    cam_look = np.array([0.5 * R, 0.4 * R, 0.5 * R])
    light_c = np.array([R / 2, y, R / 2])
    counts = {"box": 0, "cylinder": 0, "gear": 0, "lambert": 0, "dielectric": 0, "ggx": 0}
    placed = 0
    while placed < n_objects:
        kind = int(rng.integers(0, 3))
        c = rng.uniform(0.05 * R, 0.95 * R, size=3)
        s = float(np.exp(rng.uniform(np.log(scale_lo), np.log(scale_hi)))) * (R / 10.0)
        q = rng.normal(size=4)
        u = float(rng.uniform())
        alb = rng.uniform(0.1, 0.9, size=3)
        ior = float(rng.uniform(1.3, 1.7))
        alpha = float(rng.uniform(0.05, 0.5))
        f0 = rng.uniform(0.5, 0.95, size=3)
        h = 0.5 * s
        bound = h * 3 ** 0.5
        if np.linalg.norm(c - cam_pos) < bound + 0.03 * R or np.linalg.norm(c - light_c) < bound + 0.75 * light_size:
            continue
        if u < 0.4:
            mats.append(material(MAT_LAMBERT, alb)); counts["lambert"] += 1
        elif u < 0.7:
            mats.append(material(MAT_DIELECTRIC, ior=ior)); counts["dielectric"] += 1
        else:
            mats.append(material(MAT_GGX, f0, rough=alpha)); counts["ggx"] += 1
        mat = len(mats) - 1
        rot = _rot_quat(q)
        if kind == 0:
            _box_faces(mesh, c, (h, h, h), rot, mat, div=box_div); counts["box"] += 1
        elif kind == 1:
            ang = 2 * np.pi * np.arange(cyl_seg) / cyl_seg
            prof = np.stack([h * np.sin(ang), h * np.cos(ang)], axis=1)
            _prism(mesh, prof, c, h, rot, mat, centre_fan=False); counts["cylinder"] += 1
        else:
            n = 4 * gear_teeth
            ang = 2 * np.pi * (np.arange(n) + 0.5) / n
            rad = np.where((np.arange(n) // 2) % 2 == 0, h, 0.75 * h)
            prof = np.stack([rad * np.sin(ang), rad * np.cos(ang)], axis=1)
            _prism(mesh, prof, c, 0.4 * h, rot, mat, centre_fan=True); counts["gear"] += 1
        placed += 1
    verts, idx, tm = mesh.finish()
    return SceneDesc(verts, idx, tm, np.stack(mats), cam_pos=tuple(cam_pos), cam_look=tuple(cam_look), vfov_deg=50.0,
                     width=width, height=height, max_path_len=max_path_len, name="machines", meta=counts)


def mini_machines(seed=7, n_objects=24, width=48, height=32, max_path_len=6) -> SceneDesc:
    """Small cousin of `machines` (a few hundred triangles, all three materials) for CPU-side tests."""
    return machines(seed=seed, n_objects=n_objects, room=4.0, width=width, height=height, max_path_len=max_path_len,
                    box_div=1, cyl_seg=10, gear_teeth=5, scale_lo=0.2, scale_hi=1.0, light_size=1.6, light_le=20.0)


def ggx_room(seed=5, width=32, height=32, max_path_len=5, alpha=0.3) -> SceneDesc:
    """Closed room whose walls are rough conductors and dielectric/GGX blocks: every lit path has a non-zero score."""
    rng = np.random.default_rng(seed)
    R = 2.0
    mesh = _Mesh()
    mats = [material(MAT_GGX, (0.8, 0.7, 0.6), rough=alpha), material(MAT_EMITTER, le=(10, 10, 10)),
            material(MAT_DIELECTRIC, ior=1.5), material(MAT_GGX, (0.9, 0.9, 0.6), rough=0.15),
            material(MAT_LAMBERT, (0.6, 0.6, 0.7))]
    _q = mesh.quad
    _q((0, 0, 0), (0, 0, R), (R, 0, R), (R, 0, 0), 4)
    _q((0, R, 0), (R, R, 0), (R, R, R), (0, R, R), 0)
    _q((0, 0, 0), (R, 0, 0), (R, R, 0), (0, R, 0), 0)
    _q((0, 0, R), (0, R, R), (R, R, R), (R, 0, R), 0)
    _q((0, 0, 0), (0, R, 0), (0, R, R), (0, 0, R), 0)
    _q((R, 0, 0), (R, 0, R), (R, R, R), (R, R, 0), 0)
    _q((0.6, 1.99, 0.6), (1.4, 1.99, 0.6), (1.4, 1.99, 1.4), (0.6, 1.99, 1.4), 1)
    _box_faces(mesh, (0.7, 0.55, 1.2), (0.3, 0.5, 0.3), _rot_y(rng.uniform(-30, 30)), 2)   # floats above the floor: no coplanar faces
    _box_faces(mesh, (1.4, 0.3, 0.8), (0.3, 0.3, 0.3), _rot_quat(rng.normal(size=4)), 3)
    verts, idx, tm = mesh.finish()
    return SceneDesc(verts, idx, tm, np.stack(mats), cam_pos=(0.3, 1.0, 0.2), cam_look=(1.2, 0.7, 1.3), vfov_deg=60.0,
                     width=width, height=height, max_path_len=max_path_len, name="ggx_room")


def closed_furnace(albedo=0.5, emission=1.0, width=8, height=8, max_path_len=6) -> SceneDesc:
    """Camera inside a closed box: Lambert walls except an emitting ceiling (second furnace of the pins)."""
    mesh = _Mesh()
    R = 1.0
    _q = mesh.quad
    _q((0, 0, 0), (0, 0, R), (R, 0, R), (R, 0, 0), 0)
    _q((0, R, 0), (R, R, 0), (R, R, R), (0, R, R), 1)
    _q((0, 0, 0), (R, 0, 0), (R, R, 0), (0, R, 0), 0)
    _q((0, 0, R), (0, R, R), (R, R, R), (R, 0, R), 0)
    _q((0, 0, 0), (0, R, 0), (0, R, R), (0, 0, R), 0)
    _q((R, 0, 0), (R, 0, R), (R, R, R), (R, R, 0), 0)
    verts, idx, tm = mesh.finish()
    mats = np.stack([material(MAT_LAMBERT, (albedo,) * 3), material(MAT_EMITTER, le=(emission,) * 3)])
    return SceneDesc(verts, idx, tm, mats, cam_pos=(0.5, 0.5, 0.5), cam_look=(0.5, 0.2, 1.0), vfov_deg=60.0, width=width,
                     height=height, max_path_len=max_path_len, name="closed_furnace")


def mixture3(width=32, height=32) -> Analytic2DDesc:
    """Three separated wrapped-Gaussian modes on T^2 (stationarity pins); integral = 1."""
    return Analytic2DDesc(np.array([0.5, 0.3, 0.2], dtype=np.float32),
                          np.array([[0.25, 0.30], [0.70, 0.65], [0.55, 0.15]], dtype=np.float32),
                          np.array([0.06, 0.09, 0.05], dtype=np.float32), width, height, "mixture3")


def single_mode(s=0.1, width=32, height=32) -> Analytic2DDesc:
    return Analytic2DDesc(np.array([1.0], dtype=np.float32), np.array([[0.5, 0.5]], dtype=np.float32),
                          np.array([s], dtype=np.float32), width, height, "single_mode")


# --------------------------------------------------------------------------------------
# seeded test points
# --------------------------------------------------------------------------------------

def seeded_states(n: int, d: int, seed: int) -> np.ndarray:
    """n PSS points with 24-bit coordinates in [0,1) (exact in float32), float32 [n, d]."""
    rng = np.random.default_rng(seed)
    return (rng.integers(0, 1 << 24, size=(n, d)).astype(np.float64) / float(1 << 24)).astype(np.float32)


def seeded_rays(scene: SceneDesc, n: int, seed: int):
    """n rays: origins uniform in the (slightly inflated) bounding box, directions uniform on the sphere."""
    rng = np.random.default_rng(seed)
    lo, hi = scene.vertices.min(0), scene.vertices.max(0)
    pad = 0.1 * (hi - lo)
    o = rng.uniform(lo - pad, hi + pad, size=(n, 3))
    d = rng.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    return o.astype(np.float32), d.astype(np.float32)
