"""Seeded synthetic input generators (BASELINE.json configs 0-4; recipe in DESIGN.md section 5).

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path: it
produces input arrays and holds none of the rasteriser's arithmetic (no projection, no
window function, no compositing, no gradients).  The paper measures on TUM RGB-D and
Replica; neither is available, so these scenes stand in for them and take
only the image shapes / intrinsics and the workload statistics (10^4-10^6 triangles of a
few centimetres; sigma = 0.5).

World frame: z up, room centred at the origin.  Camera frame: x right, y down, z forward.
``T_cw`` (3x4, row-major ``[R|t]``) maps world to camera, PAPER.md:88-90 (Eq. 1).
Everything is generated in float64 with ``numpy.random.default_rng(seed)`` and cast to
float32 once; both sides receive the same float32 buffers.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np


# --------------------------------------------------------------------------------------
# containers
# --------------------------------------------------------------------------------------
@dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    znear: float = 0.2


@dataclass
class Params:
    sigma: float = 0.5          # PAPER.md:464 (Table S4)
    alpha_min: float = 1.0 / 255.0
    t_min: float = 1e-4
    eps_area: float = 1e-6
    lambda_dep: float = 0.05
    min_opacity: bool = False   # face opacity = min instead of mean of the vertex opacities (ablation)
    tight_binning: bool = False  # bin a face only into the tiles its triangle meets (reading S31)


@dataclass
class Scene:
    name: str
    seed: int
    cam: Camera
    params: Params
    pos: np.ndarray                 # [V,3] float32, world
    color: np.ndarray               # [V,3] float32
    opacity: np.ndarray             # [V]   float32, already activated
    faces: Optional[np.ndarray]     # None = soup (V == 3M, face m = (3m,3m+1,3m+2))
    T_gt: List[np.ndarray]          # ground-truth poses, each [3,4] float32 (one per view)
    T_start: List[np.ndarray]       # starting poses for optimisation (tracking configs)
    pos_target: Optional[np.ndarray] = None    # geometry the target frame is rendered from
    color_target: Optional[np.ndarray] = None
    meta: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return self.pos.shape[0] // 3 if self.faces is None else self.faces.shape[0]

    @property
    def V(self) -> int:
        return self.pos.shape[0]


# --------------------------------------------------------------------------------------
# small pose helpers (input generation only)
# --------------------------------------------------------------------------------------
def _hat(w):
    return np.array([[0.0, -w[2], w[1]], [w[2], 0.0, -w[0]], [-w[1], w[0], 0.0]])


def se3_exp(tau):
    """SE(3) exponential, tau = (rho, theta), translation first (reading S17)."""
    tau = np.asarray(tau, dtype=np.float64)
    rho, th = tau[:3], tau[3:]
    a = np.linalg.norm(th)
    K = _hat(th)
    if a < 1e-10:
        R = np.eye(3) + K + 0.5 * K @ K
        Vm = np.eye(3) + 0.5 * K + K @ K / 6.0
    else:
        R = np.eye(3) + np.sin(a) / a * K + (1 - np.cos(a)) / a**2 * K @ K
        Vm = np.eye(3) + (1 - np.cos(a)) / a**2 * K + (a - np.sin(a)) / a**3 * K @ K
    T = np.eye(4)
    T[:3, :3] = R
    T[:3, 3] = Vm @ rho
    return T


def left_perturb(T34, tau):
    """Exp(tau) o T for a 3x4 pose."""
    T = np.eye(4)
    T[:3, :] = np.asarray(T34, dtype=np.float64)
    return (se3_exp(tau) @ T)[:3, :]


def look_level(center, yaw):
    """Level camera at `center` looking along (cos yaw, sin yaw, 0); returns T_cw [3,4] f64."""
    f = np.array([np.cos(yaw), np.sin(yaw), 0.0])
    d = np.array([0.0, 0.0, -1.0])
    r = np.cross(d, f)
    R = np.stack([r, d, f])
    t = -R @ np.asarray(center, dtype=np.float64)
    return np.concatenate([R, t[:, None]], axis=1)


# --------------------------------------------------------------------------------------
# surface tiling generator G(surfaces, N)
# --------------------------------------------------------------------------------------
@dataclass
class _Rect:
    origin: np.ndarray   # corner
    eu: np.ndarray       # unit tangent u
    ev: np.ndarray       # unit tangent v
    a: float             # extent along u
    b: float             # extent along v

    @property
    def area(self):
        return self.a * self.b

    @property
    def normal(self):
        return np.cross(self.eu, self.ev)


@dataclass
class _Sphere:
    center: np.ndarray
    radius: float

    @property
    def area(self):
        return 4.0 * np.pi * self.radius**2


def _room_rects(L, Wd, H):
    x0, x1, y0, y1, z0, z1 = -L / 2, L / 2, -Wd / 2, Wd / 2, -H / 2, H / 2
    ex, ey, ez = np.eye(3)
    return [
        _Rect(np.array([x0, y0, z0]), ex, ey, L, Wd),   # floor
        _Rect(np.array([x0, y0, z1]), ex, ey, L, Wd),   # ceiling
        _Rect(np.array([x0, y0, z0]), ex, ez, L, H),    # wall y = y0
        _Rect(np.array([x0, y1, z0]), ex, ez, L, H),    # wall y = y1
        _Rect(np.array([x0, y0, z0]), ey, ez, Wd, H),   # wall x = x0
        _Rect(np.array([x1, y0, z0]), ey, ez, Wd, H),   # wall x = x1
    ]


def _box_rects(center_xy, floor_z, edges, yaw):
    ex = np.array([np.cos(yaw), np.sin(yaw), 0.0])
    ey = np.array([-np.sin(yaw), np.cos(yaw), 0.0])
    ez = np.array([0.0, 0.0, 1.0])
    a, b, c = edges
    o = np.array([center_xy[0], center_xy[1], floor_z]) - 0.5 * a * ex - 0.5 * b * ey
    return [
        _Rect(o + c * ez, ex, ey, a, b),          # top
        _Rect(o, ex, ez, a, c),                   # side
        _Rect(o + b * ey, ex, ez, a, c),          # side
        _Rect(o, ey, ez, b, c),                   # side
        _Rect(o + a * ex, ey, ez, b, c),          # side
    ]


def _tangent_frame(n):
    """Two unit tangents for unit normals n [N,3]."""
    helper = np.where(np.abs(n[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
    t1 = np.cross(n, helper)
    t1 /= np.linalg.norm(t1, axis=1, keepdims=True)
    t2 = np.cross(n, t1)
    return t1, t2


def _triangles_at(rng, centers, normals, e_lo, e_hi, normal_jitter):
    """Near-equilateral triangles of log-uniform edge length in the tangent plane at `centers`."""
    n = centers.shape[0]
    e = np.exp(rng.uniform(np.log(e_lo), np.log(e_hi), size=n))
    rad = e / np.sqrt(3.0)
    rot = rng.uniform(0.0, 2.0 * np.pi, size=n)
    t1, t2 = _tangent_frame(normals)
    verts = np.empty((n, 3, 3))
    for k in range(3):
        ang = rot + k * (2.0 * np.pi / 3.0)
        verts[:, k, :] = centers + rad[:, None] * (np.cos(ang)[:, None] * t1 + np.sin(ang)[:, None] * t2)
    if normal_jitter > 0:
        verts += rng.normal(0.0, normal_jitter, size=(n, 3, 1)) * normals[:, None, :]
    flip = rng.random(n) < 0.5
    verts[flip] = verts[flip][:, [0, 2, 1], :]
    return verts


def tile_surfaces(rng, surfaces, n_faces, e_lo=0.01, e_hi=0.05, normal_jitter=0.005):
    """G(surfaces, N): faces allotted in proportion to area; jittered grid on rectangles,
    iid uniform directions on spheres.  Returns vertices [n_faces, 3, 3] float64."""
    areas = np.array([s.area for s in surfaces])
    share = areas / areas.sum() * n_faces
    counts = np.floor(share).astype(np.int64)
    rem = n_faces - counts.sum()
    order = np.argsort(-(share - counts))
    counts[order[:rem]] += 1
    out = []
    for s, n in zip(surfaces, counts):
        n = int(n)
        if n == 0:
            continue
        if isinstance(s, _Rect):
            cols = max(1, int(round(np.sqrt(n * s.a / s.b))))
            rows = int(np.ceil(n / cols))
            cells = rng.permutation(rows * cols)[:n]
            ci, ri = cells % cols, cells // cols
            cu, cv = s.a / cols, s.b / rows
            u = (ci + 0.5 + rng.uniform(-0.5, 0.5, size=n)) * cu
            v = (ri + 0.5 + rng.uniform(-0.5, 0.5, size=n)) * cv
            centers = s.origin + u[:, None] * s.eu + v[:, None] * s.ev
            normals = np.broadcast_to(s.normal, (n, 3)).copy()
        else:
            d = rng.normal(size=(n, 3))
            d /= np.linalg.norm(d, axis=1, keepdims=True)
            centers = s.center + s.radius * d
            normals = d
        out.append(_triangles_at(rng, centers, normals, e_lo, e_hi, normal_jitter))
    return np.concatenate(out, axis=0)


def smooth_noise_color(rng, pts):
    """Seeded smooth 3-D noise texture, per channel a 4-octave sum of sines, clipped to [0,1]."""
    col = np.empty((pts.shape[0], 3))
    norm = sum(2.0 ** (-o) for o in range(4))
    for ch in range(3):
        acc = np.zeros(pts.shape[0])
        for o in range(4):
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            ph = rng.uniform(0.0, 2.0 * np.pi)
            acc += 2.0 ** (-o) * np.sin(2.0 * np.pi * 0.35 * 2.0**o * (pts @ d) + ph)
        col[:, ch] = 0.5 + 0.5 * acc / norm
    return np.clip(col, 0.0, 1.0)


def _furnished_room(rng, L, Wd, H, n_boxes=20, n_spheres=20):
    surfaces = _room_rects(L, Wd, H)
    for _ in range(n_boxes):
        edges = rng.uniform(0.3, 1.2, size=3)
        cxy = np.array([rng.uniform(-L / 2 + 0.8, L / 2 - 0.8), rng.uniform(-Wd / 2 + 0.8, Wd / 2 - 0.8)])
        surfaces += _box_rects(cxy, -H / 2, edges, rng.uniform(0.0, 2.0 * np.pi))
    for _ in range(n_spheres):
        r = rng.uniform(0.15, 0.5)
        c = np.array([
            rng.uniform(-L / 2 + 0.6, L / 2 - 0.6),
            rng.uniform(-Wd / 2 + 0.6, Wd / 2 - 0.6),
            -H / 2 + r + rng.uniform(0.0, 1.0),
        ])
        surfaces.append(_Sphere(c, r))
    return surfaces


def _random_unit(rng):
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def _start_pose(rng, T_gt, trans=0.02, rot_deg=1.0):
    tau = np.concatenate([trans * _random_unit(rng), np.deg2rad(rot_deg) * _random_unit(rng)])
    return left_perturb(T_gt, tau)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _soup(verts):
    return _f32(verts.reshape(-1, 3))


# --------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------
def config0(n_faces=2000, seed=0):
    """Tiny single-view render fwd+bwd (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    cam = Camera(64, 48, 60.0, 60.0, 32.0, 24.0)
    cen = np.stack([rng.uniform(-1, 1, n_faces), rng.uniform(-1, 1, n_faces), rng.uniform(2, 4, n_faces)], axis=1)
    verts = cen[:, None, :] + rng.normal(0.0, 0.05, size=(n_faces, 3, 3))
    color = rng.uniform(0.0, 1.0, size=(n_faces * 3, 3))
    opacity = 1.0 / (1.0 + np.exp(-rng.normal(size=n_faces * 3)))
    jitter = verts + rng.normal(0.0, 0.01, size=verts.shape)
    T = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
    return Scene("config0_tiny", seed, cam, Params(sigma=1.0), _soup(verts), _f32(color), _f32(opacity), None,
                 [_f32(T)], [_f32(T)], pos_target=_soup(jitter), meta={"grad": "all+pose"})


def _room_scene(name, seed, cam, room, n_faces, furnished, cam_center, yaw):
    rng = np.random.default_rng(seed)
    L, Wd, H = room
    surfaces = _furnished_room(rng, L, Wd, H) if furnished else _room_rects(L, Wd, H)
    verts = tile_surfaces(rng, surfaces, n_faces)
    pts = verts.reshape(-1, 3)
    color = smooth_noise_color(rng, pts)
    opacity = rng.uniform(0.5, 1.0, size=pts.shape[0])
    T_gt = look_level(cam_center, yaw)
    T_start = _start_pose(rng, T_gt)
    return Scene(name, seed, cam, Params(sigma=0.5), _soup(verts), _f32(color), _f32(opacity), None,
                 [_f32(T_gt)], [_f32(T_start)], meta={"grad": "pose", "room": room}), rng


def config1(n_faces=100_000, seed=1):
    """TUM-shaped tracking frame (BASELINE.json configs[1])."""
    cam = Camera(640, 480, 525.0, 525.0, 319.5, 239.5)
    sc, _ = _room_scene("config1_tum", seed, cam, (5.0, 4.0, 3.0), n_faces, False, (0.3, -0.2, 0.0), 0.6)
    return sc


def config2(n_faces=500_000, seed=2):
    """Replica-shaped tracking frame (BASELINE.json configs[2]); the headline workload."""
    cam = Camera(1200, 680, 600.0, 600.0, 599.5, 339.5)
    sc, _ = _room_scene("config2_replica_track", seed, cam, (6.0, 5.0, 3.0), n_faces, True, (0.3, -0.2, 0.0), 0.6)
    return sc


def config3(n_faces=1_000_000, seed=3, n_views=8):
    """Replica-shaped mapping step over 8 keyframes (BASELINE.json configs[3])."""
    cam = Camera(1200, 680, 600.0, 600.0, 599.5, 339.5)
    sc, rng = _room_scene("config3_replica_map", seed, cam, (6.0, 5.0, 3.0), n_faces, True, (0.3, -0.2, 0.0), 0.6)
    p0 = np.array([-1.0, -0.6, 0.0])
    ang = rng.uniform(-0.3, 0.3)
    direc = np.array([np.cos(ang), np.sin(ang), 0.0])
    lat = np.array([-direc[1], direc[0], 0.0])
    yaw0, ph = ang + rng.uniform(-0.2, 0.2), rng.uniform(0.0, 2.0 * np.pi)
    poses = []
    for i in range(n_views):
        s = i / max(1, n_views - 1)
        p = p0 + 2.0 * s * direc + 0.15 * np.sin(2 * np.pi * s) * lat
        yaw = yaw0 + np.deg2rad(30.0) * np.sin(2 * np.pi * s + ph)
        poses.append(_f32(look_level(p, yaw)))
    sc.T_gt = poses
    sc.T_start = [p.copy() for p in poses]
    sc.pos_target = sc.pos
    sc.color_target = sc.color
    sc.pos = _f32(sc.pos.astype(np.float64) + rng.normal(0.0, 0.01, size=sc.pos.shape))
    sc.color = _f32(np.clip(sc.color.astype(np.float64) + rng.normal(0.0, 0.05, size=sc.color.shape), 0.0, 1.0))
    sc.meta["grad"] = "pos+color+opacity"
    return sc


def config4(n_faces=2_000_000, seed=4):
    """Depth-complexity stress test (BASELINE.json configs[4])."""
    cam = Camera(1200, 680, 600.0, 600.0, 599.5, 339.5)
    n_surf = n_faces // 2
    n_free = n_faces - n_surf
    sc, rng = _room_scene("config4_stress", seed, cam, (6.0, 5.0, 3.0), n_surf, True, (0.0, 0.0, 0.0), 0.6)
    L, Wd, H = 6.0, 5.0, 3.0
    cen = np.stack([rng.uniform(-L / 2, L / 2, n_free), rng.uniform(-Wd / 2, Wd / 2, n_free),
                    rng.uniform(-H / 2, H / 2, n_free)], axis=1)
    nrm = rng.normal(size=(n_free, 3))
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    fverts = _triangles_at(rng, cen, nrm, 0.01, 0.10, 0.0)
    fpts = fverts.reshape(-1, 3)
    fcol = smooth_noise_color(rng, fpts)
    fop = rng.uniform(0.05, 0.4, size=fpts.shape[0])
    sc.pos = np.concatenate([sc.pos, _f32(fpts)], axis=0)
    sc.color = np.concatenate([sc.color, _f32(fcol)], axis=0)
    sc.opacity = np.concatenate([sc.opacity, _f32(fop)], axis=0)
    sc.pos_target = _f32(sc.pos.astype(np.float64) + rng.normal(0.0, 0.01, size=sc.pos.shape))
    sc.T_start = [sc.T_gt[0].copy()]
    sc.meta["grad"] = "all+pose"
    return sc


CONFIGS = [config0, config1, config2, config3, config4]


def make_config(i, **kw):
    return CONFIGS[i](**kw)


def index_soup(scene):
    """Same scene with an explicit faces[M][3] array (exercises the general indexed path)."""
    M = scene.M
    faces = np.arange(3 * M, dtype=np.int32).reshape(M, 3)
    return faces
