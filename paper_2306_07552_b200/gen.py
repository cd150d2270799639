"""Seeded synthetic workloads for the batch RGBD renderer (configs 0-4 of BASELINE.json).

These stand in for the paper's ReplicaCAD scenes, YCB objects, Fetch robot and Rearrange-Easy
episodes (PAPER.md:143,441 -- not in the container) and take only their *shape*: a 128x128 (or
64x64) 90-degree-FoV head camera at 1.2 m, one static indoor mesh shared by many
environments, a few tens of small movable objects and one articulated robot per
environment.  Recipe: SURVEY.md section 8(d), restated in DESIGN.md.

This module is the ONLY thing the oracle tests and the CUDA tests share.  It holds none of the
renderer's arithmetic (no projection, no snapping, no rasterisation): it only builds meshes, camera
poses and instance transforms as float32 / uint8 / uint32 / int32 numpy arrays.  It imports numpy and
nothing else of this package.

Randomness: numpy Philox (counter-based), key = (1000 + config, stream).  Environment n draws from
stream n, scene s from stream 2**40 + s, so any subset of environments is reproducible on its own.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

__all__ = ["Mesh", "Workload", "make_config", "CONFIG_SHAPES", "icosphere", "box_mesh"]

SCENE_STREAM0 = 2 ** 40


@dataclass
class Mesh:
    positions: np.ndarray  # [nv,3] float32
    colors: np.ndarray     # [nv,3] uint8
    indices: np.ndarray    # [nt,3] uint32

    @property
    def nv(self) -> int:
        return int(self.positions.shape[0])

    @property
    def nt(self) -> int:
        return int(self.indices.shape[0])


@dataclass
class Robot:
    """Description of an articulated robot for the scene-graph update (N12): data only.  Link l hangs off
    link parent[l] < l (-1 = the base); origin[l] is the joint frame in the parent's frame (3x4), joint_type 0
    fixed / 1 revolute / 2 prismatic about or along the unit vector axis[l]."""
    parent: np.ndarray       # [L] int32
    joint_type: np.ndarray   # [L] int32
    axis: np.ndarray         # [L,3] float32
    origin: np.ndarray       # [L,12] float32
    camera_link: int         # link the head camera is mounted on (-1 = the base)
    cam_mount: np.ndarray    # [12] float32: camera frame in that link's frame
    ee_link: int             # end-effector link (carries the held object)


@dataclass
class Workload:
    name: str
    width: int
    height: int
    fx: float
    fy: float
    znear: float
    zfar: float
    static_meshes: List[Mesh]
    dyn_meshes: List[Mesh]
    env_scene: np.ndarray   # [N] int32
    cam_pose: np.ndarray    # [N,16] float32, camera-to-world, row-major
    inst_mesh: np.ndarray   # [N,K] int32, -1 = empty slot
    inst_xform: np.ndarray  # [N,K,16] float32, object-to-world, row-major
    depth_only: bool = False
    env_ids: Optional[np.ndarray] = None  # which environments of the full config these are
    meta: Dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.env_scene.shape[0])

    @property
    def K(self) -> int:
        return int(self.inst_mesh.shape[1])

    def tris_per_env(self) -> np.ndarray:
        snt = np.array([m.nt for m in self.static_meshes], dtype=np.int64)
        dnt = np.array([m.nt for m in self.dyn_meshes] + [0], dtype=np.int64)
        return snt[self.env_scene] + dnt[self.inst_mesh].sum(axis=1)

    def subset(self, sel: Sequence[int]) -> "Workload":
        sel = np.asarray(sel, dtype=np.int64)
        ids = self.env_ids if self.env_ids is not None else np.arange(self.N)
        return Workload(self.name, self.width, self.height, self.fx, self.fy, self.znear, self.zfar,
                        self.static_meshes, self.dyn_meshes,
                        np.ascontiguousarray(self.env_scene[sel]),
                        np.ascontiguousarray(self.cam_pose[sel]),
                        np.ascontiguousarray(self.inst_mesh[sel]),
                        np.ascontiguousarray(self.inst_xform[sel]),
                        self.depth_only, ids[sel], dict(self.meta))


# name, N, W, H, n_scenes, static tris/scene, depth_only
CONFIG_SHAPES = {
    0: ("cfg0 tiny 4 envs 64x64 RGBD", 4, 64, 64, 1, 200, False),
    1: ("cfg1 256 envs 128x128 RGBD, 1 scene x 50k", 256, 128, 128, 1, 50_000, False),
    2: ("cfg2 1024 envs 128x128 RGBD, 4 scenes x 50k", 1024, 128, 128, 4, 50_000, False),
    3: ("cfg3 4096 envs 128x128 RGBD, 4 scenes x 500k", 4096, 128, 128, 4, 500_000, False),
    4: ("cfg4 16384 envs 64x64 depth-only, 8 scenes x 100k", 16384, 64, 64, 8, 100_000, True),
}


def _rng(cfg: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[1000 + cfg, stream]))


# ----------------------------------------------------------------------------------------------
# mesh primitives
# ----------------------------------------------------------------------------------------------

def _grid_patch(origin, du, dv, nu, nv):
    """(nu x nv)-cell planar grid: vertices origin + i*du/nu + j*dv/nv, 2 triangles per cell."""
    origin = np.asarray(origin, np.float64)
    du = np.asarray(du, np.float64)
    dv = np.asarray(dv, np.float64)
    i, j = np.meshgrid(np.arange(nu + 1), np.arange(nv + 1), indexing="ij")
    p = origin + (i[..., None] / nu) * du + (j[..., None] / nv) * dv
    p = p.reshape(-1, 3)
    vid = (i * (nv + 1) + j)
    a = vid[:-1, :-1].ravel()
    b = vid[1:, :-1].ravel()
    c = vid[1:, 1:].ravel()
    d = vid[:-1, 1:].ravel()
    # alternate the diagonal in a checkerboard so neither direction is favoured
    par = ((i[:-1, :-1] + j[:-1, :-1]) & 1).ravel().astype(bool)
    t0 = np.where(par[:, None], np.stack([a, b, d], 1), np.stack([a, b, c], 1))
    t1 = np.where(par[:, None], np.stack([b, c, d], 1), np.stack([a, c, d], 1))
    tri = np.empty((2 * nu * nv, 3), np.int64)
    tri[0::2] = t0
    tri[1::2] = t1
    return p, tri


def box_mesh(dims, sub, rng: Optional[np.random.Generator] = None, base_color=None,
             color_noise: int = 24) -> Mesh:
    """Axis-aligned box centred at the origin, faces grid-subdivided (a,b,c) cells along x,y,z,
    vertices shared across faces: 4(ab+bc+ca) triangles, 2(ab+bc+ca)+2 vertices."""
    a, b, c = (int(s) for s in sub)
    n = (a, b, c)
    faces = []
    # (fixed axis, side) -> grid over the other two axes, on the integer surface lattice
    for ax in range(3):
        u, v = (ax + 1) % 3, (ax + 2) % 3
        for side in (0, 1):
            iu, iv = np.meshgrid(np.arange(n[u] + 1), np.arange(n[v] + 1), indexing="ij")
            lat = np.zeros(iu.shape + (3,), np.int64)
            lat[..., ax] = side * n[ax]
            lat[..., u] = iu
            lat[..., v] = iv
            q00 = lat[:-1, :-1].reshape(-1, 3)
            q10 = lat[1:, :-1].reshape(-1, 3)
            q11 = lat[1:, 1:].reshape(-1, 3)
            q01 = lat[:-1, 1:].reshape(-1, 3)
            if side == 0:  # keep a consistent outward winding (not relied upon by the renderer)
                q10, q01 = q01, q10
            cell = np.stack([q00, q10, q11, q00, q11, q01], 1).reshape(-1, 3, 3)
            faces.append(cell)
    corners = np.concatenate(faces, 0)  # [nt,3 verts,3 lattice coords]
    flat = corners.reshape(-1, 3)
    key = (flat[:, 0] * (b + 1) + flat[:, 1]) * (c + 1) + flat[:, 2]
    uniq, first, inv = np.unique(key, return_index=True, return_inverse=True)
    # keep vertices in first-use order so consecutive triangles reference nearby vertex ids
    order = np.argsort(first, kind="stable")
    rank = np.empty_like(order)
    rank[order] = np.arange(order.size)
    idx = rank[inv].reshape(-1, 3)
    lat_u = flat[first[order]]
    dims = np.asarray(dims, np.float64)
    pos = (lat_u / np.array([a, b, c], np.float64) - 0.5) * dims
    nvv = pos.shape[0]
    if base_color is None:
        base_color = np.array([160, 160, 160])
    if rng is not None and color_noise > 0:
        col = np.clip(np.asarray(base_color)[None, :] + rng.integers(-color_noise, color_noise + 1, (nvv, 3)), 0, 255)
    else:
        col = np.broadcast_to(np.asarray(base_color)[None, :], (nvv, 3))
    return Mesh(pos.astype(np.float32), col.astype(np.uint8), idx.astype(np.uint32))


def icosphere(freq: int, rng: Optional[np.random.Generator] = None) -> Mesh:
    """Class-I geodesic sphere of frequency f on the unit sphere: 20 f^2 triangles, 10 f^2 + 2 vertices."""
    t = (1.0 + math.sqrt(5.0)) / 2.0
    base = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0], [0, -1, t], [0, 1, t], [0, -1, -t],
                     [0, 1, -t], [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], np.float64)
    faces = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2),
             (10, 7, 6), (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5),
             (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    f = int(freq)
    keys: Dict[Tuple[int, ...], int] = {}
    verts: List[np.ndarray] = []
    tris: List[Tuple[int, int, int]] = []

    def vid(fa, i, j):
        # integer barycentric weights over the 12 base vertices identify shared vertices exactly
        k = f - i - j
        w = [0] * 12
        w[fa[0]] += k
        w[fa[1]] += i
        w[fa[2]] += j
        key = tuple(w)
        if key not in keys:
            keys[key] = len(verts)
            p = (k * base[fa[0]] + i * base[fa[1]] + j * base[fa[2]]) / f
            verts.append(p / np.linalg.norm(p))
        return keys[key]

    for fa in faces:
        for i in range(f):
            for j in range(f - i):
                tris.append((vid(fa, i, j), vid(fa, i + 1, j), vid(fa, i, j + 1)))
                if i + j < f - 1:
                    tris.append((vid(fa, i + 1, j), vid(fa, i + 1, j + 1), vid(fa, i, j + 1)))
    pos = np.array(verts)
    if rng is None:
        col = np.full((pos.shape[0], 3), 200, np.int64)
    else:
        # smooth colour field + noise so interpolation is visible
        col = np.clip(128 + 100 * pos + rng.integers(-20, 21, pos.shape), 0, 255)
    return Mesh(pos.astype(np.float32), col.astype(np.uint8), np.array(tris, np.uint32))


def _concat(meshes: Sequence[Mesh]) -> Mesh:
    pos, col, idx, off = [], [], [], 0
    for m in meshes:
        pos.append(m.positions)
        col.append(m.colors)
        idx.append(m.indices.astype(np.int64) + off)
        off += m.nv
    return Mesh(np.concatenate(pos).astype(np.float32), np.concatenate(col).astype(np.uint8),
                np.concatenate(idx).astype(np.uint32))


def _placed(m: Mesh, R: np.ndarray, t: np.ndarray) -> Mesh:
    p = m.positions.astype(np.float64) @ R.T + t
    return Mesh(p.astype(np.float32), m.colors, m.indices)


def _roty(a):
    c, s = np.cos(a), np.sin(a)
    return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]], np.float64)


def _rotx(a):
    c, s = np.cos(a), np.sin(a)
    return np.array([[1, 0, 0], [0, c, -s], [0, s, c]], np.float64)


# ----------------------------------------------------------------------------------------------
# apartment-like static scene
# ----------------------------------------------------------------------------------------------

FOOT = 12.0     # footprint side, m
ROOM = 3.0      # 4x4 rooms
HEIGHT = 3.0
CELL = 0.5      # room-shell grid cell, m
DOOR_W, DOOR_H = 0.9, 2.1
N_BOXES = 300


def _shell(rng) -> Tuple[List[Mesh], List[Tuple[float, float, float, float]]]:
    """Floor, ceiling, outer walls and interior walls with door gaps.  Returns the patches and the
    interior/outer wall segments (x0,z0,x1,z1) that block movement (door gaps excluded)."""
    patches: List[Mesh] = []
    segs: List[Tuple[float, float, float, float]] = []

    def add(origin, du, dv, base):
        lu = float(np.linalg.norm(du))
        lv = float(np.linalg.norm(dv))
        nu = max(1, int(math.ceil(lu / CELL - 1e-9)))
        nv = max(1, int(math.ceil(lv / CELL - 1e-9)))
        p, tri = _grid_patch(origin, du, dv, nu, nv)
        col = np.clip(np.asarray(base)[None, :] + rng.integers(-18, 19, (p.shape[0], 3)), 0, 255)
        patches.append(Mesh(p.astype(np.float32), col.astype(np.uint8), tri.astype(np.uint32)))

    add([0, 0, 0], [FOOT, 0, 0], [0, 0, FOOT], [150, 120, 90])        # floor
    add([0, HEIGHT, 0], [FOOT, 0, 0], [0, 0, FOOT], [225, 225, 220])  # ceiling
    for (o, d) in (([0, 0, 0], [FOOT, 0, 0]), ([0, 0, FOOT], [FOOT, 0, 0]),
                   ([0, 0, 0], [0, 0, FOOT]), ([FOOT, 0, 0], [0, 0, FOOT])):
        add(o, d, [0, HEIGHT, 0], [200, 205, 210])
        segs.append((o[0], o[2], o[0] + d[0], o[2] + d[2]))
    nr = int(round(FOOT / ROOM))
    g0 = (ROOM - DOOR_W) / 2.0
    for i in range(1, nr):          # interior walls at x = i*ROOM (run along z) and z = i*ROOM (run along x)
        for j in range(nr):
            base = rng.integers(150, 235, 3)
            for along_z in (True, False):
                def P(s, y):  # point at distance s along the segment
                    return [i * ROOM, y, j * ROOM + s] if along_z else [j * ROOM + s, y, i * ROOM]
                def D(s):
                    return [0, 0, s] if along_z else [s, 0, 0]
                add(P(0, 0), D(g0), [0, HEIGHT, 0], base)
                add(P(g0 + DOOR_W, 0), D(g0), [0, HEIGHT, 0], base)
                add(P(g0, DOOR_H), D(DOOR_W), [0, HEIGHT - DOOR_H, 0], base)
                for (s0, s1) in ((0.0, g0), (g0 + DOOR_W, ROOM)):
                    a, b = P(s0, 0), P(s1, 0)
                    segs.append((a[0], a[2], b[0], b[2]))
    return patches, segs


def _tri_count(sub):
    a, b, c = sub
    return 4 * (a * b + b * c + c * a)


def _fit_sub(dims, target):
    """Largest near-isotropic subdivision of a box with at most `target` triangles."""
    best = (1, 1, 1)
    h = max(dims)
    while h > 1e-3:
        sub = tuple(max(1, int(round(d / h))) for d in dims)
        if _tri_count(sub) > target:
            break
        best = sub
        h *= 0.97
    return best


def make_scene(cfg: int, scene: int, n_tris: int) -> Tuple[Mesh, Dict]:
    """One procedural apartment: room shell (~5k triangles) + 300 furniture boxes, emitted box by box
    (so runs of 256 consecutive triangles are spatially compact), exactly n_tris triangles."""
    rng = _rng(cfg, SCENE_STREAM0 + scene)
    shell, segs = _shell(rng)
    shell_tris = sum(m.nt for m in shell)
    # furniture: footprint sides U[0.2,0.8] m, height U[0.3,2] m (continuous -> no two coplanar tops),
    # yaw U[0,2pi).  (Sides up to 2 m, as first sketched in SURVEY.md 8(d), would cover the 144 m^2 floor
    # almost three times over and leave no free space for cameras.)
    sx = rng.uniform(0.2, 0.8, N_BOXES)
    sz = rng.uniform(0.2, 0.8, N_BOXES)
    sy = rng.uniform(0.3, 2.0, N_BOXES)
    cx = rng.uniform(0.4, FOOT - 0.4, N_BOXES)
    cz = rng.uniform(0.4, FOOT - 0.4, N_BOXES)
    yaw = rng.uniform(0.0, 2 * math.pi, N_BOXES)
    budget = n_tris - shell_tris
    per_box = budget // N_BOXES
    subs = [list(_fit_sub((sx[i], sy[i], sz[i]), per_box)) for i in range(N_BOXES)]
    total = sum(_tri_count(s) for s in subs)
    # spend the remainder by refining boxes round-robin along their coarsest axis
    progress = True
    while progress:
        progress = False
        for i in range(N_BOXES):
            dims = (sx[i], sy[i], sz[i])
            ax = int(np.argmax([dims[k] / subs[i][k] for k in range(3)]))
            trial = list(subs[i])
            trial[ax] += 1
            inc = _tri_count(trial) - _tri_count(subs[i])
            if total + inc <= budget:
                subs[i] = trial
                total += inc
                progress = True
    parts: List[Mesh] = list(shell)
    for i in range(N_BOXES):
        base = rng.integers(40, 230, 3)
        m = box_mesh((sx[i], sy[i], sz[i]), subs[i], rng, base)
        parts.append(_placed(m, _roty(yaw[i]), np.array([cx[i], sy[i] / 2 + 0.002, cz[i]])))
    # fill the last few triangles with small 12-triangle cubes, then single decal triangles
    rest = budget - total
    while rest >= 12:
        d = rng.uniform(0.08, 0.2)
        m = box_mesh((d, d, d), (1, 1, 1), rng, rng.integers(40, 230, 3))
        parts.append(_placed(m, _roty(rng.uniform(0, 2 * math.pi)),
                             np.array([rng.uniform(0.5, FOOT - 0.5), d / 2 + 0.003, rng.uniform(0.5, FOOT - 0.5)])))
        rest -= 12
    for _ in range(rest):
        c = np.array([rng.uniform(0.5, FOOT - 0.5), rng.uniform(0.5, 2.5), rng.uniform(0.5, FOOT - 0.5)])
        p = c[None, :] + rng.uniform(-0.15, 0.15, (3, 3))
        parts.append(Mesh(p.astype(np.float32), rng.integers(0, 256, (3, 3)).astype(np.uint8),
                          np.array([[0, 1, 2]], np.uint32)))
    mesh = _concat(parts)
    assert mesh.nt == n_tris, (mesh.nt, n_tris)
    info = dict(boxes=np.stack([cx, cz, sx / 2, sz / 2, yaw, sy], 1), segs=np.array(segs, np.float64),
                shell_tris=shell_tris)
    return mesh, info


def _dist_boxes(px, pz, boxes):
    """XZ distance from points [...,] to every oriented box footprint [B,6] -> [..., B] (0 inside)."""
    cx, cz, hx, hz, yaw = (boxes[:, k] for k in range(5))
    dx = px[..., None] - cx
    dz = pz[..., None] - cz
    c, s = np.cos(yaw), np.sin(yaw)
    # world -> box frame (inverse of rotation about +Y by yaw)
    lx = c * dx - s * dz
    lz = s * dx + c * dz
    ox = np.maximum(np.abs(lx) - hx, 0.0)
    oz = np.maximum(np.abs(lz) - hz, 0.0)
    return np.hypot(ox, oz)


def _dist_segs(px, pz, segs):
    x0, z0, x1, z1 = (segs[:, k] for k in range(4))
    ex, ez = x1 - x0, z1 - z0
    L2 = ex * ex + ez * ez
    t = np.clip(((px[..., None] - x0) * ex + (pz[..., None] - z0) * ez) / L2, 0.0, 1.0)
    return np.hypot(px[..., None] - (x0 + t * ex), pz[..., None] - (z0 + t * ez))


# ----------------------------------------------------------------------------------------------
# robot proxy: 5 box links, 400 triangles each (2 x 6 x 11 cells)
# ----------------------------------------------------------------------------------------------

LINK_DIMS = [(0.5, 0.4, 0.5), (0.3, 0.6, 0.3), (0.10, 0.10, 0.36), (0.09, 0.09, 0.32), (0.08, 0.08, 0.26)]
LINK_SUBS = [(6, 2, 11), (6, 11, 2), (2, 6, 11), (2, 6, 11), (2, 6, 11)]


def _link_meshes(cfg: int) -> List[Mesh]:
    rng = _rng(cfg, SCENE_STREAM0 + 1000)
    cols = [(70, 70, 80), (90, 90, 110), (220, 120, 40), (230, 200, 60), (200, 60, 60)]
    return [box_mesh(d, s, rng, np.array(c)) for d, s, c in zip(LINK_DIMS, LINK_SUBS, cols)]


def _mat4(R, t):
    M = np.zeros(R.shape[:-2] + (4, 4), np.float64)
    M[..., :3, :3] = R
    M[..., :3, 3] = t
    M[..., 3, 3] = 1.0
    return M


def _robot_links(cam_xz, yaw, u):
    """Link-to-world transforms [n,5,4,4] for robots whose head camera sits at (x,1.2,z), heading yaw.
    u: [n,4] uniforms -> shoulder yaw offset and three joint pitches."""
    n = cam_xz.shape[0]
    c, s = np.cos(yaw), np.sin(yaw)
    Ry = np.zeros((n, 3, 3))
    Ry[:, 0, 0] = c; Ry[:, 0, 2] = s; Ry[:, 1, 1] = 1; Ry[:, 2, 0] = -s; Ry[:, 2, 2] = c
    base_o = np.stack([cam_xz[:, 0], np.zeros(n), cam_xz[:, 1]], 1)   # robot frame origin on the floor
    out = np.zeros((n, 5, 4, 4))

    def world(local):
        return base_o + np.einsum("nij,nj->ni", Ry, local)

    # robot frame: -Z is forward (the camera looks along -Z), +X right
    out[:, 0] = _mat4(Ry, world(np.tile([0.0, 0.30, 0.10], (n, 1))))          # base, y in [0.1,0.5]
    out[:, 1] = _mat4(Ry, world(np.tile([0.0, 0.80, 0.22], (n, 1))))          # torso behind the camera
    sh_yaw = (u[:, 0] - 0.5) * math.radians(40.0)
    a1 = (u[:, 1] - 0.5) * math.radians(60.0)
    a2 = a1 + (u[:, 2] - 0.5) * math.radians(120.0)
    a3 = a2 + (u[:, 3] - 0.5) * math.radians(120.0)
    joint = np.tile([0.17, 1.02, -0.05], (n, 1))                                # shoulder, robot frame
    for li, (ang, L) in enumerate(((a1, 0.36), (a2, 0.32), (a3, 0.26))):
        # link axis: local -Z pitched by ang about X then yawed by sh_yaw about Y (robot frame)
        cy, sy = np.cos(sh_yaw), np.sin(sh_yaw)
        cp, sp = np.cos(ang), np.sin(ang)
        Rl = np.zeros((n, 3, 3))
        # R = Ry(sh_yaw) @ Rx(ang)
        Rl[:, 0, 0] = cy; Rl[:, 0, 1] = sy * sp; Rl[:, 0, 2] = sy * cp
        Rl[:, 1, 1] = cp; Rl[:, 1, 2] = -sp
        Rl[:, 2, 0] = -sy; Rl[:, 2, 1] = cy * sp; Rl[:, 2, 2] = cy * cp
        fwd = -Rl[:, :, 2]
        centre = joint + fwd * (L / 2)
        out[:, 2 + li] = _mat4(np.einsum("nij,njk->nik", Ry, Rl), world(centre))
        joint = joint + fwd * L
    return out


def _rand_rot(u):
    """Uniform random rotations from [n,3] uniforms (Shoemake)."""
    u1, u2, u3 = u[:, 0], u[:, 1], u[:, 2]
    q = np.stack([np.sqrt(1 - u1) * np.sin(2 * np.pi * u2), np.sqrt(1 - u1) * np.cos(2 * np.pi * u2),
                  np.sqrt(u1) * np.sin(2 * np.pi * u3), np.sqrt(u1) * np.cos(2 * np.pi * u3)], 1)
    x, y, z, w = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((u.shape[0], 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


# ----------------------------------------------------------------------------------------------
# configs
# ----------------------------------------------------------------------------------------------

def _cam_pose(pos, yaw, pitch):
    """camera-to-world: camera looks along its local -Z, +Y up; yaw about world +Y, then pitch about
    the camera's +X (negative pitch looks down)."""
    n = pos.shape[0]
    M = np.zeros((n, 4, 4))
    for k in range(n):
        M[k, :3, :3] = _roty(yaw[k]) @ _rotx(pitch[k])
    M[:, :3, 3] = pos
    M[:, 3, 3] = 1
    return M


def _config0(env_ids: np.ndarray) -> Workload:
    name, N, W, H, _, nt, _ = CONFIG_SHAPES[0]
    rs = _rng(0, SCENE_STREAM0)
    pos = rs.uniform(0, 1, (nt * 3, 3)) * np.array([10.0, 3.0, 10.0])
    col = rs.integers(0, 256, (nt * 3, 3))
    static = Mesh(pos.astype(np.float32), col.astype(np.uint8), np.arange(nt * 3, dtype=np.uint32).reshape(nt, 3))
    cube = box_mesh((1.0, 1.0, 1.0), (1, 1, 1), rs, np.array([128, 128, 128]), color_noise=120)
    n = len(env_ids)
    cam = np.zeros((n, 4, 4))
    xf = np.zeros((n, 2, 4, 4))
    for r, e in enumerate(env_ids):
        g = _rng(0, int(e))
        p = np.array([g.uniform(1, 9), 1.2, g.uniform(1, 9)])
        cam[r] = _cam_pose(p[None], np.array([g.uniform(0, 2 * math.pi)]), np.array([0.0]))[0]
        for k in range(2):
            yaw = g.uniform(0, 2 * math.pi)
            t = g.uniform(0, 1, 3) * np.array([10.0, 3.0, 10.0])
            xf[r, k] = _mat4(_roty(yaw) * 0.5, t)
    return Workload(name, W, H, 1.0, 1.0, 0.1, 20.0, [static], [cube],
                    np.zeros(n, np.int32), cam.reshape(n, 16).astype(np.float32),
                    np.zeros((n, 2), np.int32), xf.reshape(n, 2, 16).astype(np.float32),
                    False, np.asarray(env_ids))


_scene_cache: Dict[Tuple[int, int, int], Tuple[Mesh, Dict]] = {}


def _scenes(cfg: int, n_scenes: int, n_tris: int):
    out = []
    for s in range(n_scenes):
        # configs 1 and 2 share the generator; config 2 runs it with 4 seeds (its own key)
        k = (cfg, s, n_tris)
        if k not in _scene_cache:
            _scene_cache[k] = make_scene(cfg, s, n_tris)
        out.append(_scene_cache[k])
    return out


N_CAND = 48      # rejection-sampling candidates per camera, drawn from the env stream
N_CAND_OBJ = 8   # ... and per object


def _config_rooms(cfg: int, env_ids: np.ndarray) -> Workload:
    name, N, W, H, n_scenes, n_tris, depth_only = CONFIG_SHAPES[cfg]
    scenes = _scenes(cfg, n_scenes, n_tris)
    lrng = _rng(cfg, SCENE_STREAM0 + 2000)
    links = _link_meshes(cfg)
    if cfg == 4:
        objs = [icosphere(5, lrng)]                       # 500 triangles
        obj_slots = [0] * 10
    elif cfg == 3:
        objs = [icosphere(7, lrng), box_mesh((0.08, 0.15, 0.25), (2, 4, 7), lrng, np.array([60, 140, 200]))]
        obj_slots = [0] * 20 + [1] * 20                   # 20 icospheres + 20 boxes of 200 triangles
    else:
        objs = [icosphere(7, lrng)]                       # 980 triangles
        obj_slots = [0] * 20
    dyn = objs + links
    n_obj = len(obj_slots)
    K = n_obj + 5
    n = len(env_ids)
    # fixed-size uniform blocks per env (stream = env id); everything after is vectorised over envs
    n_u = 1 + 3 * N_CAND + 6 + n_obj * (2 * N_CAND_OBJ + 6)
    U = np.empty((n, n_u))
    for r, e in enumerate(env_ids):
        U[r] = _rng(cfg, int(e)).random(n_u)
    env_scene = np.minimum((U[:, 0] * n_scenes).astype(np.int32), n_scenes - 1)
    o = 1
    cand = U[:, o:o + 2 * N_CAND].reshape(n, N_CAND, 2); o += 2 * N_CAND
    o += N_CAND  # reserved
    cam_u = U[:, o:o + 6]; o += 6
    obj_u = U[:, o:].reshape(n, n_obj, 2 * N_CAND_OBJ + 6)

    cam_xz = np.zeros((n, 2))
    obj_pos = np.zeros((n, n_obj, 3))
    obj_r = np.zeros((n, n_obj))
    for s in range(n_scenes):
        sel = np.nonzero(env_scene == s)[0]
        if sel.size == 0:
            continue
        boxes, segs = scenes[s][1]["boxes"], scenes[s][1]["segs"]
        # camera: first candidate >= 0.25 m from every wall segment and furniture footprint
        px = 0.3 + cand[sel, :, 0] * (FOOT - 0.6)
        pz = 0.3 + cand[sel, :, 1] * (FOOT - 0.6)
        clear = np.minimum(_dist_boxes(px, pz, boxes).min(-1), _dist_segs(px, pz, segs).min(-1))
        ok = clear >= 0.25
        first = np.where(ok.any(1), ok.argmax(1), clear.argmax(1))  # (fallback: the clearest candidate)
        cam_xz[sel, 0] = px[np.arange(sel.size), first]
        cam_xz[sel, 1] = pz[np.arange(sel.size), first]
        # objects: radius U[0.04,0.12]; half rest on the floor in free space, half on a furniture top
        ou = obj_u[sel]
        r = 0.04 + 0.08 * ou[:, :, 0]
        on_box = ou[:, :, 1] < 0.5
        cx = 0.3 + ou[:, :, 6:6 + N_CAND_OBJ] * (FOOT - 0.6)
        cz = 0.3 + ou[:, :, 6 + N_CAND_OBJ:6 + 2 * N_CAND_OBJ] * (FOOT - 0.6)
        okf = (_dist_boxes(cx, cz, boxes).min(-1) >= r[..., None] + 0.02) & \
              (_dist_segs(cx, cz, segs).min(-1) >= r[..., None] + 0.02)
        ff = np.where(okf.any(-1), okf.argmax(-1), 0)
        ii, jj = np.meshgrid(np.arange(sel.size), np.arange(n_obj), indexing="ij")
        fx_, fz_ = cx[ii, jj, ff], cz[ii, jj, ff]
        bi = np.minimum((ou[:, :, 2] * N_BOXES).astype(np.int64), N_BOXES - 1)
        bx = boxes[bi]
        lx = (ou[:, :, 3] - 0.5) * 2 * np.maximum(bx[..., 2] - r, 0.0)
        lz = (ou[:, :, 4] - 0.5) * 2 * np.maximum(bx[..., 3] - r, 0.0)
        cb, sb = np.cos(bx[..., 4]), np.sin(bx[..., 4])
        tx = bx[..., 0] + cb * lx + sb * lz
        tz = bx[..., 1] - sb * lx + cb * lz
        obj_pos[sel, :, 0] = np.where(on_box, tx, fx_)
        obj_pos[sel, :, 2] = np.where(on_box, tz, fz_)
        obj_pos[sel, :, 1] = np.where(on_box, bx[..., 5] + 0.002 + r, r)
        obj_r[sel] = r
    yaw = cam_u[:, 0] * 2 * math.pi
    pitch = -cam_u[:, 1] * math.radians(25.0)
    cam_p = np.stack([cam_xz[:, 0], np.full(n, 1.2), cam_xz[:, 1]], 1)
    cam = _cam_pose(cam_p, yaw, pitch)
    xf = np.zeros((n, K, 4, 4))
    R = _rand_rot(obj_u[:, :, 3:6].reshape(-1, 3)).reshape(n, n_obj, 3, 3)
    for j, slot_mesh in enumerate(obj_slots):
        scale = obj_r[:, j] if slot_mesh == 0 else np.ones(n)   # icospheres are unit spheres
        xf[:, j] = _mat4(R[:, j] * scale[:, None, None], obj_pos[:, j] + (0 if slot_mesh == 0 else np.array([0, 0.1, 0])))
    xf[:, n_obj:] = _robot_links(cam_xz, yaw, cam_u[:, 2:6])
    inst_mesh = np.tile(np.array(obj_slots + [len(objs) + k for k in range(5)], np.int32), (n, 1))
    return Workload(name, W, H, 1.0, 1.0, 0.1, 20.0, [m for m, _ in scenes], dyn, env_scene,
                    cam.reshape(n, 16).astype(np.float32), inst_mesh,
                    xf.reshape(n, K, 16).astype(np.float32), depth_only, np.asarray(env_ids),
                    dict(scene_info=[i for _, i in scenes]))


def make_config(cfg: int, n_envs: Optional[int] = None, env_ids: Optional[Sequence[int]] = None,
                beyond: bool = False) -> Workload:
    """Workload `cfg` (0-4) of BASELINE.json.  n_envs: first n environments; env_ids: explicit subset
    (each environment is generated from its own stream, so a subset equals the same rows of the full
    config).  beyond: allow environment ids past the config's N -- more environments of the same
    recipe, e.g. rank r of a weak-scaling run renders ids r*N .. (r+1)*N - 1."""
    if cfg not in CONFIG_SHAPES:
        raise ValueError(f"unknown config {cfg}")
    N = CONFIG_SHAPES[cfg][1]
    if env_ids is None:
        env_ids = np.arange(N if n_envs is None else min(n_envs, N))
    env_ids = np.asarray(env_ids, np.int64)
    if env_ids.size and (env_ids.min() < 0 or (env_ids.max() >= N and not beyond) or env_ids.max() >= 2 ** 40):
        raise ValueError("env id out of range")
    return _config0(env_ids) if cfg == 0 else _config_rooms(cfg, env_ids)


def robot_proxy() -> Robot:
    """The 5-link robot proxy of the room configs as a kinematic chain (stands in for the paper's Fetch: mobile
    base, lift, arm, head camera): base box -> torso (prismatic lift along +Y) -> upper arm
    (revolute about X at the shoulder) -> forearm (revolute about X at the elbow) -> hand (revolute about Y);
    the head camera sits on the torso at 1.2 m and looks along -Z, pitched down a little."""
    def T(x, y, z):
        return [1, 0, 0, x, 0, 1, 0, y, 0, 0, 1, z]
    parent = np.array([-1, 0, 1, 2, 3], np.int32)
    joint_type = np.array([0, 2, 1, 1, 1], np.int32)
    axis = np.array([[0, 1, 0], [0, 1, 0], [1, 0, 0], [1, 0, 0], [0, 1, 0]], np.float32)
    origin = np.array([T(0, 0.25, 0), T(0, 0.45, 0), T(0.2, 0.25, -0.15), T(0, 0, -0.35), T(0, 0, -0.3)], np.float32)
    p = np.float32(-0.2)   # camera pitch about X
    mount = np.array([1, 0, 0, 0, 0, np.cos(p), -np.sin(p), 0.5, 0, np.sin(p), np.cos(p), -0.1], np.float32)
    return Robot(parent, joint_type, axis, origin, 1, mount, 4)


def robot_states(robot: Robot, n: int, seed: int = 0):
    """Seeded per-environment robot state: base_pose [n,3] = (x, z, yaw), joint_pos [n,L], held_slot [n] (-1 = hand
    empty), held_xform [n,12] (held object in the end-effector frame)."""
    g = _rng(9, seed)
    L = len(robot.parent)
    base = np.stack([g.uniform(1, 11, n), g.uniform(1, 11, n), g.uniform(-np.pi, np.pi, n)], axis=1).astype(np.float32)
    joints = g.uniform(-1.2, 1.2, (n, L)).astype(np.float32)
    joints[:, robot.joint_type == 2] = g.uniform(0.0, 0.4, (n, int((robot.joint_type == 2).sum()))).astype(np.float32)
    held = np.where(g.uniform(0, 1, n) < 0.5, 0, -1).astype(np.int32)
    hx = np.tile(np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, -0.12], np.float32), (n, 1))
    hx[:, 3] = g.uniform(-0.02, 0.02, n).astype(np.float32)
    return base, joints, held, hx


# ----------------------------------------------------------------------------------------------
# collision queries (N13; Appendix G): column grids, robot spheres, resting objects
# ----------------------------------------------------------------------------------------------

SPHERE_RADII = (0.015, 0.05, 0.12)      # the paper's sphere-radius working set
COLUMN_SPACING = 0.03


@dataclass
class ColumnGrid:
    """Free space of one static scene for one sphere radius: a dense array of columns in the XZ plane, each a
    list of layers (lo, hi) of heights the sphere's CENTRE may take.  Data only."""
    x0: float
    z0: float
    spacing: float
    nx: int
    nz: int
    col_off: np.ndarray      # [nx*nz + 1] uint32, column iz*nx + ix
    layers: np.ndarray       # [n,2] float32


@dataclass
class Sphere:
    link: int
    radius_class: int
    centre: Tuple[float, float, float]


_grid_cache: Dict = {}


def column_grid(cfg: int, scene: int, radius: float, extent: Optional[Tuple[float, float, float, float]] = None) -> ColumnGrid:
    """The column grid of a procedural apartment (stands in for the paper's offline pass over a ReplicaCAD scene with
    Habitat 2.0 sphere queries): a column is closed within radius + 5 cm of a wall; furniture whose
    footprint comes within the radius blocks the heights [0, top + radius], or, for every third piece (a 'table'),
    only [0.7 top - radius, top + radius]; the floor and the ceiling bound what is left.  extent = (x0, z0, x1, z1)
    restricts the grid to a window (tests)."""
    key = (cfg, scene, radius, extent)
    if key in _grid_cache:
        return _grid_cache[key]
    n_tris = CONFIG_SHAPES[cfg][5]
    info = _scenes(cfg, scene + 1, n_tris)[scene][1]
    boxes, segs = info["boxes"], info["segs"]
    x0, z0, x1, z1 = extent if extent is not None else (0.0, 0.0, FOOT, FOOT)
    nx, nz = int(round((x1 - x0) / COLUMN_SPACING)) + 1, int(round((z1 - z0) / COLUMN_SPACING)) + 1
    col_off = np.zeros(nx * nz + 1, np.uint32)
    layers: List[Tuple[float, float]] = []
    table = (np.arange(len(boxes)) % 3) == 2
    for iz in range(nz):
        px = x0 + COLUMN_SPACING * np.arange(nx)
        pz = np.full(nx, z0 + COLUMN_SPACING * iz)
        wall = _dist_segs(px, pz, segs).min(-1) < radius + 0.05
        near = _dist_boxes(px, pz, boxes) < radius                     # [nx, B]
        for ix in range(nx):
            if not wall[ix]:
                blocked = [(0.7 * boxes[b, 5] - radius if table[b] else -1.0, boxes[b, 5] + radius) for b in np.flatnonzero(near[ix])]
                lo = radius
                for b0, b1 in sorted(blocked):
                    if b0 > lo:
                        layers.append((lo, b0))
                    lo = max(lo, b1)
                if HEIGHT - radius > lo:
                    layers.append((lo, HEIGHT - radius))
            col_off[iz * nx + ix + 1] = len(layers)
    g = ColumnGrid(float(np.float32(x0)), float(np.float32(z0)), float(np.float32(COLUMN_SPACING)), nx, nz, col_off,
                   np.asarray(layers, np.float32).reshape(-1, 2))
    _grid_cache[key] = g
    return g


def robot_spheres(robot: Robot) -> List[Sphere]:
    """Spheres of the robot proxy (the paper authors them by hand for Fetch): big ones fill the base
    and the torso, medium and small ones run along the arm links and the hand."""
    out = [Sphere(0, 2, (dx, 0.0, dz)) for dx in (-0.12, 0.12) for dz in (-0.12, 0.12)]
    out += [Sphere(1, 2, (0.0, dy, 0.0)) for dy in (-0.15, 0.05, 0.25)]
    out += [Sphere(2, 1, (0.0, 0.0, -d)) for d in (0.0, 0.09, 0.18, 0.27)]
    out += [Sphere(3, 1, (0.0, 0.0, -d)) for d in (0.04, 0.12, 0.20, 0.28)]
    out += [Sphere(4, 0, (dx, 0.0, -d)) for d in (0.02, 0.08, 0.14, 0.20) for dx in (-0.02, 0.02)]
    assert all(0 <= s.link < len(robot.parent) for s in out)
    return out


def held_object_spheres() -> List[Sphere]:
    """Spheres of the object in the gripper ("and the current grasped object, if any"): link -1, centres
    in the object's own frame; three of the 5 cm class along its vertical axis and one small one off to the side."""
    return [Sphere(-1, 1, (0.0, dy, 0.0)) for dy in (-0.06, 0.0, 0.06)] + [Sphere(-1, 0, (0.05, 0.0, 0.03))]


def collision_world(n_envs: int, seed: int = 0, cfg: int = 1, extent: Optional[Tuple[float, float, float, float]] = None):
    """A batch of collision queries shaped like the paper's step (1 target + 29 distractor objects
    per episode; App. G): the robot proxy with its spheres in n_envs environments of one apartment, 30 resting
    box-shaped objects per environment (three meshes of different extents, rigid random poses on the floor near
    the robot or further away), the hand holding object 0 in half of them.  Returns a dict of plain arrays."""
    g = _rng(10, seed)
    robot = robot_proxy()
    base, joints, held, hx = robot_states(robot, n_envs, seed=seed)
    if extent is not None:
        base[:, 0] = g.uniform(extent[0] + 0.3, extent[2] - 0.3, n_envs).astype(np.float32)
        base[:, 1] = g.uniform(extent[1] + 0.3, extent[3] - 0.3, n_envs).astype(np.float32)
    meshes = [box_mesh(d, (1, 1, 1), _rng(10, 100 + i)) for i, d in enumerate(((0.06, 0.18, 0.06), (0.16, 0.08, 0.10), (0.09, 0.09, 0.22)))]
    n_obj, L = 30, len(robot.parent)
    K = n_obj + L
    inst_mesh = np.full((n_envs, K), -1, np.int32)
    inst_mesh[:, :n_obj] = g.integers(0, 3, (n_envs, n_obj))
    inst_mesh[:, 7] = -1                                                  # an empty slot among the objects
    xf = np.tile(np.eye(4, dtype=np.float32).reshape(16), (n_envs, K, 1))
    for n in range(n_envs):
        for k in range(n_obj):
            near = g.uniform() < 0.5
            rad = g.uniform(0.2, 0.9) if near else g.uniform(1.0, 4.0)
            ang = g.uniform(0, 2 * np.pi)
            yaw, tilt = g.uniform(0, 2 * np.pi), (g.uniform(-0.5, 0.5) if g.uniform() < 0.3 else 0.0)
            cy, sy, ct, st = np.cos(yaw), np.sin(yaw), np.cos(tilt), np.sin(tilt)
            R = np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]]) @ np.array([[1, 0, 0], [0, ct, -st], [0, st, ct]])
            M = np.eye(4)
            M[:3, :3] = R
            M[:3, 3] = [base[n, 0] + rad * np.cos(ang), g.uniform(0.03, 1.3), base[n, 1] + rad * np.sin(ang)]
            xf[n, k] = M.astype(np.float32).reshape(16)
    held_slot = np.where(held >= 0, 0, -1).astype(np.int32)
    return dict(robot=robot, spheres=robot_spheres(robot), radii=np.asarray(SPHERE_RADII, np.float32), dyn_meshes=meshes,
                base_pose=base, joint_pos=joints, held_slot=held_slot, held_xform=hx, inst_mesh=inst_mesh, inst_xform=xf,
                env_scene=np.zeros(n_envs, np.int32), K=K, link_slot0=n_obj, obj_slot0=0, n_obj=n_obj, cfg=cfg)
