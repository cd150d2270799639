"""ctypes wrapper around oracle/gx_oracle.c (plain C, gcc -O2 -ffp-contract=off, OpenMP over environments).

TEST INFRASTRUCTURE, NOT PRODUCT -- see the header of gx_oracle.c.  Argument marshalling only; every
step of the definition (N0-N10) is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gx_oracle.c")
_LIB = os.path.join(_HERE, "libgx_oracle.so")
BACKGROUND_ID = 0xFFFFFFFF
FLAG_FULL_SCAN = 1

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-std=c11", "-Wall", "-Wextra",
               "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Mesh(C.Structure):
    _fields_ = [("positions", C.c_void_p), ("colors", C.c_void_p), ("indices", C.c_void_p),
                ("nv", C.c_uint32), ("nt", C.c_uint32)]


class _Camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("znear", C.c_float), ("zfar", C.c_float)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.gx_oracle_render.restype = C.c_int
        _lib.gx_oracle_raster_soup.restype = C.c_int
        _lib.gx_oracle_vertex_stage.restype = C.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _meshes(meshes):
    keep = []
    arr = (_Mesh * max(1, len(meshes)))()
    for i, m in enumerate(meshes):
        pos = np.ascontiguousarray(m.positions, np.float32)
        col = np.ascontiguousarray(m.colors, np.uint8)
        idx = np.ascontiguousarray(m.indices, np.uint32)
        keep += [pos, col, idx]
        arr[i] = _Mesh(pos.ctypes.data, col.ctypes.data, idx.ctypes.data, pos.shape[0], idx.shape[0])
    return arr, keep


def _camera(W, H, fx, fy, znear, zfar):
    return _Camera(int(W), int(H), float(fx), float(fy), float(znear), float(zfar))


def render(wl, n_threads: Optional[int] = None, want_sub: bool = False, want_count: bool = False,
           full_scan: bool = False):
    """Render a workload (any object with the fields of gen.Workload).  Returns dict(rgb, depth, id[, sub, count])."""
    lib = _load()
    N, K, W, H = wl.N, wl.K, wl.width, wl.height
    sm, k1 = _meshes(wl.static_meshes)
    dm, k2 = _meshes(wl.dyn_meshes)
    cam = _camera(W, H, wl.fx, wl.fy, wl.znear, wl.zfar)
    env_scene = np.ascontiguousarray(wl.env_scene, np.int32)
    cam_pose = np.ascontiguousarray(wl.cam_pose, np.float32)
    inst_mesh = np.ascontiguousarray(wl.inst_mesh, np.int32)
    inst_xform = np.ascontiguousarray(wl.inst_xform, np.float32)
    rgb = np.empty((N, H, W, 3), np.uint8)
    depth = np.empty((N, H, W), np.float32)
    ids = np.empty((N, H, W), np.uint32)
    sub = np.empty((N, H, W), np.uint8) if want_sub else None
    cnt = np.empty((N, H, W), np.uint32) if want_count else None
    if n_threads is None:
        n_threads = len(os.sched_getaffinity(0))
    rc = lib.gx_oracle_render(sm, C.c_int32(len(wl.static_meshes)), dm, C.c_int32(len(wl.dyn_meshes)), C.byref(cam),
                              C.c_int32(N), C.c_int32(K), _p(env_scene), _p(cam_pose), _p(inst_mesh), _p(inst_xform),
                              _p(rgb), _p(depth), _p(ids), _p(sub), _p(cnt),
                              C.c_int32(FLAG_FULL_SCAN if full_scan else 0), C.c_int32(int(n_threads)))
    if rc != 0:
        raise RuntimeError(f"gx_oracle_render failed: {rc}")
    out = dict(rgb=rgb, depth=depth, id=ids)
    if want_sub:
        out["sub"] = sub
    if want_count:
        out["count"] = cnt
    return out


def raster_soup(W, H, fx, fy, znear, zfar, verts: np.ndarray, ids: Sequence[int], want_count=False,
                full_scan=False):
    """N4-N9 on a camera-space soup: verts [nt,3,6] = (xc, yc, w, r, g, b); ids [nt]."""
    lib = _load()
    verts = np.ascontiguousarray(verts, np.float32)
    nt = verts.shape[0]
    assert verts.shape == (nt, 3, 6)
    ids = np.ascontiguousarray(ids, np.uint32)
    assert ids.shape == (nt,)
    cam = _camera(W, H, fx, fy, znear, zfar)
    rgb = np.empty((H, W, 3), np.uint8)
    depth = np.empty((H, W), np.float32)
    oid = np.empty((H, W), np.uint32)
    sub = np.empty((H, W), np.uint8)
    cnt = np.empty((H, W), np.uint32) if want_count else None
    rc = lib.gx_oracle_raster_soup(C.byref(cam), _p(verts), _p(ids), C.c_uint32(nt), _p(rgb), _p(depth), _p(oid),
                                   _p(sub), _p(cnt), C.c_int32(FLAG_FULL_SCAN if full_scan else 0))
    if rc != 0:
        raise RuntimeError(f"gx_oracle_raster_soup failed: {rc}")
    out = dict(rgb=rgb, depth=depth, id=oid, sub=sub)
    if want_count:
        out["count"] = cnt
    return out


def vertex_stage(W, H, fx, fy, znear, zfar, cam_pose, xform, positions):
    """N1-N3 + N5 per vertex.  Returns dict(xc, yc, w, q, Xi, Yi, inside)."""
    lib = _load()
    cam = _camera(W, H, fx, fy, znear, zfar)
    cam_pose = np.ascontiguousarray(cam_pose, np.float32).reshape(16)
    xf = None if xform is None else np.ascontiguousarray(xform, np.float32).reshape(16)
    pos = np.ascontiguousarray(positions, np.float32)
    nv = pos.shape[0]
    o = dict(xc=np.empty(nv, np.float32), yc=np.empty(nv, np.float32), w=np.empty(nv, np.float32),
             q=np.empty(nv, np.float32), Xi=np.empty(nv, np.int32), Yi=np.empty(nv, np.int32),
             inside=np.empty(nv, np.uint8))
    rc = lib.gx_oracle_vertex_stage(C.byref(cam), _p(cam_pose), _p(xf), _p(pos), C.c_uint32(nv), _p(o["xc"]),
                                    _p(o["yc"]), _p(o["w"]), _p(o["q"]), _p(o["Xi"]), _p(o["Yi"]), _p(o["inside"]))
    if rc != 0:
        raise RuntimeError(f"gx_oracle_vertex_stage failed: {rc}")
    return o


def pack_obs(rgb: np.ndarray, depth: np.ndarray, dmin: float, dmax: float) -> np.ndarray:
    """N11: packed observation [N,4,H,W] as uint16 bit patterns of binary16 (view as np.float16 to read)."""
    L = _load()
    rgb = np.ascontiguousarray(rgb, np.uint8)
    depth = np.ascontiguousarray(depth, np.float32)
    N, H, W = depth.shape
    out = np.empty((N, 4, H, W), np.uint16)
    L.gx_oracle_pack_obs.restype = C.c_int
    rc = L.gx_oracle_pack_obs(_p(rgb), _p(depth), C.c_int32(N), C.c_int32(H), C.c_int32(W), C.c_float(dmin), C.c_float(dmax), _p(out))
    if rc != 0:
        raise ValueError("gx_oracle_pack_obs: bad arguments")
    return out


def half_rn(x: np.ndarray) -> np.ndarray:
    """binary32 -> binary16 bit patterns with the oracle's hand-written conversion."""
    L = _load()
    x = np.ascontiguousarray(x, np.float32)
    out = np.empty(x.shape, np.uint16)
    L.gx_oracle_half_rn.restype = None
    L.gx_oracle_half_rn(_p(x), _p(out), C.c_size_t(x.size))
    return out


class _Link(C.Structure):
    _fields_ = [("parent", C.c_int32), ("joint_type", C.c_int32), ("axis", C.c_float * 3), ("origin", C.c_float * 12)]


def sincos(x: np.ndarray):
    """N12a: the definition's own binary32 sine and cosine."""
    L = _load()
    x = np.ascontiguousarray(x, np.float32)
    s, c = np.empty_like(x), np.empty_like(x)
    L.gx_oracle_sincos.restype = None
    L.gx_oracle_sincos(_p(x), _p(s), _p(c), C.c_size_t(x.size))
    return s, c


def fk(robot, base_pose, joint_pos, K: int, link_slot0: int, inst_xform: Optional[np.ndarray] = None,
       held_slot: Optional[np.ndarray] = None, held_xform: Optional[np.ndarray] = None):
    """N12: forward kinematics.  robot: any object with parent [L], joint_type [L], axis [L,3], origin [L,12],
    camera_link, cam_mount [12], ee_link (gen.Robot).  Returns (cam_pose [N,16], inst_xform [N,K,16])."""
    lib = _load()
    Ln = len(robot.parent)
    links = (_Link * Ln)()
    for l in range(Ln):
        links[l].parent = int(robot.parent[l])
        links[l].joint_type = int(robot.joint_type[l])
        for k in range(3):
            links[l].axis[k] = float(np.float32(robot.axis[l][k]))
        for k in range(12):
            links[l].origin[k] = float(np.float32(np.asarray(robot.origin[l]).reshape(12)[k]))
    base_pose = np.ascontiguousarray(base_pose, np.float32)
    joint_pos = np.ascontiguousarray(joint_pos, np.float32)
    N = base_pose.shape[0]
    assert base_pose.shape == (N, 3) and joint_pos.shape == (N, Ln)
    xf = np.zeros((N, K, 16), np.float32) if inst_xform is None else np.array(inst_xform, np.float32, copy=True).reshape(N, K, 16)
    cam = np.empty((N, 16), np.float32)
    mount = np.ascontiguousarray(robot.cam_mount, np.float32).reshape(12)
    hs = None if held_slot is None else np.ascontiguousarray(held_slot, np.int32)
    hx = None if held_xform is None else np.ascontiguousarray(held_xform, np.float32).reshape(N, 12)
    lib.gx_oracle_fk.restype = C.c_int
    rc = lib.gx_oracle_fk(links, C.c_int32(Ln), C.c_int32(int(robot.camera_link)), _p(mount), C.c_int32(int(robot.ee_link)),
                          C.c_int32(N), C.c_int32(K), C.c_int32(link_slot0), _p(base_pose), _p(joint_pos), _p(hs), _p(hx),
                          _p(cam), _p(xf))
    if rc != 0:
        raise ValueError("gx_oracle_fk: bad arguments")
    return cam, xf


class _ColumnGrid(C.Structure):
    _fields_ = [("x0", C.c_float), ("z0", C.c_float), ("spacing", C.c_float), ("nx", C.c_int32), ("nz", C.c_int32),
                ("col_off", C.c_void_p), ("layers", C.c_void_p)]


class _Sphere(C.Structure):
    _fields_ = [("link", C.c_int32), ("radius_class", C.c_int32), ("centre", C.c_float * 3)]


def collide(dyn_meshes, grids, radii, spheres, env_scene, inst_mesh, inst_xform, link_slot0: int, obj_slot0: int,
            n_obj: int, held_slot: Optional[np.ndarray] = None):
    """N13: batch collision queries.  grids: [n_static][n_radii] objects with x0, z0, spacing, nx, nz, col_off, layers
    (gen.ColumnGrid); spheres: objects with link, radius_class, centre.  Returns (static [N,S] uint8, object [N,S] int32)."""
    lib = _load()
    dm, keep = _meshes(dyn_meshes)
    n_static, n_radii = len(grids), len(radii)
    garr = (_ColumnGrid * (n_static * n_radii))()
    for i, row in enumerate(grids):
        assert len(row) == n_radii
        for j, g in enumerate(row):
            off = np.ascontiguousarray(g.col_off, np.uint32)
            lay = np.ascontiguousarray(g.layers, np.float32).reshape(-1, 2)
            keep += [off, lay]
            garr[i * n_radii + j] = _ColumnGrid(float(g.x0), float(g.z0), float(g.spacing), int(g.nx), int(g.nz),
                                                off.ctypes.data, lay.ctypes.data)
    S = len(spheres)
    sarr = (_Sphere * S)()
    for i, s in enumerate(spheres):
        sarr[i].link = int(s.link)
        sarr[i].radius_class = int(s.radius_class)
        for k in range(3):
            sarr[i].centre[k] = float(np.float32(s.centre[k]))
    rad = np.ascontiguousarray(radii, np.float32)
    env_scene = np.ascontiguousarray(env_scene, np.int32)
    inst_mesh = np.ascontiguousarray(inst_mesh, np.int32)
    inst_xform = np.ascontiguousarray(inst_xform, np.float32)
    N, K = inst_mesh.shape
    hs = None if held_slot is None else np.ascontiguousarray(held_slot, np.int32)
    out_s = np.empty((N, S), np.uint8)
    out_o = np.empty((N, S), np.int32)
    lib.gx_oracle_collide.restype = C.c_int
    rc = lib.gx_oracle_collide(dm, C.c_int32(len(dyn_meshes)), garr, C.c_int32(n_static), C.c_int32(n_radii), _p(rad), sarr,
                               C.c_int32(S), C.c_int32(N), C.c_int32(K), _p(env_scene), _p(inst_mesh), _p(inst_xform),
                               C.c_int32(link_slot0), C.c_int32(obj_slot0), C.c_int32(n_obj), _p(hs), _p(out_s), _p(out_o))
    if rc != 0:
        raise ValueError("gx_oracle_collide: bad arguments")
    return out_s, out_o
