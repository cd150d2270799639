"""Thin ctypes binding over libgx.so (include/gx.h): same names, argument marshalling only.

Every step of the render path runs in the CUDA kernels of csrc/; there is no CPU fallback.  If the
library is missing, import of this module's functions raises.  PyTorch is used by callers for device
memory and streams only; this module accepts anything with `.data_ptr()` (torch tensors), raw integer
addresses, or numpy arrays (host entry point only).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgx.so")

GX_OK, GX_ERR_INVALID_ARG, GX_ERR_CUDA, GX_ERR_OOM, GX_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
GX_BACKGROUND_ID = 0xFFFFFFFF
GX_NOALLOC_SCRATCH_BYTES = 64 << 20
EXPORTS = ("gx_create_scene", "gx_render_batch", "gx_render_batch_host", "gx_set_option", "gx_get_stat",
           "gx_render_batch_obs", "gx_set_robot", "gx_update_transforms", "gx_reserve", "gx_set_collision_world",
           "gx_collide_batch", "gx_render_batch_noalloc", "gx_destroy", "gx_last_error")


class GxMesh(C.Structure):
    _fields_ = [("positions", C.c_void_p), ("colors", C.c_void_p), ("indices", C.c_void_p),
                ("nv", C.c_uint32), ("nt", C.c_uint32)]


class GxCamera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("znear", C.c_float), ("zfar", C.c_float)]


class GxLink(C.Structure):
    _fields_ = [("parent", C.c_int32), ("joint_type", C.c_int32), ("axis", C.c_float * 3), ("origin", C.c_float * 12)]


class GxColumnGrid(C.Structure):
    _fields_ = [("x0", C.c_float), ("z0", C.c_float), ("spacing", C.c_float), ("nx", C.c_int32), ("nz", C.c_int32),
                ("col_off", C.c_void_p), ("layers", C.c_void_p)]


class GxSphere(C.Structure):
    _fields_ = [("link", C.c_int32), ("radius_class", C.c_int32), ("centre", C.c_float * 3)]


class GxError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gx error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libgx.so.  Fails loudly if it has not been built (python -m paper_2306_07552_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built; run `python -m paper_2306_07552_b200.build` "
                                    "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.gx_last_error.restype = C.c_char_p
        L.gx_destroy.restype = None
        for n in EXPORTS[:-2]:
            getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise GxError(rc, lib().gx_last_error().decode("utf-8", "replace"))


def _dev(a) -> Optional[C.c_void_p]:
    if a is None:
        return None
    if isinstance(a, int):
        return C.c_void_p(a)
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return C.c_void_p(a.data_ptr())
    raise TypeError(f"expected a device tensor or address, got {type(a)}")


def _host(a, dtype) -> Optional[C.c_void_p]:
    if a is None:
        return None
    if hasattr(a, "data_ptr"):   # CPU torch tensor (e.g. pinned)
        return C.c_void_p(a.data_ptr())
    assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous, (type(a), dtype)
    return C.c_void_p(a.ctypes.data)


def _mesh_array(meshes: Sequence):
    keep = []
    arr = (GxMesh * max(1, len(meshes)))()
    for i, m in enumerate(meshes):
        pos = np.ascontiguousarray(m.positions, np.float32)
        col = np.ascontiguousarray(m.colors, np.uint8)
        idx = np.ascontiguousarray(m.indices, np.uint32)
        keep += [pos, col, idx]
        arr[i] = GxMesh(pos.ctypes.data, col.ctypes.data, idx.ctypes.data, pos.shape[0], idx.shape[0])
    return arr, keep


def gx_create_scene(static_meshes: Sequence, dyn_meshes: Sequence, cuda_device: int = 0) -> C.c_void_p:
    """Meshes: objects with .positions [nv,3] f32, .colors [nv,3] u8, .indices [nt,3] u32 (host)."""
    sm, k1 = _mesh_array(static_meshes)
    dm, k2 = _mesh_array(dyn_meshes)
    h = C.c_void_p()
    _check(lib().gx_create_scene(sm, C.c_int32(len(static_meshes)), dm, C.c_int32(len(dyn_meshes)),
                                 C.c_int32(cuda_device), C.byref(h)))
    return h


def gx_render_batch(scene, camera: GxCamera, N: int, K: int, env_scene, cam_pose, inst_mesh, inst_xform,
                    rgb_out, depth_out, id_out=None, cuda_stream: int = 0) -> None:
    """All arrays are device tensors / addresses; enqueues on cuda_stream and returns."""
    _check(lib().gx_render_batch(scene, C.byref(camera), C.c_int32(N), C.c_int32(K), _dev(env_scene), _dev(cam_pose),
                                 _dev(inst_mesh), _dev(inst_xform), _dev(rgb_out), _dev(depth_out), _dev(id_out),
                                 C.c_void_p(cuda_stream)))


def gx_render_batch_noalloc(scene, camera: GxCamera, N: int, K: int, env_scene, cam_pose, inst_mesh, inst_xform,
                            rgb_out, depth_out, id_out=None, cuda_stream: int = 0) -> None:
    """gx_render_batch for callers that must not let the library call cudaMalloc / cudaFree (include/gx.h): same
    arguments and images, intermediate memory from the library's built-in GX_NOALLOC_SCRATCH_BYTES array; raises
    GxError(GX_ERR_UNSUPPORTED) for shapes beyond it.  Calls on one device must not overlap on the GPU."""
    _check(lib().gx_render_batch_noalloc(scene, C.byref(camera), C.c_int32(N), C.c_int32(K), _dev(env_scene),
                                         _dev(cam_pose), _dev(inst_mesh), _dev(inst_xform), _dev(rgb_out),
                                         _dev(depth_out), _dev(id_out), C.c_void_p(cuda_stream)))


def gx_render_batch_obs(scene, camera: GxCamera, N: int, K: int, env_scene, cam_pose, inst_mesh, inst_xform, obs_out,
                        depth_min: float, depth_max: float, cuda_stream: int = 0) -> None:
    """Packed observation [N,4,H,W] float16 (device tensor / address); enqueues on cuda_stream and returns."""
    _check(lib().gx_render_batch_obs(scene, C.byref(camera), C.c_int32(N), C.c_int32(K), _dev(env_scene), _dev(cam_pose),
                                     _dev(inst_mesh), _dev(inst_xform), _dev(obs_out), C.c_float(depth_min),
                                     C.c_float(depth_max), C.c_void_p(cuda_stream)))


def gx_render_batch_host(scene, camera: GxCamera, N: int, K: int, env_scene, cam_pose, inst_mesh, inst_xform,
                         rgb_out, depth_out, id_out=None) -> None:
    """All arrays are host numpy arrays (or CPU/pinned torch tensors); synchronous."""
    _check(lib().gx_render_batch_host(scene, C.byref(camera), C.c_int32(N), C.c_int32(K),
                                      _host(env_scene, np.int32), _host(cam_pose, np.float32),
                                      _host(inst_mesh, np.int32), _host(inst_xform, np.float32),
                                      _host(rgb_out, np.uint8), _host(depth_out, np.float32),
                                      _host(id_out, np.uint32)))


def gx_set_robot(scene, robot) -> None:
    """robot: an object with parent [L], joint_type [L], axis [L,3], origin [L,12], camera_link, cam_mount [12],
    ee_link (gen.Robot); host data, copied."""
    L = len(robot.parent)
    links = (GxLink * L)()
    for l in range(L):
        links[l].parent = int(robot.parent[l])
        links[l].joint_type = int(robot.joint_type[l])
        ax = np.asarray(robot.axis[l], np.float32)
        og = np.asarray(robot.origin[l], np.float32).reshape(12)
        for k in range(3):
            links[l].axis[k] = float(ax[k])
        for k in range(12):
            links[l].origin[k] = float(og[k])
    mount = np.ascontiguousarray(robot.cam_mount, np.float32).reshape(12)
    _check(lib().gx_set_robot(scene, links, C.c_int32(L), C.c_int32(int(robot.camera_link)), C.c_void_p(mount.ctypes.data),
                              C.c_int32(int(robot.ee_link))))


def gx_update_transforms(scene, N: int, K: int, link_slot0: int, base_pose, joint_pos, held_slot, held_xform, cam_pose,
                         inst_xform, cuda_stream: int = 0) -> None:
    """All arrays are device tensors / addresses; enqueues on cuda_stream and returns."""
    _check(lib().gx_update_transforms(scene, C.c_int32(N), C.c_int32(K), C.c_int32(link_slot0), _dev(base_pose), _dev(joint_pos),
                                      _dev(held_slot), _dev(held_xform), _dev(cam_pose), _dev(inst_xform),
                                      C.c_void_p(cuda_stream)))


def gx_set_collision_world(scene, grids, radii, spheres) -> None:
    """grids: [n_static][n_radii] objects with x0, z0, spacing, nx, nz, col_off, layers (gen.ColumnGrid); spheres:
    objects with link, radius_class, centre (gen.Sphere); host data, copied."""
    n_radii = len(radii)
    keep = []
    arr = (GxColumnGrid * (len(grids) * n_radii))()
    for i, row in enumerate(grids):
        if len(row) != n_radii:
            raise ValueError("one column grid per (scene, radius)")
        for j, g in enumerate(row):
            off = np.ascontiguousarray(g.col_off, np.uint32)
            lay = np.ascontiguousarray(g.layers, np.float32).reshape(-1, 2)
            keep += [off, lay]
            arr[i * n_radii + j] = GxColumnGrid(float(g.x0), float(g.z0), float(g.spacing), int(g.nx), int(g.nz),
                                                off.ctypes.data, lay.ctypes.data if lay.size else None)
    sph = (GxSphere * len(spheres))()
    for i, s in enumerate(spheres):
        sph[i].link = int(s.link)
        sph[i].radius_class = int(s.radius_class)
        for k in range(3):
            sph[i].centre[k] = float(np.float32(s.centre[k]))
    rad = np.ascontiguousarray(radii, np.float32)
    _check(lib().gx_set_collision_world(scene, arr, C.c_int32(n_radii), C.c_void_p(rad.ctypes.data), sph, C.c_int32(len(spheres))))


def gx_collide_batch(scene, N: int, K: int, env_scene, inst_mesh, inst_xform, link_slot0: int, obj_slot0: int, n_obj: int,
                     held_slot, out_static, out_object, cuda_stream: int = 0) -> None:
    """All arrays are device tensors / addresses; enqueues on cuda_stream and returns."""
    _check(lib().gx_collide_batch(scene, C.c_int32(N), C.c_int32(K), _dev(env_scene), _dev(inst_mesh), _dev(inst_xform),
                                  C.c_int32(link_slot0), C.c_int32(obj_slot0), C.c_int32(n_obj), _dev(held_slot), _dev(out_static),
                                  _dev(out_object), C.c_void_p(cuda_stream)))


def gx_reserve(scene, camera: GxCamera, N: int, K: int) -> None:
    _check(lib().gx_reserve(scene, C.byref(camera), C.c_int32(N), C.c_int32(K)))


def gx_set_option(scene, name: str, value: int) -> None:
    _check(lib().gx_set_option(scene, name.encode(), C.c_int64(value)))


def gx_get_stat(scene, name: str) -> int:
    v = C.c_int64()
    _check(lib().gx_get_stat(scene, name.encode(), C.byref(v)))
    return int(v.value)


def gx_destroy(scene) -> None:
    if scene:
        lib().gx_destroy(scene)


def gx_last_error() -> str:
    return lib().gx_last_error().decode("utf-8", "replace")


def camera_of(wl) -> GxCamera:
    """GxCamera from a gen.Workload (or anything with width/height/fx/fy/znear/zfar)."""
    return GxCamera(int(wl.width), int(wl.height), float(wl.fx), float(wl.fy), float(wl.znear), float(wl.zfar))
