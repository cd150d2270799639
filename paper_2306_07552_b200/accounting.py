"""Algorithmic byte accounting for the HBM roofline.

Harness-side numpy, float64; independent of how the kernels are written.  Per environment

    B_env = B_cull + B_geom + B_out

  B_cull = 32 B x (256-triangle clusters of the environment's static scene)
           + K x (16 B bounding sphere + 64 B transform) + 64 B camera pose
  B_geom = sum over the static clusters whose AABB, and the instances whose bounding sphere, intersect
           the view frustum (exact conservative test in float64):
           12 B per triangle (three uint32 indices) + 16 B per unique vertex referenced (3 x f32 + RGBA8)
  B_out  = H*W*7 B (RGB u8 + depth f32) or H*W*4 B (depth only)

Culling is credited (bytes of a culled cluster are not counted); intermediate records are not (whatever
the implementation writes and re-reads is its own cost).  `no_cull=True` counts every cluster and
instance, the secondary numerator SURVEY.md names.
"""
from __future__ import annotations

from typing import Dict

import numpy as np

CLUSTER_TRIS = 256


def _cluster_table(mesh) -> Dict[str, np.ndarray]:
    """Per 256-triangle cluster: AABB, triangle count, unique-vertex count."""
    idx = np.asarray(mesh.indices, np.int64)
    pos = np.asarray(mesh.positions, np.float64)
    nt = idx.shape[0]
    nc = (nt + CLUSTER_TRIS - 1) // CLUSTER_TRIS
    bmin = np.zeros((nc, 3)); bmax = np.zeros((nc, 3)); ntri = np.zeros(nc, np.int64); nuv = np.zeros(nc, np.int64)
    for c in range(nc):
        t = idx[c * CLUSTER_TRIS:(c + 1) * CLUSTER_TRIS]
        u = np.unique(t)
        p = pos[u]
        bmin[c], bmax[c] = p.min(axis=0), p.max(axis=0)
        ntri[c], nuv[c] = t.shape[0], u.shape[0]
    return dict(bmin=bmin, bmax=bmax, ntri=ntri, nuv=nuv, bytes=12 * ntri + 16 * nuv)


def _mesh_sphere(mesh):
    pos = np.asarray(mesh.positions, np.float64)
    c = 0.5 * (pos.min(axis=0) + pos.max(axis=0))
    r = float(np.sqrt(((pos - c) ** 2).sum(axis=1)).max()) if pos.shape[0] else 0.0
    nuv = int(np.unique(np.asarray(mesh.indices)).shape[0]) if mesh.nt else 0
    return c, r, 12 * mesh.nt + 16 * nuv


def _view(cam_pose):
    """World -> camera (rigid inverse), float64.  cam_pose [n,16] camera-to-world row-major."""
    C = np.asarray(cam_pose, np.float64).reshape(-1, 4, 4)
    R = C[:, :3, :3]
    t = C[:, :3, 3]
    Rt = np.transpose(R, (0, 2, 1))
    return Rt, -np.einsum("nij,nj->ni", Rt, t)


def env_bytes(wl, no_cull: bool = False) -> Dict[str, np.ndarray]:
    """Per-environment algorithmic bytes of a gen.Workload.  Returns arrays [N]: cull, geom, out, total,
    and tris (triangles of the counted clusters / instances)."""
    N, K, W, H = wl.N, wl.K, wl.width, wl.height
    fx, fy, zn, zf = float(wl.fx), float(wl.fy), float(wl.znear), float(wl.zfar)
    tabs = [_cluster_table(m) for m in wl.static_meshes]
    sph = [_mesh_sphere(m) for m in wl.dyn_meshes]
    Rt, tv = _view(wl.cam_pose)
    b_cull = np.zeros(N); b_geom = np.zeros(N); tris = np.zeros(N)
    corner = np.array([[(i >> a) & 1 for a in range(3)] for i in range(8)], np.float64)   # [8,3]
    sx, sy = np.sqrt(fx * fx + 1.0), np.sqrt(fy * fy + 1.0)
    for n in range(N):
        tab = tabs[int(wl.env_scene[n])]
        nc = tab["ntri"].shape[0]
        b_cull[n] = 32.0 * nc + 80.0 * K + 64.0
        # static clusters: 8 AABB corners in camera space; culled iff all corners are outside one plane
        P = tab["bmin"][:, None, :] + corner[None] * (tab["bmax"] - tab["bmin"])[:, None, :]   # [nc,8,3]
        Pc = P @ Rt[n].T + tv[n]
        x, y, w = Pc[..., 0], Pc[..., 1], -Pc[..., 2]
        out = ((w < zn).all(1) | (w > zf).all(1) | (fx * x > w).all(1) | (-fx * x > w).all(1) |
               (fy * y > w).all(1) | (-fy * y > w).all(1))
        vis = ~out | no_cull
        b_geom[n] += tab["bytes"][vis].sum()
        tris[n] += tab["ntri"][vis].sum()
        # instances: bounding sphere under the affine transform (radius scaled by the largest singular value)
        for k in range(K):
            m = int(wl.inst_mesh[n, k])
            if m < 0:
                continue
            c, r, nbytes = sph[m]
            M = np.asarray(wl.inst_xform[n, k], np.float64).reshape(4, 4)
            cw = M[:3, :3] @ c + M[:3, 3]
            rr = r * np.linalg.norm(M[:3, :3], 2)
            cc = Rt[n] @ cw + tv[n]
            x, y, w = cc[0], cc[1], -cc[2]
            outside = (w < zn - rr) or (w > zf + rr) or ((fx * x - w) / sx > rr) or ((-fx * x - w) / sx > rr) or \
                      ((fy * y - w) / sy > rr) or ((-fy * y - w) / sy > rr)
            if no_cull or not outside:
                b_geom[n] += nbytes
                tris[n] += wl.dyn_meshes[m].nt
    b_out = np.full(N, float(H * W * (4 if wl.depth_only else 7)))
    return dict(cull=b_cull, geom=b_geom, out=b_out, total=b_cull + b_geom + b_out, tris=tris)
