"""Pins of the CPU oracle against what the mathematics fixes (run with -m "not gpu").

The paper prints no worked rendering example (PAPER.md:91,141 give only the problem statement), so the
pins are closed forms, exact brute force, double-precision ray casting and invariants, chosen so that a
dropped term, wrong sign/index or transposed operand in oracle/gx_oracle.c fails at least one of them.
Nothing here retypes the oracle's formulas: expected values come from hand derivations
(tests/golden/), exact integer/rational geometry, numpy float64 linear algebra, or ray casting.
"""
import os

import numpy as np
import pytest

from paper_2306_07552_b200 import gen

BG = 0xFFFFFFFF
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _pose(name):
    C = np.eye(4, dtype=np.float32)
    if name == "T":
        C[:3, 3] = [1, 2, 3]
    elif name == "Y90":
        C[:3, :3] = np.array([[0, 0, 1], [0, 1, 0], [-1, 0, 0]], np.float32)
    return C


# --------------------------------------------------------------------------------------------
# N1-N5 vertex stage
# --------------------------------------------------------------------------------------------

def test_vertex_closed_form(oracle_mod):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "vertex_closed_form.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) >= 10
    for pose, px, py, pz, X, Y, w in rows:
        o = oracle_mod.vertex_stage(64, 64, 1.0, 1.0, 0.1, 20.0, _pose(pose), None,
                                    np.array([[float(px), float(py), float(pz)]], np.float32))
        assert o["inside"][0] == 1
        assert (int(o["Xi"][0]), int(o["Yi"][0]), float(o["w"][0])) == (int(X), int(Y), float(w)), (pose, px, py, pz)


def test_vertex_instance_closed_form(oracle_mod):
    # object-to-world = uniform scale 2 then translate (0,0,-6): object point (0.5,0.5,1) -> world (1,1,-4)
    M = np.eye(4, dtype=np.float32)
    M[:3, :3] *= 2
    M[:3, 3] = [0, 0, -6]
    o = oracle_mod.vertex_stage(64, 64, 1.0, 1.0, 0.1, 20.0, _pose("I"), M, np.array([[0.5, 0.5, 1.0]], np.float32))
    assert (int(o["Xi"][0]), int(o["Yi"][0]), float(o["w"][0])) == (8192 + 2048, 8192 - 2048, 4.0)
    # non-symmetric object matrix: a transposed operand would map x->z: M = rot +90 about Y then translate
    M = np.array([[0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, -4], [0, 0, 0, 1]], np.float32)
    # object (1,0,2) -> world (2,0,-1-4) = (2,0,-5)?  row2: -1*1 + 0 + 0*2 - 4 = -5 ; row0: 2
    o = oracle_mod.vertex_stage(64, 64, 1.0, 1.0, 0.1, 20.0, _pose("T"), M, np.array([[1.0, 0.0, 2.0]], np.float32))
    # camera at (1,2,3): rel = (1,-2,-8): X = (1/8)*8192+8192 = 9216, Y = (2/8)*8192+8192 = 10240, w = 8
    assert (int(o["Xi"][0]), int(o["Yi"][0]), float(o["w"][0])) == (9216, 10240, 8.0)


def test_vertex_vs_float64(oracle_mod):
    rng = np.random.default_rng(7)
    W, H, fx, fy = 128, 64, 0.5, 1.0   # non-square on purpose: swapping W/H or fx/fy must fail
    for trial in range(20):
        wl_pose = gen._cam_pose(rng.uniform(-3, 3, (1, 3)), rng.uniform(0, 6.28, 1), rng.uniform(-1, 1, 1))[0]
        A = rng.normal(size=(3, 3))
        M = np.eye(4)
        M[:3, :3] = A
        M[:3, 3] = rng.uniform(-2, 2, 3)
        pos = rng.uniform(-6, 6, (400, 3)).astype(np.float32)
        o = oracle_mod.vertex_stage(W, H, fx, fy, 0.1, 50.0, wl_pose.astype(np.float32), M.astype(np.float32), pos)
        C64 = wl_pose.astype(np.float32).astype(np.float64)
        M64 = M.astype(np.float32).astype(np.float64)
        pc = (np.linalg.inv(C64) @ M64 @ np.concatenate([pos.astype(np.float64), np.ones((400, 1))], 1).T).T
        w = -pc[:, 2]
        sel = (w > 0.5) & (np.abs(pc[:, 0] / w) < 4) & (np.abs(pc[:, 1] / w) < 4)
        if sel.sum() < 20:
            continue   # geometry seen edge-on in this trial
        assert np.all(o["inside"][sel] == 1) and np.all(o["inside"][w < 0.0999] == 0)
        Xpix = (fx * pc[:, 0] / w * 0.5 + 0.5) * W       # pixel units, x right
        Ypix = (0.5 - 0.5 * fy * pc[:, 1] / w) * H       # row 0 at the top
        assert np.max(np.abs(o["Xi"][sel] - 256 * Xpix[sel])) <= 0.51
        assert np.max(np.abs(o["Yi"][sel] - 256 * Ypix[sel])) <= 0.51
        assert np.allclose(o["w"][sel], w[sel], rtol=1e-5)
        assert np.allclose(o["q"][sel], 1 / w[sel], rtol=1e-5)


# --------------------------------------------------------------------------------------------
# helpers: camera-space soups whose snapped coordinates are known by construction
# --------------------------------------------------------------------------------------------

def _soup_from_snapped(XY, W, H, w=2.0, colors=None):
    """Triangles given by snapped integer corners XY [nt,3,2] (1/256 px) at constant view depth w (a
    power of two): xc = (X - hw) * w / hw is exact in binary32, so N5 reproduces X exactly."""
    XY = np.asarray(XY, np.float64)
    nt = XY.shape[0]
    hw, hh = 128.0 * W, 128.0 * H
    v = np.zeros((nt, 3, 6), np.float32)
    v[:, :, 0] = (XY[:, :, 0] - hw) * w / hw
    v[:, :, 1] = -(XY[:, :, 1] - hh) * w / hh
    v[:, :, 2] = w
    v[:, :, 3:] = 200.0 if colors is None else colors
    return v


def _covered_exact(tri, px, py):
    """Top-left rule from its geometric meaning, in exact integer arithmetic: the pixel centre displaced
    infinitesimally to the right and (to second order) downwards, p + (eps, eps^2), is strictly inside
    the triangle.  Orientation-free: all three edge functions must have the sign of the area."""
    (x0, y0), (x1, y1), (x2, y2) = [(int(a), int(b)) for a, b in tri]
    area = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0)
    if area == 0:
        return False
    s = 1 if area > 0 else -1
    S = 1 << 80  # eps = 2^-80: |perturbation| < 2^-40 << 1 = smallest non-zero |integer edge value|
    for (ax, ay), (bx, by) in (((x0, y0), (x1, y1)), ((x1, y1), (x2, y2)), ((x2, y2), (x0, y0))):
        # edge function scaled by S^2 at (px + 1/S, py + 1/S^2)
        e = ((bx - ax) * ((py - ay) * S * S + 1) - (by - ay) * ((px - ax) * S * S + S))
        if e * s <= 0:
            return False
    return True


# --------------------------------------------------------------------------------------------
# N6 coverage
# --------------------------------------------------------------------------------------------

@pytest.mark.parametrize("diag", [0, 1])
@pytest.mark.parametrize("flip", [0, 1])
def test_quad_closed_form(oracle_mod, diag, flip):
    W = H = 16
    offs = [0, 1, 127, 128, 129, 255]
    for ox0 in offs:
        for ox1 in offs:
            for oy0, oy1 in ((0, 128), (129, 255), (128, 127), (1, 129)):
                Xlo, Xhi = 256 * 3 + ox0, 256 * 9 + ox1
                Ylo, Yhi = 256 * 2 + oy0, 256 * 12 + oy1
                a, b, c, d = (Xlo, Ylo), (Xhi, Ylo), (Xhi, Yhi), (Xlo, Yhi)
                tris = [[a, b, c], [a, c, d]] if diag == 0 else [[a, b, d], [b, c, d]]
                if flip:
                    tris = [[t[0], t[2], t[1]] for t in tris]
                o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(tris, W, H), [0, 1],
                                           want_count=True)
                cx = 256 * np.arange(W) + 128
                cy = 256 * np.arange(H) + 128
                exp = ((cy[:, None] >= Ylo) & (cy[:, None] < Yhi)) & ((cx[None, :] >= Xlo) & (cx[None, :] < Xhi))
                assert np.array_equal(o["count"], exp.astype(np.uint32)), (ox0, ox1, oy0, oy1)
                assert np.array_equal(o["id"] != BG, exp)
                assert np.all(o["depth"][exp] == 2.0) and np.all(o["depth"][~exp] == 0.0)


def test_bruteforce_exact_integers(oracle_mod):
    """Coverage count and winning id against exact big-integer evaluation; vertices on a 64-unit lattice
    so that edges and vertices pass through pixel centres all the time; all triangles at the same depth,
    so by N9 the winner is the lowest id among the covering triangles."""
    rng = np.random.default_rng(11)
    W, H = 12, 10
    for trial in range(12):
        nt = 12
        XY = rng.integers(-8, 60, (nt, 3, 2)) * 64
        XY[:, :, 1] = np.minimum(XY[:, :, 1], 48 * 64)
        if trial % 3 == 0:  # axis-aligned and degenerate cases
            XY[::4, 1, 1] = XY[::4, 0, 1]
            XY[1::8, 2] = XY[1::8, 1]
        ids = rng.permutation(nt).astype(np.uint32) + 5
        o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, W, H), ids, want_count=True)
        cnt = np.zeros((H, W), np.uint32)
        win = np.full((H, W), BG, np.uint32)
        for j in range(H):
            for i in range(W):
                for t in range(nt):
                    if _covered_exact(XY[t], 256 * i + 128, 256 * j + 128):
                        cnt[j, i] += 1
                        win[j, i] = min(win[j, i], ids[t])
        assert cnt.max() >= 3 and (cnt == 0).any()
        assert np.array_equal(o["count"], cnt)
        assert np.array_equal(o["id"], win)


def test_watertight_grid_exactly_once(oracle_mod):
    """A triangulated surface with shared vertices, random diagonals and random windings, in perspective
    (varying depth), larger than the screen: every pixel is covered by exactly one triangle."""
    rng = np.random.default_rng(3)
    W, H = 48, 40
    n = 30
    gx, gy = np.meshgrid(np.linspace(-1.6, 1.6, n + 1), np.linspace(-1.6, 1.6, n + 1), indexing="ij")
    for trial in range(4):
        jx = gx + rng.uniform(-0.02, 0.02, gx.shape)
        jy = gy + rng.uniform(-0.02, 0.02, gy.shape)
        w = 1.0 + rng.uniform(0, 3.0) * (gx + 2) + rng.uniform(-0.2, 0.2, gx.shape)   # tilted, bumpy
        P = np.stack([jx * w, jy * w, w], -1)    # camera space (x = ndc*w for fx=1)
        tris = []
        for i in range(n):
            for j in range(n):
                a, b, c, d = P[i, j], P[i + 1, j], P[i + 1, j + 1], P[i, j + 1]
                pair = ([a, b, c], [a, c, d]) if rng.random() < 0.5 else ([a, b, d], [b, c, d])
                for t in pair:
                    if rng.random() < 0.5:
                        t = [t[0], t[2], t[1]]
                    k = rng.integers(0, 3)
                    tris.append(t[k:] + t[:k])
        v = np.zeros((len(tris), 3, 6), np.float32)
        v[:, :, :3] = np.array(tris)
        v[:, :, 3:] = 100
        o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 100.0, v, np.arange(len(tris)), want_count=True)
        assert np.all(o["count"] == 1)


def test_rotation_and_winding_leave_coverage_unchanged(oracle_mod):
    rng = np.random.default_rng(5)
    W = H = 24
    XY = rng.integers(-2 * 256, 26 * 256, (60, 3, 2))
    base = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, W, H), np.arange(60), want_count=True)
    for perm in ([1, 2, 0], [2, 0, 1], [0, 2, 1], [2, 1, 0]):
        o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY[:, perm], W, H), np.arange(60),
                                   want_count=True)
        # (the winning id may change: with areas > 2^24 the depth of a w=2 triangle rounds to 2 -/+ 1 ulp
        # depending on the order of the three terms of N7, so only coverage is invariant)
        assert np.array_equal(o["count"], base["count"])
        assert np.array_equal(o["id"] != BG, base["id"] != BG)


def test_full_scan_equals_bbox(oracle_mod):
    wl = gen.make_config(0)
    a = oracle_mod.render(wl, want_count=True)
    b = oracle_mod.render(wl, want_count=True, full_scan=True)
    for k in ("rgb", "depth", "id", "count"):
        assert np.array_equal(a[k], b[k]), k


# --------------------------------------------------------------------------------------------
# ray casting in float64 (independent of snapping, edge functions and the clip)
# --------------------------------------------------------------------------------------------

def _raycast(tri_cam, col, W, H, fx, fy, znear, zfar):
    """Nearest hit per pixel-centre ray, Moeller-Trumbore in float64, camera space, unsnapped geometry.
    tri_cam [nt,3,3] (x, y, z) with the camera looking along -z.  Returns id [-1 none], depth w, rgb."""
    j, i = np.meshgrid(np.arange(H), np.arange(W), indexing="ij")
    d = np.stack([((i + 0.5) / W * 2 - 1) / fx, (1 - (j + 0.5) / H * 2) / fy, -np.ones_like(i, float)], -1).reshape(-1, 3)
    best = np.full(d.shape[0], np.inf)
    bid = np.full(d.shape[0], -1)
    brgb = np.zeros((d.shape[0], 3))
    second = np.full(d.shape[0], np.inf)
    edge = np.zeros(d.shape[0], bool)
    for t in range(tri_cam.shape[0]):
        v0, v1, v2 = tri_cam[t]
        e1, e2 = v1 - v0, v2 - v0
        pv = np.cross(d, e2)
        det = pv @ e1
        ok = np.abs(det) > 1e-14
        inv = np.where(ok, 1.0 / np.where(ok, det, 1), 0)
        tv = -v0
        u = (pv @ tv) * inv
        qv = np.cross(tv, e1)
        vv = (d @ qv) * inv
        tt = (e2 @ qv) * inv        # ray parameter = w because d_z = -1
        hit = ok & (u >= 0) & (vv >= 0) & (u + vv <= 1) & (tt >= znear) & (tt <= zfar)
        near_edge = ok & (np.minimum(np.minimum(u, vv), 1 - u - vv) > -0.02) & (np.minimum(np.minimum(u, vv), 1 - u - vv) < 0.02)
        edge |= near_edge
        closer = hit & (tt < best)
        second = np.where(closer, best, np.where(hit & (tt < second), tt, second))
        best = np.where(closer, tt, best)
        bid = np.where(closer, t, bid)
        wgt = np.stack([1 - u - vv, u, vv], -1)
        brgb = np.where(closer[:, None], wgt @ col[t].astype(float), brgb)
    return (bid.reshape(H, W), best.reshape(H, W), brgb.reshape(H, W, 3), second.reshape(H, W), edge.reshape(H, W))


def _rel_inv_w_gradient(tri_cam, rid, rw, W, H, fx, fy):
    """|gradient of 1/w with respect to pixel coordinates| * w for the triangle hit at each pixel.
    Plane n.P = d and ray P = w*(xn/fx, yn/fy, -1) give 1/w = n.dir/d, affine in the pixel position."""
    v0, v1, v2 = tri_cam[:, 0], tri_cam[:, 1], tri_cam[:, 2]
    nrm = np.cross(v1 - v0, v2 - v0)
    d = np.einsum("ij,ij->i", nrm, v0)
    with np.errstate(divide="ignore", invalid="ignore"):
        gx = nrm[:, 0] * (2.0 / (W * fx)) / d
        gy = -nrm[:, 1] * (2.0 / (H * fy)) / d
    t = np.maximum(rid, 0)
    return np.hypot(gx[t], gy[t]) * np.where(np.isfinite(rw), rw, 0.0)


def _camera_space_triangles(wl, n):
    """float64 camera-space corners and colours of every triangle of env n, in triangle-id order."""
    C = wl.cam_pose[n].reshape(4, 4).astype(np.float64)
    Vm = np.linalg.inv(C)
    tris, cols = [], []
    parts = [(wl.static_meshes[wl.env_scene[n]], np.eye(4))]
    for k in range(wl.K):
        if wl.inst_mesh[n, k] >= 0:
            parts.append((wl.dyn_meshes[wl.inst_mesh[n, k]], wl.inst_xform[n, k].reshape(4, 4).astype(np.float64)))
    for m, M in parts:
        p = np.concatenate([m.positions.astype(np.float64), np.ones((m.nv, 1))], 1) @ (Vm @ M).T
        tris.append(p[:, :3][m.indices.astype(np.int64)])
        cols.append(m.colors[m.indices.astype(np.int64)])
    return np.concatenate(tris), np.concatenate(cols)


def test_whole_image_vs_raycast_config0(oracle_mod):
    """End-to-end check of conventions (handedness, row order, FoV, near clip, id numbering, instance
    transforms, perspective-correct depth and colour) on config 0."""
    wl = gen.make_config(0)
    o = oracle_mod.render(wl)
    n_unclipped = n_clipped = 0
    for n in range(wl.N):
        tri, col = _camera_space_triangles(wl, n)
        rid, rw, rrgb, second, edge = _raycast(tri, col, wl.width, wl.height, wl.fx, wl.fy, wl.znear, wl.zfar)
        oid = o["id"][n].astype(np.int64)
        oid[oid == BG] = -1
        same = oid == rid
        assert same.mean() >= 0.99, same.mean()
        # every disagreement sits next to a projected edge (snapping moves edges by < 1/256 px) or at a
        # near-tie of two surfaces
        bad = ~same
        assert np.all(edge[bad] | (np.abs(second[bad] - rw[bad]) < 1e-3 * rw[bad]))
        hit = same & (rid >= 0)
        rel = np.abs(o["depth"][n][hit] - rw[hit]) / rw[hit]
        # Snapping moves each vertex by <= sqrt(2)/512 px.  Inside a triangle that is the same as
        # evaluating the unsnapped affine function 1/w at a point moved by a convex combination of the
        # three shifts, so |d(depth)/depth| <= |grad_px(1/w)| * w * sqrt(2)/512 (+ float32 rounding).
        # A near-clipped triangle lies in the same plane with its new vertices on the old edges, so the
        # same bound holds for it.
        g = _rel_inv_w_gradient(tri, rid, rw, wl.width, wl.height, wl.fx, wl.fy)[hit]
        unclipped = (-tri[:, :, 2]).min(axis=1)[rid[hit]] >= wl.znear
        bound = g * (np.sqrt(2.0) / 512.0) * 1.02 + 2e-6
        n_unclipped += int(unclipped.sum())
        n_clipped += int((~unclipped).sum())
        assert np.all(rel <= bound), float((rel / bound).max())
        dc = np.abs(o["rgb"][n][hit].astype(float) - rrgb[hit])
        assert np.quantile(dc, 0.99) <= 1.0 and dc.max() <= 6.0, (np.quantile(dc, 0.99), dc.max())
        assert np.all(o["depth"][n][rid < 0][same[rid < 0]] == 0.0)
    assert n_unclipped > 20 and n_clipped > 1000   # both kinds of triangle are exercised (config 0 is mostly clipped)


# --------------------------------------------------------------------------------------------
# N4 near clip
# --------------------------------------------------------------------------------------------

def _floor_soup(n_cells, rng=None):
    """A horizontal floor 1.2 m below the camera from 2 m behind it to 6 m ahead, as an n x n grid."""
    xs = np.linspace(-8, 8, n_cells + 1)   # wide enough to span the 90-degree FoV out to w = 6
    zs = np.linspace(2, -6, n_cells + 1)   # camera space z; w = -z
    tris = []
    for i in range(n_cells):
        for j in range(n_cells):
            a = (xs[i], -1.2, zs[j]); b = (xs[i + 1], -1.2, zs[j]); c = (xs[i + 1], -1.2, zs[j + 1]); d = (xs[i], -1.2, zs[j + 1])
            tris += [[a, b, c], [a, c, d]]
    t = np.array(tris)
    v = np.zeros((t.shape[0], 3, 6), np.float32)
    v[:, :, 0] = t[:, :, 0]; v[:, :, 1] = t[:, :, 1]; v[:, :, 2] = -t[:, :, 2]
    v[:, :, 3:] = 128
    return v


def test_near_clip_invariants(oracle_mod):
    W = H = 64
    znear = 0.5
    coarse = oracle_mod.raster_soup(W, H, 1.0, 1.0, znear, 20.0, _floor_soup(1), np.arange(2), want_count=True)
    fine = oracle_mod.raster_soup(W, H, 1.0, 1.0, znear, 20.0, _floor_soup(37), np.arange(2 * 37 * 37), want_count=True)
    # the floor plane y=-1.2 seen by a level camera: pixel row j sees it at w = 1.2 / tan(angle below horizon)
    yndc = 1 - (np.arange(H) + 0.5) / H * 2
    with np.errstate(divide="ignore"):
        w_row = np.where(yndc < 0, 1.2 / -yndc, np.inf)
    vis = (w_row >= znear * 1.05) & (w_row <= 5.9)
    gone = (w_row < znear * 0.95) | ~np.isfinite(w_row)
    for o in (coarse, fine):
        assert o["count"].max() == 1                      # clipped pieces never overlap or double-cover
        assert np.all(o["count"][vis] == 1)               # exactly once where the plane is in front of the near plane
        assert np.all(o["count"][gone] == 0)              # nothing from behind the near plane
        d = o["depth"][o["id"] != BG]
        assert d.min() >= znear * (1 - 1e-6)
        rows = np.nonzero(vis)[0]
        assert np.allclose(o["depth"][rows, :], w_row[rows, None], rtol=2e-3)
    diff = np.nonzero((coarse["count"] != fine["count"]).any(1))[0]
    assert np.all(np.abs(w_row[diff] - znear) < 0.1 * znear)   # tessellation only matters at the clip line


def test_near_clip_keeps_shared_edges_watertight(oracle_mod):
    rng = np.random.default_rng(9)
    W = H = 48
    znear = 0.4
    n = 14
    # bumpy tilted sheet that dives through the near plane; shared vertices; random rotation of corners
    gx, gz = np.meshgrid(np.linspace(-3, 3, n + 1), np.linspace(1.0, -5.0, n + 1), indexing="ij")
    # (height jitter kept below the grazing slope 0.6/5 so the sheet never folds over itself in the view)
    y = -0.6 + 0.15 * gx + rng.uniform(-0.01, 0.01, gx.shape)
    P = np.stack([gx + rng.uniform(-0.05, 0.05, gx.shape), y, gz + rng.uniform(-0.05, 0.05, gx.shape)], -1)
    tris = []
    for i in range(n):
        for j in range(n):
            a, b, c, d = P[i, j], P[i + 1, j], P[i + 1, j + 1], P[i, j + 1]
            for t in (([a, b, c], [a, c, d]) if rng.random() < 0.5 else ([a, b, d], [b, c, d])):
                k = rng.integers(0, 3)
                t = t[k:] + t[:k]
                tris.append(t if rng.random() < 0.5 else [t[0], t[2], t[1]])
    t = np.array(tris)
    v = np.zeros((t.shape[0], 3, 6), np.float32)
    v[:, :, 0] = t[:, :, 0]; v[:, :, 1] = t[:, :, 1]; v[:, :, 2] = -t[:, :, 2]
    v[:, :, 3:] = 50
    o = oracle_mod.raster_soup(W, H, 1.0, 1.0, znear, 50.0, v, np.arange(t.shape[0]), want_count=True)
    assert o["count"].max() == 1
    rid, rw, _, _, edge = _raycast(t, np.zeros((t.shape[0], 3, 3)), W, H, 1.0, 1.0, znear, 50.0)
    far_from_border = np.zeros_like(edge)
    # interior of the sheet well in front of the near plane must be covered exactly once
    inside = (rid >= 0) & (rw > znear * 1.1)
    # ignore the outer silhouette of the sheet: erode by one pixel
    er = inside.copy()
    er[1:, :] &= inside[:-1, :]; er[:-1, :] &= inside[1:, :]; er[:, 1:] &= inside[:, :-1]; er[:, :-1] &= inside[:, 1:]
    assert er.sum() > 200
    assert np.all(o["count"][er] == 1)
    assert np.all(o["count"][(rid < 0) & ~_dilate(rid >= 0)] == 0)


def _dilate(m):
    d = m.copy()
    d[1:, :] |= m[:-1, :]; d[:-1, :] |= m[1:, :]; d[:, 1:] |= m[:, :-1]; d[:, :-1] |= m[:, 1:]
    return d


# --------------------------------------------------------------------------------------------
# N7 depth, N8 colour, far plane
# --------------------------------------------------------------------------------------------

def test_depth_exact_for_power_of_two(oracle_mod):
    W = H = 32
    for w in (0.5, 1.0, 4.0, 16.0):
        XY = [[(256 * 4 + 3, 256 * 5 + 77), (256 * 19 + 200, 256 * 6 + 1), (256 * 9 + 128, 256 * 20 + 130)]]
        o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, W, H, w=w), [0])
        cov = o["id"] == 0
        assert cov.sum() > 50
        assert np.all(o["depth"][cov] == np.float32(w))


def test_depth_and_far_plane_tilted(oracle_mod):
    # one big triangle receding from w=1 (bottom) to w=40 (top); zfar=10 cuts it
    W = H = 64
    v = np.zeros((1, 3, 6), np.float32)
    v[0, 0, :3] = (-3 * 1, -0.9 * 1, 1)
    v[0, 1, :3] = (3 * 1, -0.9 * 1, 1)
    v[0, 2, :3] = (0.0, 0.9 * 40, 40)
    v[0, :, 3:] = 255
    o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 10.0, v, [7])
    tri = np.array([[[-3, -0.9, -1], [3, -0.9, -1], [0, 36.0, -40]]], float)
    rid, rw, _, _, edge = _raycast(tri, np.zeros((1, 3, 3)), W, H, 1.0, 1.0, 0.1, 1e9)
    hit = (o["id"] == 7)
    assert hit.sum() > 100
    assert np.all(o["depth"][hit] <= 10.0)
    inner = (rid == 0) & ~edge
    assert np.all(hit[inner & (rw < 9.99)]) and not np.any(hit[inner & (rw > 10.01)])
    # snapping bound on the relative depth error (see test_whole_image_vs_raycast_config0)
    sel = hit & inner
    g = _rel_inv_w_gradient(tri, rid, rw, W, H, 1.0, 1.0)[sel]
    rel = np.abs(o["depth"][sel] - rw[sel]) / rw[sel]
    assert np.all(rel <= g * (np.sqrt(2.0) / 512.0) * 1.02 + 2e-6), float(rel.max())


def test_colour_constant_and_affine(oracle_mod):
    W = H = 32
    XY = np.array([[(256 * 2, 256 * 2), (256 * 30, 256 * 3), (256 * 10, 256 * 29)]])
    col = np.zeros((1, 3, 3), np.float32)
    col[0, :, :] = (13, 250, 97)
    o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, W, H, colors=col), [0])
    cov = o["id"] == 0
    assert np.all(o["rgb"][cov] == np.array([13, 250, 97], np.uint8))
    assert np.all(o["rgb"][~cov] == 0)
    # fronto-parallel -> perspective-correct interpolation reduces to affine barycentric interpolation
    col[0] = [[255, 0, 10], [0, 255, 20], [0, 0, 250]]
    o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, W, H, w=4.0, colors=col), [0])
    T = np.array([[XY[0, 0, 0], XY[0, 1, 0], XY[0, 2, 0]], [XY[0, 0, 1], XY[0, 1, 1], XY[0, 2, 1]], [1, 1, 1]], float)
    for j in range(H):
        for i in range(W):
            if cov[j, i]:
                lam = np.linalg.solve(T, np.array([256 * i + 128, 256 * j + 128, 1.0]))
                exp = lam @ col[0].astype(float)
                assert np.all(np.abs(o["rgb"][j, i].astype(float) - exp) <= 0.5 + 1e-3), (i, j)


def test_colour_perspective_correct(oracle_mod):
    # receding triangle with a colour ramp along depth: screen-space-linear interpolation would be far off
    W = H = 64
    tri = np.array([[[-2, -1, -1], [2, -1, -1], [0, 8.0, -16]]], float)
    col = np.array([[[255, 0, 0], [255, 0, 0], [0, 255, 0]]], float)
    v = np.zeros((1, 3, 6), np.float32)
    v[0, :, 0] = tri[0, :, 0]; v[0, :, 1] = tri[0, :, 1]; v[0, :, 2] = -tri[0, :, 2]; v[0, :, 3:] = col[0]
    o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 100.0, v, [0])
    rid, rw, rrgb, _, edge = _raycast(tri, col, W, H, 1.0, 1.0, 0.1, 100.0)
    sel = (o["id"] == 0) & (rid == 0) & ~edge
    assert sel.sum() > 300
    assert np.max(np.abs(o["rgb"][sel].astype(float) - rrgb[sel])) <= 1.0
    assert np.ptp(o["rgb"][sel][:, 1].astype(int)) > 100   # the ramp is actually exercised


# --------------------------------------------------------------------------------------------
# N9 resolve
# --------------------------------------------------------------------------------------------

def test_processing_order_does_not_matter(oracle_mod):
    wl = gen.make_config(0)
    tri, col = _camera_space_triangles(wl, 1)
    v = np.zeros((tri.shape[0], 3, 6), np.float32)
    v[:, :, 0] = tri[:, :, 0]; v[:, :, 1] = tri[:, :, 1]; v[:, :, 2] = -tri[:, :, 2]; v[:, :, 3:] = col
    # add exact duplicates so that exact depth ties exist
    v = np.concatenate([v, v[:40]])
    ids = np.arange(v.shape[0], dtype=np.uint32)
    base = oracle_mod.raster_soup(64, 64, 1.0, 1.0, 0.1, 20.0, v, ids)
    rng = np.random.default_rng(1)
    for _ in range(3):
        p = rng.permutation(v.shape[0])
        o = oracle_mod.raster_soup(64, 64, 1.0, 1.0, 0.1, 20.0, v[p], ids[p])
        for k in ("rgb", "depth", "id", "sub"):
            assert np.array_equal(o[k], base[k]), k
    assert not np.any((base["id"] >= tri.shape[0]) & (base["id"] != BG))   # of two coincident triangles the lower id wins
    # permuting the ids changes only pixels with an exact depth tie (here: the duplicated triangles)
    ids2 = ids.copy()
    ids2[:40], ids2[tri.shape[0]:] = ids[tri.shape[0]:], ids[:40]
    o = oracle_mod.raster_soup(64, 64, 1.0, 1.0, 0.1, 20.0, v, ids2)
    assert np.array_equal(o["depth"], base["depth"]) and np.array_equal(o["rgb"], base["rgb"])
    assert np.array_equal(o["id"], base["id"])   # winner is still the lower of the two ids {i, i+nt}


def test_coincident_triangles_lowest_id(oracle_mod):
    XY = np.array([[(100, 100), (7000, 300), (2000, 6000)]] * 3)
    for ids in ([5, 3, 9], [9, 5, 3], [3, 9, 5]):
        o = oracle_mod.raster_soup(32, 32, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(XY, 32, 32), ids)
        assert set(np.unique(o["id"])) == {3, BG}


# --------------------------------------------------------------------------------------------
# batch entry point: ids, instance slots, env independence
# --------------------------------------------------------------------------------------------

def test_render_ids_and_empty_slots(oracle_mod):
    wl = gen.make_config(0)
    full = oracle_mod.render(wl)
    ns = wl.static_meshes[0].nt
    assert full["id"][full["id"] != BG].max() < ns + 24
    assert (full["id"][full["id"] != BG] >= ns).any()      # cubes are visible somewhere
    # emptying slot 0 renumbers slot 1's triangles down by 12 and removes slot 0's fragments
    wl2 = wl.subset(np.arange(wl.N))
    wl2.inst_mesh = wl.inst_mesh.copy()
    wl2.inst_mesh[:, 0] = -1
    o2 = oracle_mod.render(wl2)
    was1 = (full["id"] >= ns + 12) & (full["id"] != BG)
    assert np.array_equal(o2["id"][was1], full["id"][was1] - 12)
    assert not np.any((o2["id"] >= ns + 12) & (o2["id"] != BG))
    # environments are independent: a subset renders to the same rows
    sub = oracle_mod.render(wl.subset([2, 0]))
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(sub[k][0], full[k][2]) and np.array_equal(sub[k][1], full[k][0])
    # threads do not change anything
    one = oracle_mod.render(wl, n_threads=1)
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(one[k], full[k])


def test_generators_are_subset_reproducible():
    a = gen.make_config(1, n_envs=6)
    b = gen.make_config(1, env_ids=[4, 1])
    assert np.array_equal(b.cam_pose, a.cam_pose[[4, 1]]) and np.array_equal(b.inst_xform, a.inst_xform[[4, 1]])
    assert a.static_meshes[0].nt == 50_000 and [m.nt for m in a.dyn_meshes] == [980, 400, 400, 400, 400, 400]
    assert a.K == 25 and np.all(a.tris_per_env() == 71_600)


# ---------------------------------------------------------------------------------------------------
# N11: packed observation (NEXT-1).  Pins: closed forms (dyadic values that binary16 holds exactly), the
# hand-written binary32 -> binary16 conversion against numpy's (a library routine, round-to-nearest-even) on
# every binary16 value, every midpoint between neighbours and random floats, and the layout.
# ---------------------------------------------------------------------------------------------------
def test_n11_half_conversion_matches_numpy_and_closed_forms(oracle_mod):
    # exact cases
    x = np.array([0.0, 1.0, 0.5, 0.25, 2.0 ** -14, 2.0 ** -24, 65504.0, 1.0 / 3.0, 2.0 ** -25, 1e-10, 70000.0], np.float32)
    got = oracle_mod.half_rn(x)
    assert got[0] == 0 and got[1] == 0x3C00 and got[2] == 0x3800 and got[3] == 0x3400
    assert got[4] == 0x0400 and got[5] == 0x0001 and got[6] == 0x7BFF
    assert got[7] == 0x3555                         # 1/3 -> 0.33325195 (nearest)
    assert got[8] == 0x0000                         # exactly half of the smallest subnormal: tie -> even (0)
    assert got[9] == 0 and got[10] == 0x7C00
    # every finite non-negative binary16 value converts to itself; every midpoint goes to the even neighbour
    h = np.arange(0, 0x7C00, dtype=np.uint16)
    v = h.view(np.float16).astype(np.float32)
    assert np.array_equal(oracle_mod.half_rn(v), h)
    mid = ((v[:-1].astype(np.float64) + v[1:].astype(np.float64)) / 2).astype(np.float32)   # exact in binary32
    exp = np.where(h[:-1] % 2 == 0, h[:-1], h[1:])
    assert np.array_equal(oracle_mod.half_rn(mid), exp)
    # random floats against numpy's conversion
    rng = np.random.Generator(np.random.Philox(key=[5, 11]))
    r = np.concatenate([rng.uniform(0, 1, 200000), rng.uniform(0, 2 ** -13, 50000), rng.uniform(0, 70000, 50000)]).astype(np.float32)
    with np.errstate(over="ignore"):
        assert np.array_equal(oracle_mod.half_rn(r), r.astype(np.float16).view(np.uint16))


def test_n11_pack_obs_layout_and_values(oracle_mod):
    rng = np.random.Generator(np.random.Philox(key=[5, 12]))
    N, H, W = 2, 4, 6
    rgb = rng.integers(0, 256, (N, H, W, 3)).astype(np.uint8)
    depth = rng.uniform(0, 12, (N, H, W)).astype(np.float32)
    depth[0, 0, 0] = 0.0            # background
    depth[0, 0, 1] = 0.5            # = dmin
    depth[0, 0, 2] = 10.5           # = dmax
    depth[0, 0, 3] = 5.5            # midpoint
    depth[0, 0, 4] = 11.0           # beyond dmax
    rgb[0, 0, 0] = (0, 255, 51)     # 51/255 = 0.2
    o = oracle_mod.pack_obs(rgb, depth, 0.5, 10.5)
    assert o.shape == (N, 4, H, W)
    f = o.view(np.float16).astype(np.float64)
    assert f[0, 0, 0, 0] == 0.0 and f[0, 1, 0, 0] == 1.0 and abs(f[0, 2, 0, 0] - 0.2) < 2 ** -12
    assert f[0, 3, 0, 0] == 0.0 and f[0, 3, 0, 1] == 0.0 and f[0, 3, 0, 2] == 1.0 and f[0, 3, 0, 3] == 0.5 and f[0, 3, 0, 4] == 1.0
    # the whole tensor against numpy float32 arithmetic + numpy's binary16 conversion
    ref = np.empty((N, 4, H, W), np.float16)
    ref[:, :3] = (rgb.astype(np.float32) / np.float32(255.0)).transpose(0, 3, 1, 2).astype(np.float16)
    ref[:, 3] = ((np.clip(depth, np.float32(0.5), np.float32(10.5)) - np.float32(0.5)) / np.float32(10.0)).astype(np.float16)
    assert np.array_equal(o, ref.view(np.uint16))
    with pytest.raises(ValueError):
        oracle_mod.pack_obs(rgb, depth, 1.0, 1.0)


# --------------------------------------------------------------------------------------------
# equality boundaries of N3 / N5 / N7 / N9 (each is a separate clause of the definition)
# --------------------------------------------------------------------------------------------

def test_snap_is_round_half_even(oracle_mod):
    """N5: X lands on exactly k + 0.5 sub-pixel units; ties go to the even integer (rintf), which
    floor(x + 0.5) gets wrong for every even k.  Values derived by hand in tests/golden/vertex_closed_form.txt;
    here the same construction over many k, expected values from exact rationals."""
    from fractions import Fraction as F
    W = H = 64
    ks = list(range(4090, 4110)) + list(range(12280, 12300))
    pos = np.array([[float(F(2 * k + 1 - 2 * 8192, 8192)), float(-F(2 * k + 1 - 2 * 8192, 8192)), -2.0] for k in ks], np.float32)
    for k, p in zip(ks, pos):   # the inputs are exact in binary32
        assert F(float(p[0])) == F(2 * k + 1 - 2 * 8192, 8192)
    o = oracle_mod.vertex_stage(W, H, 1.0, 1.0, 0.1, 20.0, _pose("I"), None, pos)
    want = np.array([k if k % 2 == 0 else k + 1 for k in ks])   # nearest even of k + 1/2
    assert np.array_equal(o["Xi"], want)
    assert np.array_equal(o["Yi"], want)
    # the same rule on the raster path (N5 inside the triangle pipeline): a quad whose corners land on exactly
    # 256 i + 128.5 snaps to 256 i + 128 (even), i.e. onto the pixel centres: by the closed form of
    # test_quad_closed_form it then covers columns 5..19 and rows 7..12 (left/top inclusive, right/bottom
    # exclusive).  Rounding half up would give 256 i + 129 and shift the cover to columns 6..20, rows 8..13.
    W = H = 64
    x0, x1, y0, y1 = 256 * 5 + 128.5, 256 * 20 + 128.5, 256 * 7 + 128.5, 256 * 13 + 128.5
    XY = [[(x0, y0), (x1, y0), (x1, y1)], [(x0, y0), (x1, y1), (x0, y1)]]
    soup = _soup_from_snapped(XY, W, H, w=2.0)
    assert np.all(soup[:, :, :2].astype(np.float64) * 4096 % 0.5 == 0)   # inputs exact in binary32
    r = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, soup, [0, 1], want_count=True)
    want_cov = np.zeros((H, W), bool)
    want_cov[7:13, 5:20] = True
    assert np.array_equal(r["id"] != BG, want_cov) and r["count"].max() == 1


def test_vertex_on_the_near_plane_is_inside(oracle_mod):
    """N3: inside iff w >= znear, so a triangle with a vertex at exactly w == znear is not clipped.  Not being
    clipped is observable without knowing any formula: with znear lowered by one ulp all three vertices are
    strictly inside, and the two images must be bit-identical.  If the vertex counted as outside, N4 would
    rebuild it as fma(1, x_out - x_in, x_in), which rounds (x_in is large and not dyadic), and the snapped
    corner, and with it the depth bits, would move."""
    W = H = 256
    zn = np.float32(0.5)
    v = np.zeros((1, 3, 6), np.float32)
    v[0, 0] = (-1003.7, 0.3, 3.0, 250, 10, 30)     # far off-screen to the left: large, non-dyadic x
    v[0, 1] = (0.9, -777.77, 2.0, 20, 240, 60)
    v[0, 2] = (0.1, 0.2, zn, 90, 80, 255)          # exactly on the near plane
    below = float(np.nextafter(zn, np.float32(0)))
    for perm in ((0, 1, 2), (1, 2, 0), (2, 0, 1), (0, 2, 1)):
        vv = np.ascontiguousarray(v[:, list(perm)])
        a = oracle_mod.raster_soup(W, H, 1.0, 1.0, float(zn), 20.0, vv, [3], want_count=True)
        b = oracle_mod.raster_soup(W, H, 1.0, 1.0, below, 20.0, vv, [3], want_count=True)
        assert (a["id"] == 3).sum() > 1000
        assert a["count"].max() == 1 and a["sub"].max() == 0
        for k in ("id", "rgb", "count"):
            assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a["depth"].view(np.uint32), b["depth"].view(np.uint32))
    # and the vertex stage says so directly
    o = oracle_mod.vertex_stage(64, 64, 1.0, 1.0, 0.5, 20.0, _pose("I"), None,
                                np.array([[0.0, 0.0, -0.5], [0.0, 0.0, np.nextafter(np.float32(-0.5), np.float32(0))]], np.float32))
    assert list(o["inside"]) == [1, 0]


def test_far_plane_is_inclusive(oracle_mod):
    """N7: a fragment is dropped iff depth > zfar.  A fronto-parallel quad of <= 16x16 px at a power-of-two depth d
    has depth exactly d at every covered pixel (test_depth_exact_for_power_of_two), so with zfar == d it is kept
    and with zfar one ulp below d it is dropped, entirely."""
    W = H = 32
    d = 16.0
    x0, y0, x1, y1 = 256 * 5 + 7, 256 * 9 + 200, 256 * 18 + 130, 256 * 21 + 1
    XY = [[(x0, y0), (x1, y0), (x1, y1)], [(x0, y0), (x1, y1), (x0, y1)]]
    soup = _soup_from_snapped(XY, W, H, w=d)
    keep = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, d, soup, [0, 1])
    cov = keep["id"] != BG
    # pixel centres with x0 <= 256i+128 < x1 (i = 5..18) and y0 <= 256j+128 < y1 (j = 10..20)
    assert cov.sum() == 14 * 11 and cov[10:21, 5:19].all()
    assert np.all(keep["depth"][cov] == np.float32(d))
    drop = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, float(np.nextafter(np.float32(d), np.float32(0))), soup, [0, 1])
    assert np.all(drop["id"] == BG) and np.all(drop["depth"] == 0.0) and np.all(drop["rgb"] == 0)


def test_clip_pieces_tie_goes_to_sub_zero(oracle_mod):
    """N9, third key: the two pieces of a near-clipped triangle keep the parent id; where both cover a pixel at
    exactly equal depth, sub 0 wins.  Construction: vertex a sits exactly on a pixel centre at w = 1 (q = 1) and
    just inside a near plane at 1 - 2^-k, so the second piece (a, P(b,c), P(a,c)) is a sliver whose apex a can
    land on either side of its base after snapping; when it folds over the first piece, the pixel at a is covered
    by both (count == 2).  At that pixel the edge functions of both pieces are (A, 0, 0), so depth = A / (A * 1)
    = 1 exactly in both: an exact tie.  The search is seeded and bounded; it uses only the coverage count."""
    W = H = 16
    hw = 128.0 * W
    rng = np.random.default_rng(11)
    found = 0
    for _ in range(40000):
        i, j = rng.integers(2, 14, 2)
        zn = np.float32(1.0 - 2.0 ** -int(rng.integers(8, 22)))
        a = [(256 * i + 128 - hw) / hw, -(256 * j + 128 - hw) / hw, 1.0]
        wb, wc = np.float32(rng.uniform(1.0, 3.0)), np.float32(rng.uniform(0.2, 0.999))
        b = [rng.uniform(-1, 1) * wb, rng.uniform(-1, 1) * wb, wb]
        c = [rng.uniform(-1, 1) * wc, rng.uniform(-1, 1) * wc, wc]
        v = np.zeros((1, 3, 6), np.float32)
        for s, p in zip(rng.permutation(3), (a, b, c)):
            v[0, s, :3] = p
        v[0, :, 3:] = rng.integers(0, 256, (3, 3))
        o = oracle_mod.raster_soup(W, H, 1.0, 1.0, float(zn), 20.0, v, [5], want_count=True)
        if o["count"][j, i] == 2:
            found += 1
            assert o["id"][j, i] == 5
            assert o["depth"][j, i] == np.float32(1.0)     # the exact tie
            assert o["sub"][j, i] == 0
            if found >= 6:
                break
    assert found >= 6, found


def test_colour_rounds_half_to_even(oracle_mod):
    """N8: `rintf(v)` -- an exact tie goes to the even integer.  floor(v + 0.5) differs at every
    even m + 1/2, which the +-0.5 bound of test_colour_constant_and_affine cannot see.
    Construction, every value by hand: a fronto-parallel right triangle at w = 2 (q = 1/2 exactly) with corners
    v0 = (3, 4.5) px, v1 = (11, 4.5) px, v2 = (3, 12.5) px, so A = 2048 * 2048 = 2^22.  Vertices 0 and 1 carry the
    colour a, vertex 2 carries a + b with b odd.  On pixel row 8 (centre y = 8.5 px, half way down) the weight of
    vertex 2 is E_2 / A = 1/2 for every covered pixel, all products and sums are integers below 2^30 with few
    significant bits (exact in binary32), so v = a + b / 2 = a + m + 1/2 exactly with b = 2 m + 1: the byte must be
    a + m for even a + m and a + m + 1 for odd a + m."""
    W = H = 16
    XY = [[(256 * 3, 256 * 4 + 128), (256 * 11, 256 * 4 + 128), (256 * 3, 256 * 12 + 128)]]
    row = 8
    # row 8: covered from x = 3 px to the hypotenuse at x = 3 + 8 * (1 - 1/2) = 7 px: centres 3.5 .. 6.5 (7.5 is outside)
    cols = [3, 4, 5, 6]
    checked_even = checked_odd = 0
    for a in (0, 10, 101):
        for b0 in range(1, 256 - a, 6):
            bs = [b for b in (b0, b0 + 2, b0 + 4) if a + b <= 255]
            while len(bs) < 3:
                bs.append(bs[-1])
            col = np.zeros((1, 3, 3), np.float32)
            col[0, 0, :] = a
            col[0, 1, :] = a
            col[0, 2, :] = [a + b for b in bs]
            for flip in (0, 1):
                xy = [[XY[0][0], XY[0][2], XY[0][1]]] if flip else XY
                cc = col[:, [0, 2, 1], :] if flip else col
                o = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, _soup_from_snapped(xy, W, H, w=2.0, colors=cc), [0])
                cov = np.nonzero(o["id"][row] == 0)[0]
                assert list(cov) == cols
                for ch, b in enumerate(bs):
                    m = (b - 1) // 2                      # v = a + m + 1/2
                    lo = a + m
                    want = lo if lo % 2 == 0 else lo + 1
                    assert np.all(o["rgb"][row, cols, ch] == want), (a, b, flip, o["rgb"][row, cols, ch], want)
                    checked_even += lo % 2 == 0
                    checked_odd += lo % 2 == 1
    assert checked_even > 50 and checked_odd > 50


def test_snap_clamps_at_two_to_the_28(oracle_mod):
    """N5: X and Y are clamped to +-2^28 before the conversion ('clamp to +-2^28 with fminf/fmaxf').
    By hand at W = H = 128 (hw = hh = 16384), identity camera, fx = fy = 1, w = 1/8 (q = 8, inside: w >= znear):
      x = 4096  -> X = 4096 * 8 * 16384 + 16384 = 2^29 + 2^14  -> clamped to  2^28;   x = -4096 -> -2^29 + 2^14 -> -2^28
      y = 4096  -> Y = -(2^29) + 2^14 -> -2^28;                                        y = -4096 -> +2^28
      x = 256   -> X = 256 * 8 * 16384 + 16384 = 2^25 + 2^14 = 33570816: large, inside the clamp, exact in binary32
      x = 2047.875 (= 2^11 - 2^-3) -> X = (2^14 - 1) * 16384 + 16384 = 2^28 exactly: the largest unclamped value."""
    W = H = 128
    L = 1 << 28
    pos = np.array([[4096.0, 4096.0, -0.125], [-4096.0, -4096.0, -0.125], [256.0, -256.0, -0.125],
                    [2047.875, -2047.875, -0.125], [1.0e6, -1.0e6, -0.125]], np.float32)
    o = oracle_mod.vertex_stage(W, H, 1.0, 1.0, 0.1, 20.0, _pose("I"), None, pos)
    assert np.all(o["inside"] == 1)
    assert list(o["Xi"]) == [L, -L, (1 << 25) + (1 << 14), L, L]
    assert list(o["Yi"]) == [-L, L, (1 << 25) + (1 << 14), L, L]
    # the raster path (N5 inside the triangle pipeline) clamps the same way: a triangle with one corner far to the
    # right, v2 = (x = 4096, y = 0, w = 1/8) -> (2^28, 16384) after the clamp, and two corners on the screen at w = 2.
    # Its upper edge leaves v0 one sub-pixel above the centres of pixel row 20 and sinks so slowly that where it
    # crosses that row of centres depends on where v2 ends up: at 2^28 it crosses inside the frame (near column 104),
    # unclamped (2^29 + 2^14) it would not cross at all, at 2^24 it would cross near column 16.  Expected coverage: the
    # plain inequality definition in exact integers on the clamped corner.
    X0, Y0, Y1 = 256 * 10, 256 * 20 + 127, 256 * 100
    on = _soup_from_snapped([[(X0, Y0), (X0, Y1), (X0, Y1)]], W, H, w=2.0)[0]
    soup = np.zeros((1, 3, 6), np.float32)
    soup[0, 0] = on[0]
    soup[0, 1] = on[1]
    soup[0, 2] = [4096.0, 0.0, 0.125, 200.0, 200.0, 200.0]
    r = oracle_mod.raster_soup(W, H, 1.0, 1.0, 0.1, 20.0, soup, [0])
    got = r["id"] != BG
    corners = [(X0, Y0), (X0, Y1), (L, 128 * H)]
    want = np.zeros((H, W), bool)
    for j in range(H):
        for i in range(W):
            want[j, i] = _covered_exact(corners, 256 * i + 128, 256 * j + 128)
    assert np.array_equal(got, want), int((got != want).sum())
    # the pin really depends on the clamp value: the other two candidate corners give other images
    for other in ((1 << 29) + (1 << 14), 1 << 24):
        alt = [(X0, Y0), (X0, Y1), (other, 128 * H)]
        assert any(_covered_exact(alt, 256 * i + 128, 256 * 20 + 128) != want[20, i] for i in range(W)), other
    assert want[20].any() and not want[20].all()
