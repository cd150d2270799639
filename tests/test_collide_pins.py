"""Pins of the oracle's batch collision queries N13 (PAPER.md:111-119 and Appendix G,
PAPER.md:443-459).  The paper prints no worked example, so the pins are closed forms (hand-made column grids, a
sphere touching a box face and a box corner at exactly its radius with dyadic numbers), the special cases the
definition names (inclusive layer bounds, nearest column with ties to even, outside the grid, empty and held
slots, lowest slot wins) and a float64 brute force on random inputs.  CPU only; GPU parity: tests/test_gpu_collide.py."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2306_07552_b200 import gen

I44 = np.eye(4, dtype=np.float32).reshape(16)


def _grid(x0, z0, sp, nx, nz, cols):
    """cols[iz][ix] = list of (lo, hi)"""
    off, lay = [0], []
    for iz in range(nz):
        for ix in range(nx):
            lay += cols[iz][ix]
            off.append(len(lay))
    return gen.ColumnGrid(x0, z0, sp, nx, nz, np.asarray(off, np.uint32), np.asarray(lay, np.float32).reshape(-1, 2))


def _boxmesh(lo, hi):
    p = np.array([[x, y, z] for x in (lo[0], hi[0]) for y in (lo[1], hi[1]) for z in (lo[2], hi[2])], np.float32)
    return gen.Mesh(p, np.zeros((8, 3), np.uint8), np.array([[0, 1, 2]], np.uint32))


def _query(oracle_mod, centres, rclass, grids, radii, meshes=(), inst_mesh=None, obj_xf=None, held=None, link_xf=None):
    """One environment, one link (slot K-1, transform link_xf), spheres at `centres` in the link frame."""
    n_obj = 0 if inst_mesh is None else len(inst_mesh)
    K = n_obj + 1
    xf = np.tile(I44, (1, K, 1))
    if obj_xf is not None:
        xf[0, :n_obj] = np.asarray(obj_xf, np.float32).reshape(n_obj, 16)
    if link_xf is not None:
        xf[0, K - 1] = np.asarray(link_xf, np.float32).reshape(16)
    im = np.full((1, K), -1, np.int32)
    if inst_mesh is not None:
        im[0, :n_obj] = inst_mesh
    sph = [gen.Sphere(0, rc, tuple(c)) for c, rc in zip(centres, rclass)]
    s, o = oracle_mod.collide(list(meshes), grids, radii, sph, np.zeros(1, np.int32), im, xf, K - 1, 0, n_obj,
                              None if held is None else np.array([held], np.int32))
    return s[0], o[0]


OPEN = [[(-100.0, 100.0)]]


def _open_grid(n_radii=1):
    return [[_grid(-50.0, -50.0, 100.0, 1, 1, [[[(-100.0, 100.0)]]]) for _ in range(n_radii)]]


def test_column_layers_inclusive_bounds_and_linear_search(oracle_mod):
    g = [[_grid(0.0, 0.0, 0.25, 3, 2, [[[(0.5, 1.0), (1.5, 2.0)], [], [(0.25, 2.75)]],
                                       [[(0.125, 0.375)], [(1.0, 1.0)], []]])]]
    below = np.nextafter(np.float32(0.5), np.float32(0)); above = np.nextafter(np.float32(2.0), np.float32(3))
    c = [(0, 0.5, 0), (0, below, 0), (0, 1.0, 0), (0, 1.25, 0), (0, 1.5, 0), (0, 2.0, 0), (0, above, 0),   # column (0,0): two layers
         (0.25, 1.0, 0), (0.5, 1.0, 0),                                                                      # (1,0) closed, (2,0) open
         (0, 0.25, 0.25), (0, 1.0, 0.25), (0.25, 1.0, 0.25), (0.5, 1.0, 0.25)]                              # row iz = 1
    s, _ = _query(oracle_mod, c, [0] * len(c), g, [0.05])
    assert list(s) == [0, 1, 0, 1, 0, 0, 1, 1, 0, 0, 1, 0, 1]


def test_nearest_column_ties_to_even_and_outside(oracle_mod):
    # columns 0 and 2 open, column 1 closed: x = 0.5 and 1.5 spacings are ties (-> 0 and 2), 0.51 -> 1
    g = [[_grid(1.0, -2.0, 0.5, 3, 1, [[[(0.0, 9.0)], [], [(0.0, 9.0)]]])]]
    xs = [1.0, 1.25, 1.2578125, 1.5, 1.75, 1.7421875, 2.0, 2.25, 2.2578125, 0.75, 0.7421875]
    s, _ = _query(oracle_mod, [(x, 1.0, -2.0) for x in xs], [0] * len(xs), g, [0.05])
    assert list(s) == [0, 0, 1, 1, 0, 1, 0, 0, 1, 0, 1]      # the last two: -0.5 -> column 0 (tie to even), beyond -> outside
    s, _ = _query(oracle_mod, [(1.0, 1.0, -1.7), (1.0, 1.0, -2.3), (1.0, 1.0, -1.76)], [0, 0, 0], g, [0.05])
    assert list(s) == [1, 1, 0]                               # z rounds to row 1 / -1: outside the grid is obstructed


def test_grid_is_chosen_by_scene_and_radius_class(oracle_mod):
    op, cl = _grid(-50.0, -50.0, 100.0, 1, 1, [[[(-100.0, 100.0)]]]), _grid(-50.0, -50.0, 100.0, 1, 1, [[[]]])
    grids = [[op, cl], [cl, op]]
    sph = [gen.Sphere(0, 0, (0, 0, 0)), gen.Sphere(0, 1, (0, 0, 0))]
    xf = np.tile(I44, (2, 1, 1))
    s, _ = oracle_mod.collide([], grids, [0.05, 0.12], sph, np.array([0, 1], np.int32), np.full((2, 1), -1, np.int32), xf, 0, 0, 0)
    assert s.tolist() == [[0, 1], [1, 0]]


def test_sphere_box_touching_face_corner_inside(oracle_mod):
    m = _boxmesh((-0.5, -0.25, -0.125), (0.5, 0.25, 0.125))
    r = [0.25, 0.3125]
    far = float(np.nextafter(np.float32(0.75), np.float32(1)))
    c = [(0.75, 0, 0), (far, 0, 0), (0, 0.5, 0), (0, 0, -0.375), (0, 0, 0), (0.4, 0.2, 0.1), (-0.75, 0.25, 0.125)]
    _, o = _query(oracle_mod, c, [0] * len(c), _open_grid(2), r, [m], [0], [I44])
    assert list(o) == [0, -1, 0, 0, 0, 0, 0]
    # corner: offset (3/16, 4/16, 0) from the corner (0.5, 0.25, 0.125): distance exactly 5/16
    c = [(0.6875, 0.5, 0.125), (0.6875, 0.5, 0.125), (float(np.nextafter(np.float32(0.6875), np.float32(1))), 0.5, 0.125), (0.6875, 0.5, 0.15)]
    _, o = _query(oracle_mod, c, [1, 0, 1, 1], _open_grid(2), r, [m], [0], [I44])
    assert list(o) == [0, -1, -1, -1]


def test_box_pose_uses_the_inverse_rotation_and_the_mesh_box_centre(oracle_mod):
    m = _boxmesh((0.0, 0.0, 0.0), (1.0, 0.5, 0.25))          # box not centred on the mesh origin
    Ry = np.array([[0, 0, 1, 2.0], [0, 1, 0, 1.0], [-1, 0, 0, -3.0], [0, 0, 0, 1]], np.float32)   # +90 degrees about Y, then translate
    # world = R local + t: local (1, .5, .25) -> world (2.25, 1.5, -4); the box spans x 2..2.25, y 1..1.5, z -4..-3
    c = [(2.125, 1.25, -3.5), (2.5, 1.25, -3.5), (2.5625, 1.25, -3.5), (2.125, 1.25, -2.75), (2.125, 1.25, -2.6875),
         (1.75, 1.25, -3.5), (1.6875, 1.25, -3.5), (2.125, 1.25, -4.25), (2.125, 0.75, -3.5), (2.125, 0.6875, -3.5)]
    _, o = _query(oracle_mod, c, [0] * len(c), _open_grid(), [0.25], [m], [0], [Ry.reshape(16)])
    assert list(o) == [0, 0, -1, 0, -1, 0, -1, 0, 0, -1]


def test_lowest_slot_wins_empty_and_held_slots_are_skipped(oracle_mod):
    m = _boxmesh((-0.5, -0.5, -0.5), (0.5, 0.5, 0.5))
    far = I44.copy(); far[3] = 10.0
    xfs = [far, far, far, I44, far, I44, I44]
    q = lambda im, held=None: int(_query(oracle_mod, [(0, 0, 0)], [0], _open_grid(), [0.05], [m], im, xfs, held)[1][0])
    assert q([0] * 7) == 3
    assert q([0, 0, 0, -1, 0, 0, 0]) == 5
    assert q([0] * 7, held=3) == 5
    assert q([0, 0, 0, -1, 0, -1, 0], held=6) == -1
    assert q([0] * 7, held=0) == 3


def test_sphere_centre_comes_from_the_link_transform(oracle_mod):
    g = [[_grid(0.0, 0.0, 1.0, 4, 4, [[[(float(iz), float(iz))] if ix == 2 else [] for ix in range(4)] for iz in range(4)])]]
    # link: rotate +90 degrees about Z (x -> y), translate (2, 0, 3): centre (1, 0, 0) -> (2, 1, 3): column (2, 3) wants y == 3
    W = np.array([[0, -1, 0, 2.0], [1, 0, 0, 0.0], [0, 0, 1, 3.0], [0, 0, 0, 1]], np.float32)
    s, _ = _query(oracle_mod, [(3.0, 0, 0), (1.0, 0, 0), (3.0, 0, -1.0), (3.0, 1.0, 0)], [0] * 4, g, [0.05], link_xf=W.reshape(16))
    assert list(s) == [0, 1, 1, 1]       # (2,3,3) free; (2,1,3) not; (2,3,2): column (2,2) wants y == 2; (1,3,3): column 1 closed


def test_random_against_float64_brute_force(oracle_mod):
    ext = (3.0, 3.0, 6.0, 6.0)
    grids = [[gen.column_grid(1, 0, r, ext) for r in gen.SPHERE_RADII]]
    w = gen.collision_world(48, seed=4, extent=ext)
    _, xf = oracle_mod.fk(w["robot"], w["base_pose"], w["joint_pos"], w["K"], w["link_slot0"], inst_xform=w["inst_xform"],
                          held_slot=w["held_slot"], held_xform=w["held_xform"])
    s, o = oracle_mod.collide(w["dyn_meshes"], grids, w["radii"], w["spheres"], w["env_scene"], w["inst_mesh"], xf,
                              w["link_slot0"], 0, w["n_obj"], w["held_slot"])
    assert 0.05 < s.mean() < 0.95 and (o >= 0).mean() > 0.01
    n_checked = 0
    for n in range(48):
        for si, sp in enumerate(w["spheres"]):
            Wl = xf[n, w["link_slot0"] + sp.link].astype(np.float64).reshape(4, 4)
            c = Wl[:3, :3] @ np.asarray(sp.centre, np.float64) + Wl[:3, 3]
            g = grids[0][sp.radius_class]
            fx, fz = (c[0] - g.x0) / g.spacing, (c[2] - g.z0) / g.spacing
            if min(abs(fx - np.floor(fx) - 0.5), abs(fz - np.floor(fz) - 0.5)) > 1e-3:
                ix, iz = int(np.rint(fx)), int(np.rint(fz))
                hit, sure = True, True
                if 0 <= ix < g.nx and 0 <= iz < g.nz:
                    for lo, hi in g.layers[g.col_off[iz * g.nx + ix]:g.col_off[iz * g.nx + ix + 1]].astype(np.float64):
                        if lo <= c[1] <= hi:
                            hit = False
                        if min(abs(c[1] - lo), abs(c[1] - hi)) < 1e-5:
                            sure = False
                if sure:
                    assert s[n, si] == hit, (n, si)
                    n_checked += 1
            r = float(w["radii"][sp.radius_class])
            first, sure = -1, True
            for k in range(w["n_obj"]):
                if w["inst_mesh"][n, k] < 0 or w["held_slot"][n] == k:
                    continue
                P = w["dyn_meshes"][w["inst_mesh"][n, k]].positions.astype(np.float64)
                bc, bh = 0.5 * (P.min(0) + P.max(0)), 0.5 * (P.max(0) - P.min(0))
                M = xf[n, k].astype(np.float64).reshape(4, 4)
                rel = M[:3, :3].T @ (c - M[:3, 3]) - bc
                d = np.linalg.norm(rel - np.clip(rel, -bh, bh))
                if abs(d - r) < 1e-5:
                    sure = False
                    break
                if d <= r:
                    first = k
                    break
            if sure:
                assert o[n, si] == first, (n, si, o[n, si], first)
                n_checked += 1
    assert n_checked > 2000


def test_bad_arguments(oracle_mod):
    with pytest.raises(ValueError):      # radius class out of range
        _query(oracle_mod, [(0, 0, 0)], [3], _open_grid(), [0.05])
    with pytest.raises(AssertionError):  # one grid per (scene, radius)
        _query(oracle_mod, [(0, 0, 0)], [0], _open_grid(), [0.05, 0.12])
    with pytest.raises(ValueError):      # scene index out of range
        oracle_mod.collide([], _open_grid(), [0.05], [gen.Sphere(0, 0, (0, 0, 0))], np.array([1], np.int32),
                           np.full((1, 1), -1, np.int32), np.tile(I44, (1, 1, 1)), 0, 0, 0)


def test_spheres_of_the_grasped_object(oracle_mod):
    """'we approximate the robot (and the current grasped object, if any) with a set of spheres': a
    sphere with link == -1 rides on the object in the gripper, inst_xform[n][held_slot[n]].  By hand:
    column grid with spacing 1, column (ix, iz) free only at height y == iz for ix == 2 (as in the link-transform pin);
    the held object (slot 1) is turned +90 degrees about Z and stands at (2, 0, 3): its sphere at (3, 0, 0) in the
    object's frame is at (2, 3, 3) in the world -> free; at (1, 0, 0) -> (2, 1, 3) -> obstructed.  The robot-link sphere
    (link 0, identity transform in slot 2) at the same local points lands elsewhere: (3, 0, 0) -> column 3, closed.
    Boxes: slot 0 holds a unit cube at the origin shifted to x = 2.5, so it spans x in [2, 3]; the held sphere at world
    (2, 3, 3) is far from it; a held sphere at local (0, 0.25, -3) -> world (1.75, 0, 0) is 0.25 from the face x = 2:
    radius 0.25 touches (inclusive) -> slot 0.  The held object's own box (slot 1) is never reported.
    With nothing held (held_slot -1, or no held_slot array) the sphere does not exist: (0, -1)."""
    g = [[_grid(0.0, 0.0, 1.0, 4, 4, [[[(float(iz), float(iz))] if ix == 2 else [] for ix in range(4)] for iz in range(4)])]]
    cube = _boxmesh((-0.5, -0.5, -0.5), (0.5, 0.5, 0.5))
    Hm = np.array([[0, -1, 0, 2.0], [1, 0, 0, 0.0], [0, 0, 1, 3.0], [0, 0, 0, 1]], np.float32).reshape(16)
    box = I44.copy(); box[3] = 2.5
    K = 3
    xf = np.stack([box, Hm, I44]).reshape(1, K, 16)
    im = np.array([[0, 0, -1]], np.int32)
    sph = [gen.Sphere(-1, 0, (3.0, 0.0, 0.0)), gen.Sphere(-1, 0, (1.0, 0.0, 0.0)), gen.Sphere(0, 0, (3.0, 0.0, 0.0)),
           gen.Sphere(-1, 0, (0.0, 0.25, -3.0)), gen.Sphere(-1, 0, (0.0, 0.2578125, -3.0)), gen.Sphere(-1, 0, (0.0, 0.0, 0.0))]
    call = lambda held: oracle_mod.collide([cube], g, [0.25], sph, np.zeros(1, np.int32), im, xf, 2, 0, 2, held)
    s, o = call(np.array([1], np.int32))
    # world centres: (2,3,3) free | (2,1,3) column (2,3) wants y == 3 | link sphere (3,0,0): column 3 is closed |
    # (1.75,0,0) and (1.7421875,0,0): nearest column (2,0), free at y == 0 | (2,0,3): column (2,3) wants y == 3
    assert list(s[0]) == [0, 1, 1, 0, 0, 1]
    assert list(o[0]) == [-1, -1, 0, 0, -1, -1]      # link sphere (3,0,0) touches the face x = 3; held: exactly r -> 0, one step beyond -> none;
    #                                                  the sphere at the held object's own centre never reports slot 1
    for held in (np.array([-1], np.int32), None):
        s, o = call(held)
        assert list(s[0][[0, 1, 3, 4, 5]]) == [0] * 5 and list(o[0][[0, 1, 3, 4, 5]]) == [-1] * 5
        assert s[0][2] == 1 and o[0][2] == 0         # the robot's own sphere is unaffected
    # held slot that is also inside the object window but empty in inst_mesh: the transform still carries the sphere
    im2 = np.array([[0, -1, -1]], np.int32)
    s, o = oracle_mod.collide([cube], g, [0.25], sph, np.zeros(1, np.int32), im2, xf, 2, 0, 2, np.array([1], np.int32))
    assert list(s[0]) == [0, 1, 1, 0, 0, 1] and list(o[0]) == [-1, -1, 0, 0, -1, -1]
    with pytest.raises(ValueError):                  # link below -1
        oracle_mod.collide([cube], g, [0.25], [gen.Sphere(-2, 0, (0, 0, 0))], np.zeros(1, np.int32), im, xf, 2, 0, 2, None)
    with pytest.raises(ValueError):                  # held slot beyond K
        oracle_mod.collide([cube], g, [0.25], sph, np.zeros(1, np.int32), im, xf, 2, 0, 2, np.array([3], np.int32))
