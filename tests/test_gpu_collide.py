"""GPU parity of the batch collision queries N13 (gx_set_collision_world / gx_collide_batch) against oracle.collide:
every byte and every slot equal, through the C ABI, with the sphere centres coming from gx_update_transforms
(App. G)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2306_07552_b200 import gen

pytestmark = pytest.mark.gpu


def _gpu(w, grids, xf_after_fk=None, n_obj=None, obj_slot0=0, held=True):
    import torch
    from paper_2306_07552_b200 import binding as gx
    dev = torch.device("cuda:0")
    room = gen.Mesh(np.zeros((3, 3), np.float32), np.zeros((3, 3), np.uint8), np.array([[0, 1, 2]], np.uint32))
    sc = gx.gx_create_scene([room] * len(grids), w["dyn_meshes"], 0)
    try:
        gx.gx_set_robot(sc, w["robot"])
        gx.gx_set_collision_world(sc, grids, w["radii"], w["spheres"])
        N, K, S = w["inst_mesh"].shape[0], w["K"], len(w["spheres"])
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        d_xf = t(w["inst_xform"].astype(np.float32))
        d_cam = torch.zeros((N, 16), dtype=torch.float32, device=dev)
        s = torch.cuda.current_stream().cuda_stream
        d_held = t(w["held_slot"]) if held else None
        if xf_after_fk is None:
            gx.gx_update_transforms(sc, N, K, w["link_slot0"], t(w["base_pose"]), t(w["joint_pos"]), d_held,
                                    t(w["held_xform"]) if held else None, d_cam, d_xf, s)
        else:
            d_xf = t(xf_after_fk)
        out_s = torch.full((N, S), 9, dtype=torch.uint8, device=dev)
        out_o = torch.full((N, S), -7, dtype=torch.int32, device=dev)
        gx.gx_collide_batch(sc, N, K, t(w["env_scene"]), t(w["inst_mesh"]), d_xf, w["link_slot0"], obj_slot0,
                            w["n_obj"] if n_obj is None else n_obj, d_held, out_s, out_o, s)
        torch.cuda.synchronize()
        return out_s.cpu().numpy(), out_o.cpu().numpy(), d_xf.cpu().numpy()
    finally:
        gx.gx_destroy(sc)


def test_collide_matches_oracle_after_fk(oracle_mod):
    ext = (3.0, 3.0, 6.0, 6.0)
    grids = [[gen.column_grid(1, 0, r, ext) for r in gen.SPHERE_RADII]]
    for n, held in ((1, True), (37, True), (1030, False)):      # ragged last block of 4 warps
        w = gen.collision_world(n, seed=n, extent=ext)
        n_robot = len(w["spheres"])
        w["spheres"] = w["spheres"] + gen.held_object_spheres()       # link -1: they ride on the grasped object
        hs, hx = (w["held_slot"], w["held_xform"]) if held else (None, None)
        _, xf = oracle_mod.fk(w["robot"], w["base_pose"], w["joint_pos"], w["K"], w["link_slot0"], inst_xform=w["inst_xform"],
                              held_slot=hs, held_xform=hx)
        so, oo = oracle_mod.collide(w["dyn_meshes"], grids, w["radii"], w["spheres"], w["env_scene"], w["inst_mesh"], xf,
                                    w["link_slot0"], 0, w["n_obj"], hs)
        sg, og, xg = _gpu(w, grids, held=held)
        assert np.array_equal(xf.view(np.uint32), xg.reshape(xf.shape).view(np.uint32))
        assert np.array_equal(so, sg) and np.array_equal(oo, og)
        if n > 30:
            assert 0.05 < so.mean() < 0.95 and (oo >= 0).any() and (oo < 0).any()
        holding = (w["held_slot"] >= 0) if held else np.zeros(n, bool)
        assert not so[~holding, n_robot:].any() and (oo[~holding, n_robot:] == -1).all()     # nothing held: no such sphere
        if n == 37:
            assert holding.any() and so[holding, n_robot:].any() and not so[holding, n_robot:].all()
            assert not (oo[holding, n_robot:] == 0).any()             # never its own box (slot 0 is the held object)


def test_collide_two_scenes_object_windows_and_many_objects(oracle_mod):
    """Two static scenes with different grids, object slots that do not start at 0, more objects than one staging round
    (70 > 64), more spheres than one warp round (40 > 32)."""
    ext = (3.0, 3.0, 5.0, 5.0)
    grids = [[gen.column_grid(1, 0, r, ext) for r in gen.SPHERE_RADII], [gen.column_grid(1, 0, r, (4.0, 4.0, 6.0, 6.0)) for r in gen.SPHERE_RADII]]
    w = gen.collision_world(50, seed=9, extent=(3.5, 3.5, 5.5, 5.5))
    rng = np.random.default_rng(2)
    w["env_scene"] = rng.integers(0, 2, 50).astype(np.int32)
    w["spheres"] = w["spheres"] + [gen.Sphere(int(rng.integers(-1, 5)), int(rng.integers(0, 3)), tuple(rng.uniform(-0.3, 0.3, 3))) for _ in range(13)]
    # 70 object slots: the 30 of the generator, then 40 more copies jittered
    N, L = 50, 5
    K = 70 + L
    im = np.full((N, K), -1, np.int32)
    xf = np.tile(np.eye(4, dtype=np.float32).reshape(16), (N, K, 1))
    im[:, :30], xf[:, :30] = w["inst_mesh"][:, :30], w["inst_xform"][:, :30]
    im[:, 30:70] = rng.integers(-1, 3, (N, 40))
    xf[:, 30:70] = w["inst_xform"][:, rng.integers(0, 30, 40)]
    xf[:, 30:70, [3, 7, 11]] += rng.uniform(-0.4, 0.4, (N, 40, 3)).astype(np.float32)
    w.update(inst_mesh=im, inst_xform=xf, K=K, link_slot0=70, n_obj=70)
    _, xfo = oracle_mod.fk(w["robot"], w["base_pose"], w["joint_pos"], K, 70, inst_xform=xf, held_slot=w["held_slot"], held_xform=w["held_xform"])
    for obj0, nobj in ((0, 70), (5, 60), (33, 37), (0, 0)):
        so, oo = oracle_mod.collide(w["dyn_meshes"], grids, w["radii"], w["spheres"], w["env_scene"], im, xfo, 70, obj0, nobj, w["held_slot"])
        sg, og, _ = _gpu(w, grids, n_obj=nobj, obj_slot0=obj0)
        assert np.array_equal(so, sg) and np.array_equal(oo, og), (obj0, nobj)
    assert (oo == -1).all()


def test_collide_argument_errors():
    import torch
    from paper_2306_07552_b200 import binding as gx
    m = gen.Mesh(np.zeros((3, 3), np.float32), np.zeros((3, 3), np.uint8), np.array([[0, 1, 2]], np.uint32))
    sc = gx.gx_create_scene([m], [m], 0)
    try:
        z = torch.zeros(256, device="cuda:0")
        zi, zb = z.int(), z.to(torch.uint8)
        with pytest.raises(gx.GxError):        # no collision world yet
            gx.gx_collide_batch(sc, 1, 6, zi, zi, z, 1, 0, 1, None, zb, zi)
        g = gen.ColumnGrid(0.0, 0.0, 0.03, 2, 2, np.array([0, 1, 1, 2, 2], np.uint32), np.array([[0, 1], [0, 1]], np.float32))
        with pytest.raises(gx.GxError):        # radius class out of range
            gx.gx_set_collision_world(sc, [[g]], [0.05], [gen.Sphere(0, 1, (0, 0, 0))])
        bad = gen.ColumnGrid(0.0, 0.0, 0.03, 2, 2, np.array([0, 2, 1, 2, 2], np.uint32), np.array([[0, 1], [0, 1]], np.float32))
        with pytest.raises(gx.GxError):        # col_off not ascending
            gx.gx_set_collision_world(sc, [[bad]], [0.05], [gen.Sphere(0, 0, (0, 0, 0))])
        gx.gx_set_collision_world(sc, [[g]], [0.05], [gen.Sphere(4, 0, (0, 0, 0))])
        with pytest.raises(gx.GxError):        # link 4 at slot 2 + 4 does not fit K = 6
            gx.gx_collide_batch(sc, 1, 6, zi, zi, z, 2, 0, 1, None, zb, zi)
        with pytest.raises(gx.GxError):        # object window outside K
            gx.gx_collide_batch(sc, 1, 6, zi, zi, z, 1, 3, 4, None, zb, zi)
    finally:
        gx.gx_destroy(sc)
