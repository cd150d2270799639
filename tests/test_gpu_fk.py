"""GPU parity of the scene-graph update N12 (gx_set_robot / gx_update_transforms) against oracle.fk: bit-exact on
every matrix entry, through the C ABI; then the transforms it writes are rendered and compared with the oracle's
render of the oracle's transforms (Table 5)."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2306_07552_b200 import gen
from gx_harness import compare, render_gpu

pytestmark = pytest.mark.gpu


def _gpu_fk(robot, base, joints, K, slot0, xf0, held=None, hx=None):
    import torch
    from paper_2306_07552_b200 import binding as gx
    dev = torch.device("cuda:0")
    m = gen.Mesh(np.zeros((3, 3), np.float32), np.zeros((3, 3), np.uint8), np.array([[0, 1, 2]], np.uint32))
    sc = gx.gx_create_scene([m], [m], 0)
    try:
        gx.gx_set_robot(sc, robot)
        N = base.shape[0]
        d_xf = torch.from_numpy(np.ascontiguousarray(xf0, np.float32)).to(dev)
        d_cam = torch.full((N, 16), 7.0, dtype=torch.float32, device=dev)
        args = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) if a is not None else None for a in (base, joints, held, hx)]
        gx.gx_update_transforms(sc, N, K, slot0, args[0], args[1], args[2], args[3], d_cam, d_xf,
                                torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_cam.cpu().numpy(), d_xf.cpu().numpy()
    finally:
        gx.gx_destroy(sc)


def test_fk_bit_exact_proxy_robot(oracle_mod):
    r = gen.robot_proxy()
    for n in (1, 3, 1024, 4099):              # a ragged last block of 4 warps
        base, th, held, hx = gen.robot_states(r, n, seed=n)
        K, slot0 = 25, 20
        xf0 = np.random.default_rng(n).uniform(-1, 1, (n, K, 16)).astype(np.float32)
        cam_o, xf_o = oracle_mod.fk(r, base, th, K, slot0, inst_xform=xf0, held_slot=held, held_xform=hx)
        cam_g, xf_g = _gpu_fk(r, base, th, K, slot0, xf0, held, hx)
        assert np.array_equal(cam_o.view(np.uint32), cam_g.view(np.uint32))
        assert np.array_equal(xf_o.view(np.uint32), xf_g.reshape(n, K, 16).view(np.uint32))
        assert np.array_equal(xf_g.reshape(n, K, 16)[:, 1:slot0], xf0[:, 1:slot0])        # untouched slots keep their bits
        # without held objects nothing but the link slots changes
        cam_g2, xf_g2 = _gpu_fk(r, base, th, K, slot0, xf0)
        cam_o2, xf_o2 = oracle_mod.fk(r, base, th, K, slot0, inst_xform=xf0)
        assert np.array_equal(xf_o2.view(np.uint32), xf_g2.reshape(n, K, 16).view(np.uint32)) and np.array_equal(cam_o2, cam_g2)


def test_fk_bit_exact_random_trees_and_large_angles(oracle_mod):
    rng = np.random.default_rng(5)
    for trial in range(8):
        L = int(rng.integers(1, 65)) if trial else 64
        parent = np.array([-1] + [int(rng.integers(-1, l)) for l in range(1, L)], np.int32)
        jt = rng.integers(0, 3, L).astype(np.int32)
        axis = rng.normal(size=(L, 3))
        axis = (axis / np.linalg.norm(axis, axis=1, keepdims=True)).astype(np.float32)
        origin = np.tile(np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], np.float32), (L, 1))
        origin[:, [3, 7, 11]] = rng.uniform(-0.3, 0.3, (L, 3))
        origin[:, [0, 1, 4, 5]] = np.stack([np.cos(0.3), -np.sin(0.3), np.sin(0.3), np.cos(0.3)]).astype(np.float32)
        r = gen.Robot(parent, jt, axis, origin, int(rng.integers(-1, L)), np.array([1, 0, 0, 0.1, 0, 1, 0, 0.2, 0, 0, 1, 0.3], np.float32),
                      int(rng.integers(-1, L)))
        N, K, slot0 = 37, L + 2, 1
        base = np.stack([rng.uniform(-9, 9, N), rng.uniform(-9, 9, N), rng.uniform(-40, 40, N)], axis=1).astype(np.float32)
        th = rng.uniform(-30, 30, (N, L)).astype(np.float32)
        held = rng.integers(-1, K, N).astype(np.int32)
        hx = np.tile(np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, -0.1], np.float32), (N, 1))
        xf0 = np.zeros((N, K, 16), np.float32)
        cam_o, xf_o = oracle_mod.fk(r, base, th, K, slot0, inst_xform=xf0, held_slot=held, held_xform=hx)
        cam_g, xf_g = _gpu_fk(r, base, th, K, slot0, xf0, held, hx)
        assert np.array_equal(cam_o.view(np.uint32), cam_g.view(np.uint32)), trial
        assert np.array_equal(xf_o.view(np.uint32), xf_g.reshape(N, K, 16).view(np.uint32)), trial


def test_fk_then_render_matches_oracle(oracle_mod):
    """The whole step as the simulator would drive it: robot state -> gx_update_transforms -> gx_render_batch on the same
    stream, against the oracle's FK followed by the oracle's render (camera on the robot's torso, links in slots
    20..24 of a config-1 room, a held icosphere in slot 0 of half the environments)."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(1, n_envs=12)
    r = gen.robot_proxy()
    base, th, held, hx = gen.robot_states(r, wl.N, seed=3)
    base[:, :2] = wl.cam_pose.reshape(wl.N, 4, 4)[:, [0, 2], 3]       # stand where the config's camera stood (free space)
    cam_o, xf_o = oracle_mod.fk(r, base, th, wl.K, 20, inst_xform=wl.inst_xform, held_slot=held, held_xform=hx)
    wl_o = gen.Workload(wl.name, wl.width, wl.height, wl.fx, wl.fy, wl.znear, wl.zfar, wl.static_meshes, wl.dyn_meshes,
                        wl.env_scene, cam_o, wl.inst_mesh, xf_o, wl.depth_only, wl.env_ids, dict(wl.meta))
    o = oracle_mod.render(wl_o)
    dev = torch.device("cuda:0")
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        gx.gx_set_robot(sc, r)
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        d_xf, d_cam = t(wl.inst_xform.astype(np.float32)), torch.zeros((wl.N, 16), dtype=torch.float32, device=dev)
        s = torch.cuda.current_stream().cuda_stream
        gx.gx_update_transforms(sc, wl.N, wl.K, 20, t(base), t(th), t(held), t(hx), d_cam, d_xf, s)
        rgb = torch.zeros((wl.N, wl.height, wl.width, 3), dtype=torch.uint8, device=dev)
        depth = torch.zeros((wl.N, wl.height, wl.width), dtype=torch.float32, device=dev)
        ids = torch.zeros((wl.N, wl.height, wl.width), dtype=torch.int32, device=dev)
        gx.gx_render_batch(sc, gx.camera_of(wl), wl.N, wl.K, t(wl.env_scene.astype(np.int32)), d_cam, t(wl.inst_mesh.astype(np.int32)),
                           d_xf, rgb, depth, ids, s)
        torch.cuda.synchronize()
        g = dict(rgb=rgb.cpu().numpy(), depth=depth.cpu().numpy(), id=ids.cpu().numpy().view(np.uint32))
    finally:
        gx.gx_destroy(sc)
    rep = compare(o, g)
    assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
    assert (o["id"] != 0xFFFFFFFF).mean() > 0.9


def test_fk_argument_errors():
    from paper_2306_07552_b200 import binding as gx
    import torch
    m = gen.Mesh(np.zeros((3, 3), np.float32), np.zeros((3, 3), np.uint8), np.array([[0, 1, 2]], np.uint32))
    sc = gx.gx_create_scene([m], [m], 0)
    try:
        z = torch.zeros(64, device="cuda:0")
        with pytest.raises(gx.GxError):        # no robot yet
            gx.gx_update_transforms(sc, 1, 5, 0, z, z, None, None, z, z)
        bad = gen.robot_proxy()
        bad.parent = np.array([-1, 1, 1, 2, 3], np.int32)   # link 1 is its own parent
        with pytest.raises(gx.GxError):
            gx.gx_set_robot(sc, bad)
        gx.gx_set_robot(sc, gen.robot_proxy())
        with pytest.raises(gx.GxError):        # 5 links do not fit slots [3, 8) of K = 5
            gx.gx_update_transforms(sc, 1, 5, 3, z, z, None, None, z, z)
        with pytest.raises(gx.GxError):        # held_slot without held_xform
            gx.gx_update_transforms(sc, 1, 5, 0, z, z, z.int(), None, z, z)
    finally:
        gx.gx_destroy(sc)
