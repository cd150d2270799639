"""Shared helpers of the GPU parity tests: run a gen.Workload through the C ABI (via the ctypes binding)
and compare with the oracle's images.  Test infrastructure only."""
from __future__ import annotations

import numpy as np

BG = 0xFFFFFFFF


def render_gpu(wl, want_id=True, want_rgb=None, cull=1, stats=False, scene=None, host_api=False, options=None):
    """Render a workload on cuda:0 through gx_render_batch.  Returns dict(rgb, depth, id[, stats])."""
    import torch
    from paper_2306_07552_b200 import binding as gx

    if want_rgb is None:
        want_rgb = not wl.depth_only
    own = scene is None
    if own:
        scene = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        gx.gx_set_option(scene, "cull", cull)
        gx.gx_set_option(scene, "stats", 1 if stats else 0)
        for name, value in (options or {}).items():
            gx.gx_set_option(scene, name, value)
        cam = gx.camera_of(wl)
        N, K, H, W = wl.N, wl.K, wl.height, wl.width
        out = {}
        if host_api:
            rgb = np.empty((N, H, W, 3), np.uint8) if want_rgb else None
            depth = np.empty((N, H, W), np.float32)
            ids = np.empty((N, H, W), np.uint32) if want_id else None
            gx.gx_render_batch_host(scene, cam, N, K, np.ascontiguousarray(wl.env_scene, np.int32),
                                    np.ascontiguousarray(wl.cam_pose, np.float32),
                                    np.ascontiguousarray(wl.inst_mesh, np.int32) if K else None,
                                    np.ascontiguousarray(wl.inst_xform, np.float32) if K else None, rgb, depth, ids)
            out = dict(rgb=rgb, depth=depth, id=ids)
        else:
            dev = torch.device("cuda:0")
            env_scene = torch.from_numpy(np.ascontiguousarray(wl.env_scene, np.int32)).to(dev)
            cam_pose = torch.from_numpy(np.ascontiguousarray(wl.cam_pose, np.float32)).to(dev)
            inst_mesh = torch.from_numpy(np.ascontiguousarray(wl.inst_mesh, np.int32)).to(dev) if K else None
            inst_xform = torch.from_numpy(np.ascontiguousarray(wl.inst_xform, np.float32)).to(dev) if K else None
            rgb = torch.full((N, H, W, 3), 77, dtype=torch.uint8, device=dev) if want_rgb else None
            depth = torch.full((N, H, W), -1.0, dtype=torch.float32, device=dev)
            ids = torch.full((N, H, W), 12345, dtype=torch.int32, device=dev) if want_id else None
            stream = torch.cuda.current_stream().cuda_stream
            gx.gx_render_batch(scene, cam, N, K, env_scene, cam_pose, inst_mesh, inst_xform, rgb, depth, ids, stream)
            torch.cuda.synchronize()
            out = dict(rgb=rgb.cpu().numpy() if want_rgb else None, depth=depth.cpu().numpy(),
                       id=ids.cpu().numpy().view(np.uint32) if want_id else None)
        if stats:
            out["stats"] = {k: gx.gx_get_stat(scene, k) for k in
                            ("clusters_tested", "clusters_drawn", "triangles_in", "triangles_raster", "fragments",
                             "records_occluded", "blocks_drawn", "tile_refs", "triangles_hidden", "subclusters_hidden",
                             "large_records", "large_draws", "bound_violations", "waves", "sum_slots", "max_env_slots",
                             "bad_ids", "launches")}
            assert out["stats"]["bound_violations"] == 0, out["stats"]     # the kernels' own bounds checks (stats build)
        return out
    finally:
        if own:
            gx.gx_destroy(scene)


def compare(o, g, check_rgb=True):
    """north_star tolerances, complete: coverage bit-exact; depth within 1e-5 relative at EVERY pixel; the id
    equal, except that where the GPU picked another triangle its depth must still be within 1e-5 relative of the
    oracle's winner (two surfaces inside the depth tolerance) and such pixels must stay <= 1e-4 of all pixels; RGB
    within +-1 LSB everywhere except exactly those id-mismatch pixels (their colour belongs to the other
    triangle).  Nothing else is exempt.  Returns a dict of counts for reporting."""
    oid, gid = o["id"], g["id"]
    cov_o, cov_g = oid != BG, gid != BG
    assert np.array_equal(cov_o, cov_g), f"coverage differs at {int((cov_o != cov_g).sum())} pixels"
    od, gd = o["depth"], g["depth"]
    od64, gd64 = od.astype(np.float64), gd.astype(np.float64)
    assert np.all(np.isfinite(gd64)), "non-finite depth"
    assert np.all(gd[~cov_o] == 0.0) and np.all(od[~cov_o] == 0.0), "background depth must be exactly 0"
    rel = np.zeros_like(od64)
    rel[cov_o] = np.abs(od64[cov_o] - gd64[cov_o]) / np.abs(od64[cov_o])
    assert rel.max(initial=0.0) <= 1e-5, f"max relative depth error {rel.max():.3e}"
    id_diff = oid != gid
    n_id = int(id_diff.sum())
    # an id mismatch is only legitimate between two surfaces within the depth tolerance of each other
    assert np.all(rel[id_diff] <= 1e-5), "id mismatch at a pixel whose depths differ by more than the tolerance"
    assert n_id <= 1e-4 * oid.size, f"{n_id} id mismatches of {oid.size} pixels"
    n_rgb = 0
    max_rgb = 0
    if check_rgb and g.get("rgb") is not None:
        d = np.abs(o["rgb"].astype(np.int32) - g["rgb"].astype(np.int32)).max(axis=-1)
        bad = (d > 1) & ~id_diff
        n_rgb = int((d > 0).sum())
        max_rgb = int(d[~id_diff].max()) if (~id_diff).any() else 0
        assert not bad.any(), f"{int(bad.sum())} pixels with RGB error > 1 LSB (max {int(d.max())})"
        assert np.all(g["rgb"][~cov_o] == 0), "background RGB must be 0"
    return dict(id_mismatch=n_id, depth_bits_differ=int((od.view(np.uint32) != gd.view(np.uint32)).sum()),
                max_rel_depth=float(rel.max(initial=0.0)), rgb_differ=n_rgb, max_rgb=max_rgb)
