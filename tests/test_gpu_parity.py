"""GPU parity: the CUDA path (through the C ABI, include/gx.h) against the CPU oracle, element by element,
on the same seeded workloads (`-m gpu`, needs a B200).

Tolerances are north_star's (BASELINE.json): coverage and winning triangle id bit-exact, depth within 1e-5
relative, RGB within +-1 LSB; ids may differ only where two surfaces are within the depth tolerance, on
<= 1e-4 of pixels.  The kernels implement DESIGN.md N1-N9 operation by operation, so the tests additionally
require what is expected in practice: depth bit-identical and zero id mismatches.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2306_07552_b200 import gen
from gx_harness import BG, compare, render_gpu

pytestmark = pytest.mark.gpu


def _check(oracle_mod, wl, **kw):
    o = oracle_mod.render(wl)
    g = render_gpu(wl, **kw)
    rep = compare(o, g, check_rgb=not wl.depth_only)
    assert rep["id_mismatch"] == 0, rep
    assert rep["depth_bits_differ"] == 0, rep
    assert rep["rgb_differ"] == 0, rep       # N8 is implemented verbatim: not just within +-1 LSB, the same bytes
    return o, g, rep


def test_config0_full(oracle_mod):
    """BASELINE.json configs[0]: 4 envs, 64x64, 200-triangle soup + 2 cubes per env."""
    wl = gen.make_config(0)
    o, g, rep = _check(oracle_mod, wl)
    assert (o["id"] != BG).mean() > 0.2      # the scene is actually visible


@pytest.mark.parametrize("cfg,n", [(1, 24), (2, 24)])
def test_room_configs_subset(oracle_mod, cfg, n):
    """configs[1], configs[2]: first n environments (several frames, thousands of clusters, near-plane
    crossings through the robot arm and the floor)."""
    wl = gen.make_config(cfg, n_envs=n)
    o, g, rep = _check(oracle_mod, wl)
    assert (o["id"] != BG).mean() > 0.9


def _all_off(wl):
    """The same call with every culling device off (N10): no frustum culling of clusters or runs, no hi-Z, no
    occluder scheme."""
    return render_gpu(wl, cull=0, options=dict(subcull=0, hiz=0, occlusion=0))


def _same_images(a, b, wl, what):
    for k in ("depth", "id") + (() if wl.depth_only else ("rgb",)):
        x, y = a[k], b[k]
        if k == "depth":
            x, y = x.view(np.uint32), y.view(np.uint32)
        assert np.array_equal(x, y), f"{what}: {k} differs in {int((x != y).reshape(wl.N, -1).any(axis=1).sum())} environments"


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_configs_0_to_2_every_environment(oracle_mod, cfg):
    """'Parity is checked on all envs of configs 0-2'.  configs[0], [1], [2] at full size in the launch
    configuration bench.py times (one call of N = 4 / 256 / 1024 environments): the oracle renders every environment
    and every pixel of every environment must match (coverage, id, depth bits, RGB bytes).  Then N10 at full size:
    the same call with all culling off gives the same images, and so does the timed configuration (id_out NULL)."""
    wl = gen.make_config(cfg)
    assert wl.N == gen.CONFIG_SHAPES[cfg][1]
    o, g, rep = _check(oracle_mod, wl)
    _same_images(g, _all_off(wl), wl, "culling off")
    g2 = render_gpu(wl, want_id=False)     # timed configuration: no id output
    assert np.array_equal(g["depth"].view(np.uint32), g2["depth"].view(np.uint32))
    assert np.array_equal(g["rgb"], g2["rgb"])


def test_config3_and_4_sampled(oracle_mod):
    """configs[3] (500k-triangle scenes, K=45) and configs[4] (64x64 depth-only): a seeded subset of
    environments, rendered by both sides."""
    for cfg, n in ((3, 6), (4, 16)):
        rng = np.random.Generator(np.random.Philox(key=[77, cfg]))
        N = gen.CONFIG_SHAPES[cfg][1]
        sel = np.sort(rng.choice(N, n, replace=False))
        wl = gen.make_config(cfg, env_ids=sel)
        _check(oracle_mod, wl)


@pytest.mark.parametrize("cfg", [3, 4])
def test_config3_and_4_full_batch(oracle_mod, cfg):
    """configs[3] (4096 envs, 500k-triangle scenes) and configs[4] (16384 envs, 64x64 depth-only) at full size,
    in the launch configuration bench.py --config times.  The oracle renders the population SURVEY.md 8(d)
    prescribes -- the 256 environments its timed sample uses (the first 256) plus 64 seeded random others -- one by
    one; the GPU renders the whole batch and those 320 rows must match.  The first call sizes the record arena from
    defaults, the second from the first call's slot bounds; on cfg 3 the arena budget cannot hold the whole batch,
    so the later waves run inside the cooperative tail kernel: all must match.  Then N10 over EVERY environment of
    the batch: the call with all culling off (frustum, runs, hi-Z, occluder scheme) gives the same images."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(cfg)
    rng = np.random.Generator(np.random.Philox(key=[78, cfg]))
    sel = np.sort(np.concatenate([np.arange(256), 256 + rng.choice(wl.N - 256, 64, replace=False)]))
    o = oracle_mod.render(wl.subset(sel))
    scene = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        g1 = render_gpu(wl, scene=scene, stats=True)
        torch.cuda.synchronize()
        g2 = render_gpu(wl, scene=scene, stats=True)
    finally:
        gx.gx_destroy(scene)
    assert g1["stats"]["bad_ids"] == 0 and g1["stats"]["waves"] >= 1 and g2["stats"]["waves"] >= 1
    if cfg == 3:
        assert g1["stats"]["waves"] > 1      # 4096 environments of ~10^5 slots each do not fit 4 GB at once
    for g in (g1, g2):
        gs = {k: (v[sel] if isinstance(v, np.ndarray) else None) for k, v in g.items()}
        rep = compare(o, gs, check_rgb=not wl.depth_only)
        assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
    for k in ("depth", "id") + (() if wl.depth_only else ("rgb",)):
        assert np.array_equal(g1[k], g2[k]), k
    del g2
    _same_images(g1, _all_off(wl), wl, "culling off")


def test_cull_is_conservative(oracle_mod):
    """N10: the image with frustum culling of clusters and sub-clusters and with hi-Z rejection in the tiles equals
    the image with all of them off, bit for bit."""
    wl = gen.make_config(1, n_envs=16)
    a = render_gpu(wl, cull=1, stats=True, options=dict(occlusion=0))
    a2 = render_gpu(wl, cull=1, stats=True)     # occluder scheme (default at this frame size)
    b = render_gpu(wl, cull=0, stats=True, options=dict(hiz=0))
    c = render_gpu(wl, cull=1, stats=True, options=dict(subcull=0))
    d = render_gpu(wl, cull=1, stats=True, options=dict(hiz=0))
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a2[k], b[k]), k
        assert np.array_equal(c[k], b[k]), k
        assert np.array_equal(d[k], b[k]), k
    assert a["stats"]["clusters_drawn"] < b["stats"]["clusters_drawn"]
    assert b["stats"]["clusters_drawn"] == b["stats"]["clusters_tested"]
    assert a["stats"]["triangles_raster"] == b["stats"]["triangles_raster"]     # frustum culling only drops what covers nothing
    assert a2["stats"]["triangles_raster"] < a["stats"]["triangles_raster"]     # the occluder scheme drops hidden triangles too
    assert a2["stats"]["triangles_in"] < a["stats"]["triangles_in"]
    assert a["stats"]["triangles_in"] < c["stats"]["triangles_in"] < b["stats"]["triangles_in"]
    assert a["stats"]["records_occluded"] > 0 and d["stats"]["records_occluded"] == 0
    assert a["stats"]["fragments"] < d["stats"]["fragments"]


def test_waves_and_option_variants(oracle_mod):
    """The pipeline against the oracle, then against itself under every switch that moves work around: an arena
    too small for the batch (several waves of environments, the later ones inside the cooperative tail kernel, down
    to one environment per wave), the block path for every record size (big_px), no hi-Z, no sub-cluster culling:
    all bit-identical."""
    wl = gen.make_config(2, n_envs=20)
    o = oracle_mod.render(wl)
    ref = render_gpu(wl, stats=True)
    rep = compare(o, ref)
    assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
    # cull, item packing, 2 x (geometry, bin, raster), the run culling of the second phase, tail: the occluder scheme is on by default for 128x128 frames
    assert ref["stats"]["waves"] == 1 and ref["stats"]["launches"] == 10 and ref["stats"]["bad_ids"] == 0
    assert ref["stats"]["subclusters_hidden"] > 0 and ref["stats"]["triangles_hidden"] > 0
    assert ref["stats"]["max_env_slots"] * wl.N >= ref["stats"]["sum_slots"] > ref["stats"]["triangles_raster"]
    per_env = ref["stats"]["max_env_slots"]
    variants = {
        "arena for ~3 environments": dict(arena_slots=3 * per_env),
        "arena for 1 environment": dict(arena_slots=1),
        "arena by budget": dict(pool_bytes=88 * 7 * per_env),
        "block path for every record": dict(big_px=1),
        "block path from 4 px": dict(big_px=4),
        "block path from 8 px": dict(big_px=8),
        "no hi-Z": dict(hiz=0),
        "no sub-cluster culling": dict(subcull=0),
        "no hi-Z, blocks from 2 px, 2 environments per wave": dict(hiz=0, big_px=2, arena_slots=2 * per_env),
        "single pass (no occluder phase)": dict(occlusion=0),
        "single pass, 1 environment per wave": dict(occlusion=0, arena_slots=1),
        "every sub-cluster an occluder": dict(occl_area=0),
        "no sub-cluster an occluder (but those at the near plane)": dict(occl_area=1 << 20),
        "occluders from 8 px per triangle, 3 environments per wave": dict(occl_area=8, arena_slots=3 * per_env),
        "two CTAs per SM, bin CTAs of 256 threads": dict(ctas_per_sm=2, bin_threads=256),
        "large path from 16 px": dict(big_px=16),
        "large path from 32 px": dict(big_px=32),
    }
    for name, opts in variants.items():
        g = render_gpu(wl, stats=True, options=opts)
        for k in ("rgb", "depth", "id"):
            assert np.array_equal(ref[k], g[k]), (name, k)
        if name == "arena for 1 environment":      # (the arena never shrinks below the largest possible environment)
            assert g["stats"]["waves"] >= 3, g["stats"]
        if name == "arena by budget":
            assert 1 < g["stats"]["waves"] < wl.N, g["stats"]
        if name.startswith("single pass"):
            assert g["stats"]["subclusters_hidden"] == 0 and g["stats"]["triangles_hidden"] == 0
        if name == "single pass (no occluder phase)":
            assert g["stats"]["launches"] == 6
        if name == "block path for every record":
            # (only records of a single pixel stay on the small path)
            assert g["stats"]["tile_refs"] < ref["stats"]["tile_refs"] and g["stats"]["blocks_drawn"] > ref["stats"]["blocks_drawn"]
    assert ref["stats"]["records_occluded"] > 0 and ref["stats"]["tile_refs"] > 0


def test_sharding_and_determinism():
    """concatenating per-shard outputs equals the single call, bit-identical; and the same
    call ten times gives the same bits (the order in which warps append records and fill tile lists differs from
    run to run; the image must not)."""
    wl = gen.make_config(1, n_envs=20)
    full = render_gpu(wl)
    again = render_gpu(wl)
    big = gen.make_config(2, n_envs=64)
    first = render_gpu(big)
    for _ in range(9):
        nxt = render_gpu(big)
        for k in ("rgb", "depth", "id"):
            assert np.array_equal(first[k], nxt[k]), k
    parts = [render_gpu(wl.subset(np.arange(a, b))) for a, b in ((0, 7), (7, 8), (8, 20))]
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(full[k], again[k]), k
        assert np.array_equal(full[k], np.concatenate([p[k] for p in parts])), k


def test_host_entry_point_matches_device_entry_point():
    wl = gen.make_config(0)
    a = render_gpu(wl)
    b = render_gpu(wl, host_api=True)
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(a[k], b[k]), k


def test_depth_only_and_empty_slots(oracle_mod):
    """rgb_out = NULL (config 4's mode) on config 0; empty instance slots (-1) keep later ids in place."""
    wl = gen.make_config(0)
    wl.inst_mesh = wl.inst_mesh.copy()
    wl.inst_mesh[1, 0] = -1
    wl.inst_mesh[2, :] = -1
    o = oracle_mod.render(wl)
    g = render_gpu(wl, want_rgb=False)
    compare(o, g, check_rgb=False)
    assert np.array_equal(o["id"], g["id"])
    g = render_gpu(wl)
    compare(o, g)


def _quad_workload(W, H, z, half, K=0):
    """One fronto-parallel quad at view depth z facing an identity camera."""
    pos = np.array([[-half, -half, -z], [half, -half, -z], [half, half, -z], [-half, half, -z]], np.float32)
    col = np.array([[255, 0, 0], [0, 255, 0], [0, 0, 255], [255, 255, 255]], np.uint8)
    idx = np.array([[0, 1, 2], [0, 2, 3]], np.uint32)
    m = gen.Mesh(pos, col, idx)
    cam = np.eye(4, dtype=np.float32).reshape(1, 16)
    return gen.Workload("quad", W, H, 1.0, 1.0, 0.1, 20.0, [m], [m], np.zeros(1, np.int32), cam,
                        np.full((1, K), -1, np.int32), np.tile(np.eye(4, dtype=np.float32).reshape(1, 1, 16), (1, K, 1)))


def test_edge_cases(oracle_mod):
    """Degenerate inputs: K = 0; all slots empty; a frame with nothing in view (all background); a quad that
    fills the whole frame and crosses all four image borders; the far plane; the maximum frame size 256x256 and
    the smallest 16x16; non-square frames."""
    # K = 0, small quad: closed form -- pixel rectangle at exactly depth 2
    wl = _quad_workload(64, 64, 2.0, 0.5)
    g = render_gpu(wl)
    o = oracle_mod.render(wl)
    compare(o, g)
    cov = g["id"][0] != BG
    assert cov.sum() == 16 * 16 and cov[24:40, 24:40].all()   # x = +-0.5 at w = 2 -> ndc +-0.25 -> pixels 24..40
    assert np.all(g["depth"][0][cov] == 2.0) and np.all(g["depth"][0][~cov] == 0.0)
    assert np.all(g["rgb"][0][~cov] == 0)
    # all slots empty
    wl = _quad_workload(64, 64, 2.0, 0.5, K=3)
    compare(oracle_mod.render(wl), render_gpu(wl))
    # nothing in view: camera turned away (looks along +Z)
    wl = _quad_workload(32, 48, 2.0, 0.5)
    wl.cam_pose = np.array([[-1, 0, 0, 0, 0, 1, 0, 0, 0, 0, -1, 0, 0, 0, 0, 1]], np.float32)
    g = render_gpu(wl)
    assert np.all(g["id"] == BG) and np.all(g["depth"] == 0) and np.all(g["rgb"] == 0)
    # huge quad over the whole frame, partially behind the camera after a pitch: near clip + all borders
    for (W, H) in ((128, 128), (16, 16), (128, 64), (48, 112), (128, 96), (96, 128), (64, 128), (112, 80), (256, 256), (224, 224),
                   (256, 16), (16, 256)):
        wl = _quad_workload(W, H, 1.0, 50.0)
        c, s = np.cos(1.2), np.sin(1.2)
        wl.cam_pose = np.array([[1, 0, 0, 0, 0, c, -s, 0.3, 0, s, c, 0, 0, 0, 0, 1]], np.float32)
        wl.fy = 1.0
        wl.fx = H / W
        o = oracle_mod.render(wl)
        g = render_gpu(wl)
        rep = compare(o, g)
        assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0
        assert (o["id"] != BG).any()
    # far plane: quad at 25 m with zfar 20 is dropped, at 19 m kept
    wl = _quad_workload(64, 64, 25.0, 5.0)
    assert np.all(render_gpu(wl)["id"] == BG)
    wl = _quad_workload(64, 64, 19.0, 5.0)
    compare(oracle_mod.render(wl), render_gpu(wl))


def test_random_soup_large_triangles(oracle_mod):
    """Triangles far larger than the frame, random winding, many crossing the near plane, exact depth ties
    (duplicated triangles under different ids): exercises the int64 edge path and the (depth, id, sub) order."""
    rng = np.random.Generator(np.random.Philox(key=[77, 100]))
    nt = 600
    pos = (rng.uniform(-1, 1, (nt * 3, 3)) * np.array([6.0, 3.0, 6.0])).astype(np.float32)
    pos[3 * 300:] = pos[:3 * 300]                      # second half duplicates the first: exact ties
    col = rng.integers(0, 256, (nt * 3, 3)).astype(np.uint8)
    col[3 * 300:] = col[:3 * 300]
    m = gen.Mesh(pos, col, np.arange(nt * 3, dtype=np.uint32).reshape(nt, 3))
    n = 6
    cam = np.zeros((n, 4, 4), np.float32)
    for k in range(n):
        a = rng.uniform(0, 2 * np.pi)
        cam[k] = np.array([[np.cos(a), 0, np.sin(a), rng.uniform(-1, 1)], [0, 1, 0, rng.uniform(-1, 1)],
                           [-np.sin(a), 0, np.cos(a), rng.uniform(-1, 1)], [0, 0, 0, 1]])
    wl = gen.Workload("soup", 128, 128, 1.0, 1.0, 0.1, 20.0, [m], [], np.zeros(n, np.int32),
                      cam.reshape(n, 16), np.zeros((n, 0), np.int32), np.zeros((n, 0, 16), np.float32))
    o = oracle_mod.render(wl)
    g = render_gpu(wl)
    rep = compare(o, g)
    assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
    assert (o["id"][o["id"] != BG] < 300).all()        # lower id wins every exact tie


def _one_triangle_scenes(tris, cols, W, H):
    """One static mesh per triangle (camera-space corners (xc, yc, w) -> world (xc, yc, -w) under the identity camera),
    one environment per mesh."""
    meshes = []
    for t, c in zip(tris, cols):
        pos = np.array([[v[0], v[1], -v[2]] for v in t], np.float32)
        meshes.append(gen.Mesh(pos, np.asarray(c, np.uint8).reshape(3, 3), np.array([[0, 1, 2]], np.uint32)))
    n = len(meshes)
    cam = np.tile(np.eye(4, dtype=np.float32).reshape(1, 16), (n, 1))
    return gen.Workload("one triangle per scene", W, H, 1.0, 1.0, 0.1, 20.0, meshes, [], np.arange(n, dtype=np.int32), cam,
                        np.zeros((n, 0), np.int32), np.zeros((n, 0, 16), np.float32))


def test_clamped_vertices_and_colour_ties(oracle_mod):
    """The two clauses of the definition that ordinary scenes never reach, through gx_render_batch:
    N5's clamp of the snapped coordinates to +-2^28 (vertices thousands of metres to the side at w just beyond the
    near plane; int32 corner differences up to 2^29 and int64 edge values up to 2^58 on the wide path), and N8's
    round-half-to-even of a colour that lands exactly on m + 1/2 (tests/test_oracle_pins.py derives both by hand:
    test_snap_clamps_at_two_to_the_28, test_colour_rounds_half_to_even)."""
    # --- clamp: the pin's triangle, its three quarter-turn images, and triangles with two and three clamped corners
    W = H = 128
    hw = 128.0 * W
    cam_xy = lambda X, Y, w: ((X - hw) * w / hw, -(Y - hw) * w / hw, w)
    X0, Y0, Y1 = 256 * 10, 256 * 20 + 127, 256 * 100
    base = [cam_xy(X0, Y0, 2.0), cam_xy(X0, Y1, 2.0), (4096.0, 0.0, 0.125)]
    tris = []
    for turn in range(4):
        t = base
        for _ in range(turn):
            t = [(-v[1], v[0], v[2]) for v in t]
        tris.append(t)
    tris.append([cam_xy(256 * 60 + 3, 256 * 70 + 5, 2.0), (-4096.0, -4096.0, 0.125), (4096.0, -3000.0, 0.125)])
    tris.append([cam_xy(256 * 30 + 77, 256 * 12 + 200, 4.0), (4096.0, 4096.0, 0.125), (5000.0, -4096.0, 0.125)])
    tris.append([(-4096.0, 4096.0, 0.125), (4096.0, 4096.0, 0.125), (100.0, -6000.0, 0.125)])
    tris.append([(-1.0e6, 3.0, 0.125), (2.0e6, 5.0, 0.125), (7.0, -1.0e6, 0.25)])
    rng = np.random.Generator(np.random.Philox(key=[77, 101]))
    cols = rng.integers(0, 256, (len(tris), 3, 3))
    wl = _one_triangle_scenes(tris, cols, W, H)
    o, g, rep = _check(oracle_mod, wl)
    cov = (o["id"] != BG).reshape(wl.N, -1).mean(axis=1)
    assert (cov[:4] > 0.05).all() and (cov > 0).all(), cov          # every one of them is on the screen
    g0 = render_gpu(wl, cull=0, options=dict(hiz=0, occlusion=0))
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(g[k], g0[k]), k
    # --- colour ties: the pin's triangle at 16x16, vertex 2 carries a + b with b odd, row 8 has weight 1/2 exactly
    W = H = 16
    hw = 128.0 * W
    XY = [(256 * 3, 256 * 4 + 128), (256 * 11, 256 * 4 + 128), (256 * 3, 256 * 12 + 128)]
    tris, cols, want = [], [], []
    for a in (0, 10, 101):
        for b0 in range(1, 256 - a - 4, 6):
            bs = (b0, b0 + 2, b0 + 4)
            for flip in (0, 1):
                order = (0, 2, 1) if flip else (0, 1, 2)
                c = np.array([[a] * 3, [a] * 3, [a + b for b in bs]])
                tris.append([cam_xy(XY[k][0], XY[k][1], 2.0) for k in order])
                cols.append(c[list(order)])
                lo = [a + (b - 1) // 2 for b in bs]
                want.append([v if v % 2 == 0 else v + 1 for v in lo])
    wl = _one_triangle_scenes(tris, cols, W, H)
    o, g, rep = _check(oracle_mod, wl)
    want = np.array(want, np.uint8)
    for col_px in (3, 4, 5, 6):
        assert np.array_equal(g["rgb"][:, 8, col_px, :], want), col_px     # the hand values, not only the oracle's
    assert np.all(g["id"][:, 8, 3:7] == 0) and np.all(g["id"][:, 8, 7] == BG)


def test_reference_area_fallback(oracle_mod):
    """Records of 17..31 pixels reference up to 3x3 tiles; when the exact count does not fit the environment's
    reference area (4 words per record slot) the bin stage sends them down the large path instead.  300 stacked
    triangles whose boxes all span pixels 15..45 of a 64x64 frame (9 tiles each, no slot to spare) force that;
    big_px = 16 never needs it.  All three renders equal the oracle."""
    nt, W = 300, 64
    pos = np.zeros((nt * 3, 3), np.float32)
    for i in range(nt):
        d = 2.0 + 0.01 * i
        for k, (px, py) in enumerate(((15.3, 15.3), (45.7, 15.3), (15.3, 45.7))):
            pos[3 * i + k] = ((px / 32.0 - 1.0) * d, -(py / 32.0 - 1.0) * d, -d)
    rng = np.random.Generator(np.random.Philox(key=[78, 100]))
    col = rng.integers(0, 256, (nt * 3, 3)).astype(np.uint8)
    m = gen.Mesh(pos, col, np.arange(nt * 3, dtype=np.uint32).reshape(nt, 3))
    cam = np.eye(4, dtype=np.float32).reshape(1, 16)
    wl = gen.Workload("stack", W, W, 1.0, 1.0, 0.1, 20.0, [m], [], np.zeros(1, np.int32), cam,
                      np.zeros((1, 0), np.int32), np.zeros((1, 0, 16), np.float32))
    o = oracle_mod.render(wl)
    for opts in ({"hiz": 0}, {"hiz": 0, "big_px": 16}, {}):
        g = render_gpu(wl, stats=True, options=opts)
        rep = compare(o, g)
        assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, (opts, rep)
        if opts == {"hiz": 0}:                       # fell back: every record on the large path, no tile references
            assert g["stats"]["tile_refs"] == 0 and g["stats"]["large_records"] == nt, g["stats"]
        if opts.get("big_px") == 16:
            assert g["stats"]["large_records"] == nt


def test_reserve_then_no_growth(oracle_mod):
    """gx_reserve sizes the arena and the tables for a call shape ahead of time: the render calls that follow leave
    "arena_bytes" and "scratch_bytes" unchanged (ADVICE: no hidden allocation in the steady state), and the budget
    option bounds the arena."""
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(1, n_envs=24)
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        gx.gx_set_option(sc, "pool_bytes", 256 << 20)
        gx.gx_reserve(sc, gx.camera_of(wl), wl.N, wl.K)
        a0, s0 = gx.gx_get_stat(sc, "arena_bytes"), gx.gx_get_stat(sc, "scratch_bytes")
        assert 0 < a0 <= (256 << 20) + 88 * (4 * 71600 + 64) and s0 > 0
        o = oracle_mod.render(wl)
        for _ in range(3):
            g = render_gpu(wl, scene=sc)
            assert compare(o, g)["id_mismatch"] == 0
            assert gx.gx_get_stat(sc, "arena_bytes") == a0 and gx.gx_get_stat(sc, "scratch_bytes") == s0
    finally:
        gx.gx_destroy(sc)


def test_cuda_graph_capture_and_replay(oracle_mod):
    """gx_render_batch can be captured into a CUDA graph once the handle holds its buffers (gx_reserve or one plain
    call): inside the capture it allocates nothing and reads nothing back; replays give the oracle's images, also
    with new poses written into the same input tensors and with an arena so small that the captured call needs
    several waves (host rounds and the cooperative tail kernel inside the graph)."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(1, n_envs=16)
    wl2 = gen.make_config(1, env_ids=np.arange(16, 32))
    o1, o2 = oracle_mod.render(wl), oracle_mod.render(wl2)
    dev = torch.device("cuda:0")
    for opts in ({}, {"arena_slots": 1}):
        sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
        try:
            for k, v in opts.items():
                gx.gx_set_option(sc, k, v)
            cam = gx.camera_of(wl)
            N, K, H, W = wl.N, wl.K, wl.height, wl.width
            t = lambda a, ty: torch.from_numpy(np.ascontiguousarray(a, ty)).to(dev)
            d = [t(wl.env_scene, np.int32), t(wl.cam_pose, np.float32), t(wl.inst_mesh, np.int32), t(wl.inst_xform, np.float32)]
            rgb = torch.zeros((N, H, W, 3), dtype=torch.uint8, device=dev)
            depth = torch.zeros((N, H, W), dtype=torch.float32, device=dev)
            ids = torch.zeros((N, H, W), dtype=torch.int32, device=dev)
            g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
            if not opts:     # without buffers the capture is refused, and the refusal leaves the capture usable
                with pytest.raises(gx.GxError):
                    with torch.cuda.graph(torch.cuda.CUDAGraph(), stream=s):
                        gx.gx_render_batch(sc, cam, N, K, d[0], d[1], d[2], d[3], rgb, depth, ids, torch.cuda.current_stream().cuda_stream)
            gx.gx_reserve(sc, cam, N, K)
            with torch.cuda.graph(g, stream=s):
                gx.gx_render_batch(sc, cam, N, K, d[0], d[1], d[2], d[3], rgb, depth, ids, torch.cuda.current_stream().cuda_stream)
            for o, w in ((o1, wl), (o2, wl2), (o1, wl)):
                d[0].copy_(t(w.env_scene, np.int32)); d[1].copy_(t(w.cam_pose, np.float32))
                d[2].copy_(t(w.inst_mesh, np.int32)); d[3].copy_(t(w.inst_xform, np.float32))
                depth.fill_(-1.0)
                g.replay()
                torch.cuda.synchronize()
                got = dict(rgb=rgb.cpu().numpy(), depth=depth.cpu().numpy(), id=ids.cpu().numpy().view(np.uint32))
                rep = compare(o, got)
                assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0 and rep["rgb_differ"] == 0, (opts, rep)
            if opts:
                assert gx.gx_get_stat(sc, "waves") > 1
        finally:
            gx.gx_destroy(sc)


def test_cuda_graph_survives_growth_of_the_handle(oracle_mod):
    """A captured call bakes the handle's arena and table addresses into the graph.  Later plain calls that make the
    handle grow (more environments; a larger arena) must not free what the graph uses: the old buffers are retired
    until gx_destroy, replaying the earlier graph still gives the oracle's images, and so does a second graph captured
    after the growth.  Inside a capture "arena_slots" can never hand out more slots than the handle holds."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(1, n_envs=8)
    big = gen.make_config(1, n_envs=48)
    o, ob = oracle_mod.render(wl), oracle_mod.render(big)
    dev = torch.device("cuda:0")
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        cam = gx.camera_of(wl)
        N, K, H, W = wl.N, wl.K, wl.height, wl.width
        t = lambda a, ty: torch.from_numpy(np.ascontiguousarray(a, ty)).to(dev)
        d = [t(wl.env_scene, np.int32), t(wl.cam_pose, np.float32), t(wl.inst_mesh, np.int32), t(wl.inst_xform, np.float32)]
        rgb = torch.zeros((N, H, W, 3), dtype=torch.uint8, device=dev)
        depth = torch.zeros((N, H, W), dtype=torch.float32, device=dev)
        ids = torch.zeros((N, H, W), dtype=torch.int32, device=dev)
        s = torch.cuda.Stream()

        def capture():
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                gx.gx_render_batch(sc, cam, N, K, d[0], d[1], d[2], d[3], rgb, depth, ids, torch.cuda.current_stream().cuda_stream)
            return g

        def replay_ok(g, what):
            depth.fill_(-1.0); ids.fill_(7); rgb.fill_(9)
            g.replay()
            torch.cuda.synchronize()
            got = dict(rgb=rgb.cpu().numpy(), depth=depth.cpu().numpy(), id=ids.cpu().numpy().view(np.uint32))
            rep = compare(o, got)
            assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0 and rep["rgb_differ"] == 0, (what, rep)

        gx.gx_set_option(sc, "arena_slots", 400000)         # a small arena (worst case of one environment: ~300k slots)
        gx.gx_reserve(sc, cam, N, K)
        a0, s0 = gx.gx_get_stat(sc, "arena_bytes"), gx.gx_get_stat(sc, "scratch_bytes")
        g1 = capture()
        replay_ok(g1, "first graph")
        # inside a capture the option may ask for more than is held: more waves, never slots past the allocation
        gx.gx_set_option(sc, "arena_slots", 4000000)
        g1b = capture()
        assert gx.gx_get_stat(sc, "arena_bytes") == a0
        replay_ok(g1b, "graph captured with arena_slots beyond the held arena")
        # plain calls that grow both the arena and the tables
        gx.gx_set_option(sc, "arena_slots", 0)
        for _ in range(2):
            gb = render_gpu(big, scene=sc)
            rep = compare(ob, gb)
            assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
        assert gx.gx_get_stat(sc, "arena_bytes") > a0 and gx.gx_get_stat(sc, "scratch_bytes") > s0
        junk = [torch.full((1 << 26,), 0x7F, dtype=torch.uint8, device=dev) for _ in range(4)]   # reuse whatever was freed
        replay_ok(g1, "first graph after the handle grew")
        replay_ok(g1b, "second graph after the handle grew")
        g2 = capture()
        replay_ok(g2, "graph captured after the growth")
        replay_ok(g1, "first graph again")
        del junk
    finally:
        gx.gx_destroy(sc)


def test_failed_arena_growth_leaves_the_handle_usable(oracle_mod):
    """The arena is three arrays that grow one after the other.  When the device runs out of memory in the middle (the
    first array fits, the second does not) the call returns GX_ERR_OOM and the handle must not keep the old arena
    size with a missing array: the next, smaller call allocates afresh and renders the oracle's images."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(1, n_envs=6)
    o = oracle_mod.render(wl)
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        g = render_gpu(wl, scene=sc)                         # the handle holds an arena and renders
        assert compare(o, g)["id_mismatch"] == 0
        torch.cuda.empty_cache()
        free, _total = torch.cuda.mem_get_info()
        # 64 + 8 + 16 bytes per slot in three arrays: at free / 70 slots the first (64 B) fits and the second cannot
        slots = int(free // 70)
        if slots >= 0xFFFFFF00:
            pytest.skip("more free device memory than a 2^32-slot arena can use up")
        gx.gx_set_option(sc, "arena_slots", slots)
        with pytest.raises(gx.GxError) as ei:
            render_gpu(wl, scene=sc)
        assert ei.value.code == gx.GX_ERR_OOM, str(ei.value)
        assert gx.gx_get_stat(sc, "arena_bytes") == 0        # nothing usable is claimed
        gx.gx_set_option(sc, "arena_slots", 0)
        for _ in range(2):
            g = render_gpu(wl, scene=sc)
            rep = compare(o, g)
            assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0 and rep["rgb_differ"] == 0, rep
    finally:
        gx.gx_destroy(sc)


def test_argument_errors():
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(0)
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        d = torch.zeros(4 * 64 * 64, device="cuda")
        es = torch.zeros(4, dtype=torch.int32, device="cuda")
        cp = torch.zeros(64, device="cuda")
        for cam, N in ((gx.GxCamera(60, 64, 1, 1, 0.1, 20), 4), (gx.GxCamera(64, 64, 1, 1, 0.0, 20), 4),
                       (gx.GxCamera(64, 64, 1, 1, 1.0, 0.5), 4), (gx.GxCamera(64, 64, 1, 1, 0.1, 20), 0)):
            with pytest.raises(gx.GxError) as e:
                gx.gx_render_batch(sc, cam, N, 0, es, cp, None, None, None, d)
            assert e.value.code == gx.GX_ERR_INVALID_ARG
        with pytest.raises(gx.GxError) as e:
            gx.gx_render_batch(sc, gx.GxCamera(272, 128, 1, 1, 0.1, 20), 4, 0, es, cp, None, None, None, d)
        assert e.value.code == gx.GX_ERR_UNSUPPORTED
        with pytest.raises(gx.GxError):
            gx.gx_set_option(sc, "nope", 1)
    finally:
        gx.gx_destroy(sc)


def test_packed_observation(oracle_mod):
    """N11 / NEXT-1: gx_render_batch_obs writes the [N,4,H,W] binary16 observation bit-identical to the oracle's
    packing of the oracle's images -- with the default switches, with every record on the block path, without hi-Z
    and through the waves of the tail kernel."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    for wl in (gen.make_config(0), gen.make_config(2, n_envs=12)):
        o = oracle_mod.render(wl)
        ref = oracle_mod.pack_obs(o["rgb"], o["depth"], 0.1, 10.0)
        for opts in ({}, {"big_px": 1}, {"arena_slots": 1}, {"hiz": 0}):
            sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
            try:
                for k, v in opts.items():
                    gx.gx_set_option(sc, k, v)
                dev = torch.device("cuda:0")
                t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).to(dev)
                K = wl.K
                obs = torch.full((wl.N, 4, wl.height, wl.width), 7.0, dtype=torch.float16, device=dev)
                gx.gx_render_batch_obs(sc, gx.camera_of(wl), wl.N, K, t(wl.env_scene, np.int32), t(wl.cam_pose, np.float32),
                                       t(wl.inst_mesh, np.int32) if K else None, t(wl.inst_xform, np.float32) if K else None,
                                       obs, 0.1, 10.0, torch.cuda.current_stream().cuda_stream)
                torch.cuda.synchronize()
                got = obs.cpu().numpy().view(np.uint16)
                # all four planes exact: N8 and N11 are implemented operation by operation, so the packed values are the
                # oracle's packing of the oracle's bytes
                assert np.array_equal(got[:, 3], ref[:, 3]), opts
                assert np.array_equal(got[:, :3], ref[:, :3]), opts
                with pytest.raises(gx.GxError):
                    gx.gx_render_batch_obs(sc, gx.camera_of(wl), wl.N, K, t(wl.env_scene, np.int32), t(wl.cam_pose, np.float32),
                                           t(wl.inst_mesh, np.int32) if K else None, t(wl.inst_xform, np.float32) if K else None,
                                           obs, 1.0, 1.0, 0)
            finally:
                gx.gx_destroy(sc)


@pytest.mark.parametrize("W,H", [(128, 96), (96, 128), (64, 128), (80, 48), (224, 224), (256, 144), (256, 256)])
def test_other_frame_shapes_room_scene(oracle_mod, W, H):
    """NEXT-3: frame shapes other than the configs' -- the room scene of configs[1] rendered at W x H (fx = fy * H / W),
    up to the 256x256 limit (Table 1 of the paper compares simulators at 128 to 256 pixels): more tiles
    per frame, more triangles on the block path and on the int64 path."""
    wl = gen.make_config(1, n_envs=6 if W * H <= 128 * 128 else 3)
    wl.width, wl.height = W, H
    wl.fy = 1.0
    wl.fx = H / W
    o = oracle_mod.render(wl)
    for opts in ({}, {"big_px": 6}, {"hiz": 0, "arena_slots": 1}):
        g = render_gpu(wl, options=opts)
        rep = compare(o, g)
        assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, (opts, rep)


def test_second_camera_is_a_second_slot(oracle_mod):
    """NEXT-3, several cameras per environment (the third-person debug view of PAPER.md:465-467): a second camera
    is a second environment slot with the same scene id and instance transforms and its own camera pose; the call
    renders both.  Checked against the oracle rendering the same doubled batch."""
    wl = gen.make_config(1, n_envs=4)
    other = gen.make_config(1, env_ids=[100, 101, 102, 103])     # poses of other environments of the same scene
    two = wl.subset(np.repeat(np.arange(4), 2))
    two.cam_pose = two.cam_pose.copy()
    two.cam_pose[1::2] = other.cam_pose                       # odd slots: the second camera, same instances
    o = oracle_mod.render(two)
    g = render_gpu(two)
    rep = compare(o, g)
    assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
    assert not np.array_equal(g["depth"][0], g["depth"][1])


def test_out_of_range_mesh_ids_are_empty_slots():
    """include/gx.h: an out-of-range env_scene / inst_mesh value is a precondition violation; the library treats
    the slot as empty and counts it instead of reading out of bounds."""
    wl = gen.make_config(0)
    ok = render_gpu(wl, stats=True)
    assert ok["stats"]["bad_ids"] == 0
    bad = wl.subset(np.arange(wl.N))
    bad.inst_mesh = bad.inst_mesh.copy()
    bad.inst_mesh[0, 0] = 7          # only mesh 0 exists
    bad.env_scene = bad.env_scene.copy()
    bad.env_scene[3] = 5
    g = render_gpu(bad, stats=True)
    assert g["stats"]["bad_ids"] == 2
    assert np.all(g["id"][3] == BG)                       # no scene: background
    for k in ("rgb", "depth", "id"):
        assert np.array_equal(g[k][1:3], ok[k][1:3])


def test_handle_reuse_varying_batches_and_host_subbatches(oracle_mod):
    """One handle, calls of different sizes and options in a row (the arena and its history-based sizing and the
    scratch buffers are reused and regrown), and the host entry point with a batch that is not a multiple of its
    sub-batches: every call must match the oracle."""
    import torch
    from paper_2306_07552_b200 import binding as gx
    wl = gen.make_config(2, n_envs=40)
    o = oracle_mod.render(wl)
    sc = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        for sel, opts in ((np.arange(40), {}), (np.arange(7), {"big_px": 3}), (np.arange(5, 38), {"hiz": 0}),
                          (np.arange(40), {"arena_slots": 100000, "hiz": 1, "big_px": 16}), (np.arange(1), {"arena_slots": 0}),
                          (np.arange(40), {"subcull": 0})):
            sub = wl.subset(sel)
            g = render_gpu(sub, scene=sc, options=opts)
            rep = compare({k: v[sel] for k, v in o.items()}, g)
            assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, (opts, rep)
            torch.cuda.synchronize()
    finally:
        gx.gx_destroy(sc)
    # host entry point: 1100 environments (the 40 environments repeated), uneven last sub-batch
    rep_idx = np.arange(1100) % 40
    big = wl.subset(rep_idx)
    g = render_gpu(big, host_api=True)
    rep = compare({k: v[rep_idx] for k, v in o.items()}, g)
    assert rep["id_mismatch"] == 0 and rep["depth_bits_differ"] == 0, rep
