"""gx_render_batch_noalloc (include/gx.h) against gx_render_batch.

Why the entry point exists: gx_render_batch keeps its record arena and per-call tables in buffers it gets from
cudaMalloc and returns with cudaFree when they must grow.  A renderer that lives inside somebody else's process
often may not do that: a simulation worker in a training process whose tensor allocator already holds the rest
of the device (a cudaMalloc of the arena fails, or takes what the policy's next batch needs), or a render call
issued while the policy's inference runs on other streams (cudaMalloc / cudaFree wait for the whole device, so a
growing render call stalls them all).  For those callers gx_render_batch_noalloc takes its intermediate memory
from one GX_NOALLOC_SCRATCH_BYTES (64 MiB) array built into the library's device image and never allocates.

What is checked here, on a B200:
  * the images equal gx_render_batch's byte for byte (depth bits, ids, RGB -- the tolerance the parity tests of
    this repository use for the CUDA path against itself: none), on calls made one right after the other with
    no synchronisation between them, where the second call is smaller than, or of another frame shape than, the
    first, so that anything left in the shared array by the first call would show if it were read;
  * several waves (the 40-environment call does not fit the arena left in the array in one go);
  * a shape beyond the array is refused with GX_ERR_UNSUPPORTED, a message that names the limit, and no write;
  * the handle's allocating path still works afterwards and gives the same images.

The file sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`, and a failure here must not
hide the parity tests.  It needs nothing from the tests before it and passes alone in a fresh process, where its
first call is also the first use of the library on the device (the per-device set-up of the entry point).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import pytest

from paper_2306_07552_b200 import gen


def _upload(wl):
    import torch
    dev = torch.device("cuda:0")
    K = wl.K
    return dict(
        env_scene=torch.from_numpy(np.ascontiguousarray(wl.env_scene, np.int32)).to(dev),
        cam_pose=torch.from_numpy(np.ascontiguousarray(wl.cam_pose, np.float32)).to(dev),
        inst_mesh=torch.from_numpy(np.ascontiguousarray(wl.inst_mesh, np.int32)).to(dev) if K else None,
        inst_xform=torch.from_numpy(np.ascontiguousarray(wl.inst_xform, np.float32)).to(dev) if K else None)


def _outputs(wl):
    """Caller-owned outputs, pre-filled with values no render produces."""
    import torch
    dev = torch.device("cuda:0")
    N, H, W = wl.N, wl.height, wl.width
    return dict(rgb=torch.full((N, H, W, 3), 77, dtype=torch.uint8, device=dev),
                depth=torch.full((N, H, W), -1.0, dtype=torch.float32, device=dev),
                id=torch.full((N, H, W), 12345, dtype=torch.int32, device=dev))


def _enqueue(fn, scene, wl, inp, out):
    import torch
    from paper_2306_07552_b200 import binding as gx
    fn(scene, gx.camera_of(wl), wl.N, wl.K, inp["env_scene"], inp["cam_pose"], inp["inst_mesh"], inp["inst_xform"],
       out["rgb"], out["depth"], out["id"], torch.cuda.current_stream().cuda_stream)


def _host(out):
    return dict(rgb=out["rgb"].cpu().numpy(), depth=out["depth"].cpu().numpy().view(np.uint32),
                id=out["id"].cpu().numpy().view(np.uint32))


def _same(a, b, what):
    for k in ("id", "depth", "rgb"):
        assert np.array_equal(a[k], b[k]), f"{what}: {k} differs at {int((a[k] != b[k]).sum())} elements"


@pytest.mark.gpu
@pytest.mark.parametrize("options", [{}, {"occlusion": 0}, {"hiz": 0, "big_px": 6}])
def test_noalloc_equals_render_batch_on_calls_in_a_row(options):
    import torch
    from paper_2306_07552_b200 import binding as gx

    assert torch.cuda.is_available()
    # one scene handle, three call shapes: 40 environments of configs[2] (several waves in the 64 MiB array), 7 other
    # environments of it in another order (a smaller call right after a larger one), and the same 40 again
    big = gen.make_config(2, env_ids=np.arange(40))
    small = gen.make_config(2, env_ids=np.array([1000, 17, 512, 3, 256, 900, 41]))
    scene = gx.gx_create_scene(big.static_meshes, big.dyn_meshes, 0)
    try:
        for name, value in options.items():
            gx.gx_set_option(scene, name, value)
        calls = [big, small, big]
        inputs = [_upload(wl) for wl in calls]
        ref = []
        for wl, inp in zip(calls[:2], inputs[:2]):          # the existing, allocating path
            out = _outputs(wl)
            _enqueue(gx.gx_render_batch, scene, wl, inp, out)
            torch.cuda.synchronize()
            ref.append(_host(out))
        assert (ref[0]["id"] != 0xFFFFFFFF).mean() > 0.9     # something is actually drawn
        outs = [_outputs(wl) for wl in calls]
        for wl, inp, out in zip(calls, inputs, outs):        # in a row on one stream, nothing in between
            _enqueue(gx.gx_render_batch_noalloc, scene, wl, inp, out)
        torch.cuda.synchronize()
        got = [_host(o) for o in outs]
        _same(ref[0], got[0], "first call (40 environments)")
        _same(ref[1], got[1], "second call (7 environments, right after the first)")
        _same(ref[0], got[2], "third call (the first again)")
        # the allocating path of the same handle is undisturbed
        out = _outputs(small)
        _enqueue(gx.gx_render_batch, scene, small, inputs[1], out)
        torch.cuda.synchronize()
        _same(ref[1], _host(out), "gx_render_batch after the no-alloc calls")
    finally:
        gx.gx_destroy(scene)


@pytest.mark.gpu
def test_noalloc_other_frame_shapes_share_the_array():
    """configs[0] (64x64, K = 2) and a 128x128 room call alternate on the same device array: the table layout of one
    call lies across the other's, so stale words are everywhere a missing clear would read them."""
    import torch
    from paper_2306_07552_b200 import binding as gx

    tiny = gen.make_config(0)
    room = gen.make_config(1, n_envs=5)
    s_tiny = gx.gx_create_scene(tiny.static_meshes, tiny.dyn_meshes, 0)
    s_room = gx.gx_create_scene(room.static_meshes, room.dyn_meshes, 0)
    try:
        pairs = [(s_tiny, tiny), (s_room, room), (s_tiny, tiny), (s_room, room)]
        inputs = {id(wl): _upload(wl) for _, wl in pairs}
        ref = {}
        for sc, wl in pairs[:2]:
            out = _outputs(wl)
            _enqueue(gx.gx_render_batch, sc, wl, inputs[id(wl)], out)
            torch.cuda.synchronize()
            ref[id(wl)] = _host(out)
        outs = [_outputs(wl) for _, wl in pairs]
        for (sc, wl), out in zip(pairs, outs):               # two handles, one stream: ordered, so no race on the array
            _enqueue(gx.gx_render_batch_noalloc, sc, wl, inputs[id(wl)], out)
        torch.cuda.synchronize()
        for k, ((_, wl), out) in enumerate(zip(pairs, outs)):
            _same(ref[id(wl)], _host(out), f"call {k} ({wl.name})")
    finally:
        gx.gx_destroy(s_tiny)
        gx.gx_destroy(s_room)


@pytest.mark.gpu
def test_noalloc_refuses_shapes_beyond_the_array():
    """1024 environments at 128x128 need about 157 MB of tables alone: UNSUPPORTED, a message with the numbers, and
    not a byte of the outputs written."""
    import torch
    from paper_2306_07552_b200 import binding as gx

    wl = gen.make_config(2, n_envs=2)
    scene = gx.gx_create_scene(wl.static_meshes, wl.dyn_meshes, 0)
    try:
        dev = torch.device("cuda:0")
        N, K, H, W = 1024, wl.K, wl.height, wl.width
        env_scene = torch.zeros(N, dtype=torch.int32, device=dev)
        cam_pose = torch.from_numpy(np.ascontiguousarray(wl.cam_pose[:1], np.float32)).to(dev).repeat(N, 1).contiguous()
        inst_mesh = torch.full((N, K), -1, dtype=torch.int32, device=dev)
        inst_xform = torch.zeros((N, K, 16), dtype=torch.float32, device=dev)
        rgb = torch.full((N, H, W, 3), 77, dtype=torch.uint8, device=dev)
        depth = torch.full((N, H, W), -1.0, dtype=torch.float32, device=dev)
        with pytest.raises(gx.GxError) as ei:
            gx.gx_render_batch_noalloc(scene, gx.camera_of(wl), N, K, env_scene, cam_pose, inst_mesh, inst_xform, rgb, depth,
                                       None, torch.cuda.current_stream().cuda_stream)
        assert ei.value.code == gx.GX_ERR_UNSUPPORTED
        msg = str(ei.value)
        assert "GX_NOALLOC_SCRATCH_BYTES" in msg and str(gx.GX_NOALLOC_SCRATCH_BYTES) in msg, msg
        torch.cuda.synchronize()
        assert bool((rgb == 77).all()) and bool((depth == -1.0).all())
        # the same handle renders a batch that does fit right afterwards
        sub = gen.make_config(2, n_envs=2)
        out = _outputs(sub)
        _enqueue(gx.gx_render_batch_noalloc, scene, sub, _upload(sub), out)
        torch.cuda.synchronize()
        assert (_host(out)["id"] != 0xFFFFFFFF).mean() > 0.9
    finally:
        gx.gx_destroy(scene)


def test_noalloc_argument_errors_need_no_gpu():
    from paper_2306_07552_b200 import binding as gx, build
    lib = ctypes.CDLL(build.build())
    lib.gx_last_error.restype = ctypes.c_char_p
    assert lib.gx_render_batch_noalloc(None, None, 0, 0, None, None, None, None, None, None, None, None) == gx.GX_ERR_INVALID_ARG
    assert b"NULL" in lib.gx_last_error()
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "gx.h")).read()
    assert "#define GX_NOALLOC_SCRATCH_BYTES (64u << 20)" in hdr and gx.GX_NOALLOC_SCRATCH_BYTES == 64 << 20
