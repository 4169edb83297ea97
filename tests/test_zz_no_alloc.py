"""gs_loss_silhouette_static: the entry point that allocates nothing (scratch in a static device array of
GS_RASTER_STATIC_BYTES inside the library, include/gradsim.h) against the existing path gs_loss_silhouette, on two calls in a
row.  Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests:
it depends on no state but the library's own array, whose previous contents each call overwrites or clears."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2104_02646_b200 import gradsim as gs
from paper_2104_02646_b200 import scenes


def _camera(W, H, sigma):
    th, ph = 0.3, -0.45
    Ry = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]])
    Rx = np.array([[1, 0, 0], [0, np.cos(ph), -np.sin(ph)], [0, np.sin(ph), np.cos(ph)]])
    return gs.make_camera(Rx @ Ry, np.array([-0.1, 0.05, 0.9]), 2.2, 2.4, W, H, sigma)


def _scene(E, seed, amp):
    sc = scenes.make_scene(1, small=True)
    r = scenes.rng_for(1, "misc", seed)
    x = (sc.x0[0][None] + amp * r.normal(size=(E,) + sc.x0[0].shape)).astype(np.float32)
    x[:, :, 1] += 0.02 * np.sin(40 * x[:, :, 0])
    return x, np.ascontiguousarray(sc.tris, dtype=np.int32)


def test_problem_beyond_the_static_block_is_rejected_without_a_device():
    """the size check precedes every CUDA call: GS_EINVAL and a message that names the limit, also on a box without a GPU"""
    L = gs.lib()
    E, N, Mt = 400, 1089, 1922
    assert L.gs_raster_scratch_bytes(E, N, Mt) > gs.RASTER_STATIC_BYTES
    cam = _camera(16, 16, 1e-3)
    one = C.c_void_p(256)  # never dereferenced
    assert L.gs_loss_silhouette_static(E, N, one, Mt, one, C.byref(cam), one, 1.0, 0, one, None, None, None) == gs.GS_EINVAL
    msg = L.gs_last_error()
    assert b"GS_RASTER_STATIC_BYTES" in msg and str(gs.RASTER_STATIC_BYTES).encode() in msg
    assert L.gs_loss_silhouette_static(0, N, one, Mt, one, C.byref(cam), one, 1.0, 0, one, None, None, None) == gs.GS_EINVAL
    assert L.gs_loss_silhouette_static(1, N, one, Mt, one, C.byref(cam), None, 1.0, 0, one, None, None, None) == gs.GS_EINVAL  # no target
    src = open(gs.__file__.replace("gradsim.py", "../include/gradsim.h")).read()
    assert "#define GS_RASTER_STATIC_BYTES (8u << 20)" in src and gs.RASTER_STATIC_BYTES == 8 << 20


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    """Two different problems back to back through the shared array (the second smaller, so that stale records of the first
    lie beyond its own and stale NDC gradients under them), then the first again: image <= 1e-5 absolute, loss <= 1e-4
    relative, dL/dx <= 2e-3 of the array's maximum (the tolerances of tests/test_gpu_raster.py; the two paths run the same
    kernels, only the float atomics' order differs), and no device memory is allocated by the calls."""
    d = lambda a: torch.as_tensor(a, device="cuda:0")
    cases = []
    for E, seed, amp, W, H, sigma in [(3, 201, 0.004, 64, 48, 3e-4), (1, 202, 0.006, 45, 37, 3e-3), (3, 201, 0.004, 64, 48, 3e-4)]:
        x, tris = _scene(E, seed, amp)
        cam = _camera(W, H, sigma)
        xd, td = d(x), d(tris)
        target = gs.render_silhouette(d(x + np.float32(0.01)), td, cam)
        ref_loss, ref_adj, ref_img = gs.loss_silhouette(xd, td, cam, target, want_image=True)
        outs = (torch.full((E,), 7.0, device="cuda:0"), torch.full_like(xd, 7.0), torch.full((E, H, W), 7.0, device="cuda:0"))
        cases.append((xd, td, cam, target, ref_loss, ref_adj, ref_img, outs))
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for xd, td, cam, target, _, _, _, (loss, adj, img) in cases:  # back to back, no synchronisation in between
        gs.loss_silhouette_static(xd, td, cam, target, loss, adj=adj, image=img)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= before  # nothing was taken from the device (the array was there since load)
    for _, _, _, _, ref_loss, ref_adj, ref_img, (loss, adj, img) in cases:
        assert float(ref_img.max()) > 0.99 and float(ref_adj.abs().max()) > 0
        assert float((img - ref_img).abs().max()) <= 1e-5
        assert float(((loss - ref_loss).abs() / ref_loss.abs()).max()) <= 1e-4
        assert float((adj - ref_adj).abs().max()) <= 2e-3 * float(ref_adj.abs().max())
    # accumulate keeps the caller's loss; gradients and image stay optional
    xd, td, cam, target, ref_loss, _, _, (loss, _, _) = cases[0]
    gs.loss_silhouette_static(xd, td, cam, target, loss, accumulate=True)
    assert float(((loss - 2 * ref_loss).abs() / ref_loss.abs()).max()) <= 2e-4
