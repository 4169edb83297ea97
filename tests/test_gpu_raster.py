"""Parity of the CUDA soft-silhouette rasteriser and its adjoint (csrc/gs_raster.cu, through the C ABI) with the fp64
oracle (oracle/raster_oracle.py), pixel by pixel and vertex by vertex, and the pixels-to-parameters loop of the paper
closed through the physics adjoint (render the unrolled state, compare with the target image, backpropagate)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from oracle import raster_oracle as ro
from paper_2104_02646_b200 import gradsim as gs
from paper_2104_02646_b200 import scenes

from gpu_util import dev, host, rel_inf

pytestmark = pytest.mark.gpu


def _camera(W, H, sigma, look=(0.3, -0.45)):
    th, ph = look
    Ry = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]])
    Rx = np.array([[1, 0, 0], [0, np.cos(ph), -np.sin(ph)], [0, np.sin(ph), np.cos(ph)]])
    R = Rx @ Ry
    return R, np.array([-0.1, 0.05, 0.9]), 2.2, 2.4, W, H, sigma


def _itris(a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.int32), device="cuda:0")


@pytest.mark.parametrize("W,H,sigma", [(64, 48, 3e-4), (45, 37, 3e-3), (130, 70, 1e-5)])
def test_silhouette_and_gradient_match_the_oracle(W, H, sigma):
    """A deformed 12 x 12 cloth sheet (242 triangles, two environments with different shapes) seen by a rotated, off-axis
    camera: image <= 1e-5 absolute, loss <= 1e-4 relative, dL/dx <= 2e-3 (A18 norm); sizes that are not multiples of the
    16-pixel tile; a wide and a narrow edge blur."""
    sc = scenes.make_scene(1, small=True)
    r = scenes.rng_for(1, "misc", 91)
    x = np.stack([sc.x0[0] + 0.004 * r.normal(size=sc.x0[0].shape), sc.x0[0] + 0.004 * r.normal(size=sc.x0[0].shape)]).astype(np.float32)
    x[:, :, 1] += 0.02 * np.sin(40 * x[:, :, 0])  # wrinkles: overlapping projections
    cam_args = _camera(W, H, sigma)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    tris = sc.tris
    img = host(gs.render_silhouette(dev(x), _itris(tris), cg))
    ref = np.stack([ro.silhouette(x[e], tris, co) for e in range(2)])
    assert ref.max() > 0.99 and ref.min() < 0.01 and ((ref > 0.05) & (ref < 0.95)).sum() > 20
    assert np.abs(img - ref).max() <= 1e-5
    target = np.stack([ro.silhouette(x[e] + 0.01 * r.normal(size=x[e].shape), tris, co) for e in range(2)]).astype(np.float32)
    loss, adj, im2 = gs.loss_silhouette(dev(x), _itris(tris), cg, dev(target), want_image=True)
    Lg = [ro.silhouette_loss_and_grad(x[e], tris, co, target[e]) for e in range(2)]
    assert rel_inf(host(loss), np.array([l for l, _ in Lg])) <= 1e-4
    gref = np.stack([g for _, g in Lg])
    assert np.abs(gref).max() > 0
    assert rel_inf(host(adj), gref) <= 2e-3
    assert np.abs(host(im2) - ref).max() <= 1e-5
    # accumulate + explicit scale
    loss2, _, _ = gs.loss_silhouette(dev(x), _itris(tris), cg, dev(target), scale=0.5 / (W * H), loss=loss, accumulate=True, want_adj=False)
    assert rel_inf(host(loss2), 1.5 * np.array([l for l, _ in Lg])) <= 1e-4


def test_raster_edge_cases():
    cam_args = _camera(33, 20, 1e-3)
    cg, co = gs.make_camera(*cam_args), ro.Camera(*cam_args)
    x = np.array([[[0.0, 0.0, 0.0], [0.2, 0.0, 0.0], [0.0, 0.0, 0.2], [0.1, 0.3, -5.0]]], np.float32)
    # no triangles: background everywhere, zero gradient
    img = host(gs.render_silhouette(dev(x), _itris(np.zeros((0, 3))), cg))
    assert np.all(img == 0)
    # a triangle with a vertex behind the near plane is not drawn; the other one is
    tris = np.array([[0, 1, 2], [0, 1, 3]])
    assert ro.project(x[0].astype(np.float64), co)[1][3] < 0
    img = host(gs.render_silhouette(dev(x), _itris(tris), cg))
    assert np.abs(img - ro.silhouette(x[0], tris, co)).max() <= 1e-5 and img.max() > 0.9
    # bad arguments come back as codes
    bad = gs.make_camera(*_camera(0, 20, 1e-3))
    with pytest.raises(gs.GradSimError) as e:
        gs.render_silhouette(dev(x), _itris(tris), bad)
    assert e.value.code == gs.GS_EINVAL


def test_pixels_to_parameters_gradient_through_the_rollout():
    """The loop of PAPER.md:216: unroll the cloth, render the final state, pixelwise MSE against a target image, and
    backpropagate through rasteriser AND physics: dL/dv0 and dL/dk_mu from the CUDA path against the two oracles chained the
    same way (airborne sheet: no contact-branch flips, A20)."""
    sc = scenes.make_scene(1, small=True)
    sc.plane_d = -1e6
    sc.v0 = (sc.v0 + scenes.rng_for(1, "misc", 92).normal(0, 0.2, sc.v0.shape)).astype(np.float32)
    sc.v0[:, sc.pinned.astype(bool)] = 0
    T = sc.n_substeps
    cam_args = _camera(96, 64, 1e-3)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    # oracle chain
    o = orc.Oracle(sc)
    rollo = o.rollout(sc.x0, sc.v0, T, rec_times=[T])
    xT = rollo["xT"]
    target = ro.silhouette(xT[0] + np.array([0.01, 0.0, 0.005]), sc.tris, co).astype(np.float32)[None]
    L, gx = ro.silhouette_loss_and_grad(xT[0], sc.tris, co, target[0].astype(np.float64))
    o.zero_grads()
    ax0, av0 = o.rollout_backward(rollo, [T], gx[None, None])
    # CUDA chain
    m = gs.Model(sc)
    tape = m.tape(T)
    m.zero_grads()
    xTg, _ = tape.rollout(dev(sc.x0), dev(sc.v0))
    loss, adj, _ = gs.loss_silhouette(xTg, _itris(sc.tris), cg, dev(target))
    ax0g, av0g = tape.backward(adj_x_T=adj)
    assert rel_inf(host(loss), np.array([L])) <= 1e-3
    assert rel_inf(host(av0g), av0) <= 2e-3 and rel_inf(host(ax0g), ax0) <= 2e-3
    assert rel_inf(host(m.param_grads("tri_mu")), o.grads("tri_mu")) <= 2e-3


# ------------------------------------------------------------------------------------------ colour channel (reading A22b)
SHADE = (0.05, 1e-3, 3.0, (0.1, 0.2, 0.3))  # gamma, eps, far, background


@pytest.mark.parametrize("W,H,sigma", [(64, 48, 3e-4), (45, 37, 3e-3)])
def test_rgb_image_and_gradients_match_the_oracle(W, H, sigma):
    """The wrinkled 12 x 12 sheet of the silhouette test with random vertex colours, two environments: image <= 1e-4
    absolute per channel (a weight D_j e^{zbar_j / gamma} carries the fp32 rounding of s_j / sigma, up to 40 x 1e-6 relative), loss <= 1e-4 relative, dL/dx and dL/dcolour <= 2e-3 (A18 norm), image sizes that are not multiples
    of the tile, overlapping projections (the depth softmax decides), many exterior pixels inside the 40 sigma cut."""
    sc = scenes.make_scene(1, small=True)
    r = scenes.rng_for(1, "misc", 93)
    x = np.stack([sc.x0[0] + 0.004 * r.normal(size=sc.x0[0].shape), sc.x0[0] + 0.004 * r.normal(size=sc.x0[0].shape)]).astype(np.float32)
    x[:, :, 1] += 0.02 * np.sin(40 * x[:, :, 0])
    col = r.uniform(0.0, 1.0, x.shape).astype(np.float32)
    cam_args = _camera(W, H, sigma)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    so, sg = ro.Shading(*SHADE), gs.make_shading(*SHADE)
    tris = sc.tris
    img = host(gs.render_rgb(dev(x), _itris(tris), dev(col), cg, sg))
    ref = np.stack([ro.rgb(x[e], tris, col[e], co, so) for e in range(2)])
    assert img.shape == ref.shape == (2, 3, H, W)
    assert np.abs(ref - np.array(SHADE[3])[None, :, None, None]).max() > 0.3  # the sheet is visible
    assert np.abs(img - ref).max() <= 1e-4
    target = np.stack([ro.rgb(x[e] + 0.01 * r.normal(size=x[e].shape), tris, r.uniform(0, 1, col[e].shape), co, so) for e in range(2)]).astype(np.float32)
    loss, adj, adj_c, im2 = gs.loss_rgb(dev(x), _itris(tris), dev(col), cg, sg, dev(target), want_image=True)
    Lg = [ro.rgb_loss_and_grads(x[e], tris, col[e], co, so, target[e]) for e in range(2)]
    assert rel_inf(host(loss), np.array([l[0] for l in Lg])) <= 1e-4
    gx, gc = np.stack([l[1] for l in Lg]), np.stack([l[2] for l in Lg])
    assert np.abs(gx).max() > 0 and np.abs(gc).max() > 0
    assert rel_inf(host(adj), gx) <= 2e-3
    assert rel_inf(host(adj_c), gc) <= 2e-3
    assert np.abs(host(im2) - ref).max() <= 1e-4
    # accumulate + explicit scale; gradients on request only
    loss2, a2, c2, _ = gs.loss_rgb(dev(x), _itris(tris), dev(col), cg, sg, dev(target), scale=0.5 / (3 * W * H), loss=loss, accumulate=True, want_adj=False,
                                   want_adj_colour=False)
    assert a2 is None and c2 is None
    assert rel_inf(host(loss2), 1.5 * np.array([l[0] for l in Lg])) <= 1e-4


def test_rgb_small_gamma_and_edge_cases():
    """A sharp depth softmax (gamma = 2e-3: exponents of several hundred, held by the running maximum) still matches; no
    triangles -> the background exactly; a degenerate triangle and one behind the near plane are skipped; bad shading
    parameters come back as codes."""
    sc = scenes.make_scene(1, small=True)
    r = scenes.rng_for(1, "misc", 94)
    x = (sc.x0[:1] + 0.004 * r.normal(size=sc.x0[:1].shape)).astype(np.float32)
    x[:, :, 1] += 0.02 * np.sin(40 * x[:, :, 0])
    col = r.uniform(0.0, 1.0, x.shape).astype(np.float32)
    cam_args = _camera(80, 56, 1e-3)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    sharp = (2e-3, 1e-3, 3.0, (0.0, 0.0, 0.0))
    img = host(gs.render_rgb(dev(x), _itris(sc.tris), dev(col), cg, gs.make_shading(*sharp)))
    ref = ro.rgb(x[0], sc.tris, col[0], co, ro.Shading(*sharp))[None]
    # zbar / gamma ~ 350: an fp32 rounding of zbar moves a weight by ~ 4e-5 relative per ulp -- 1e-3 absolute on the image
    assert np.abs(img - ref).max() <= 1e-3 and np.abs(img - ref).mean() <= 2e-5
    sg, so = gs.make_shading(*SHADE), ro.Shading(*SHADE)
    img0 = host(gs.render_rgb(dev(x), _itris(np.zeros((0, 3))), dev(col), cg, sg))
    assert all(np.all(img0[0, c] == np.float32(SHADE[3][c])) for c in range(3))
    x4 = np.array([[[0.0, 0.0, 0.0], [0.2, 0.0, 0.0], [0.0, 0.0, 0.2], [0.1, 0.3, -5.0], [0.1, 0.0, 0.0]]], np.float32)
    c4 = r.uniform(0, 1, x4.shape).astype(np.float32)
    tris = np.array([[0, 1, 2], [0, 1, 3], [0, 4, 1]])  # drawn, behind the near plane, collinear
    img4 = host(gs.render_rgb(dev(x4), _itris(tris), dev(c4), cg, sg))
    assert np.abs(img4[0] - ro.rgb(x4[0], tris, c4[0], co, so)).max() <= 2e-5
    assert np.abs(img4[0] - ro.rgb(x4[0], tris[:1], c4[0], co, so)).max() <= 2e-5
    for bad in [(0.0, 1e-3, 3.0, (0, 0, 0)), (0.05, 1e-3, 1e-4, (0, 0, 0))]:
        with pytest.raises(gs.GradSimError) as e:
            gs.render_rgb(dev(x4), _itris(tris), dev(c4), cg, gs.make_shading(*bad))
        assert e.value.code == gs.GS_EINVAL


def test_colour_pixels_to_parameters_gradient_through_the_rollout():
    """PAPER.md:216 with the colour image: unroll the airborne sheet, render x_T in colour, pixelwise MSE, and back through
    rasteriser and physics: dL/dv0, dL/dx0 and dL/dk_mu against the two oracles chained the same way; dL/dcolour at x_T."""
    sc = scenes.make_scene(1, small=True)
    sc.plane_d = -1e6
    sc.v0 = (sc.v0 + scenes.rng_for(1, "misc", 95).normal(0, 0.2, sc.v0.shape)).astype(np.float32)
    sc.v0[:, sc.pinned.astype(bool)] = 0
    T = sc.n_substeps
    cam_args = _camera(96, 64, 1e-3)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    so, sg = ro.Shading(*SHADE), gs.make_shading(*SHADE)
    r = scenes.rng_for(1, "misc", 96)
    col = r.uniform(0.0, 1.0, sc.x0.shape).astype(np.float32)
    o = orc.Oracle(sc)
    rollo = o.rollout(sc.x0, sc.v0, T, rec_times=[T])
    xT = rollo["xT"]
    target = ro.rgb(xT[0] + np.array([0.01, 0.0, 0.005]), sc.tris, r.uniform(0, 1, col[0].shape), co, so).astype(np.float32)[None]
    L, gx, gc = ro.rgb_loss_and_grads(xT[0], sc.tris, col[0], co, so, target[0].astype(np.float64))
    o.zero_grads()
    ax0, av0 = o.rollout_backward(rollo, [T], gx[None, None])
    m = gs.Model(sc)
    tape = m.tape(T)
    m.zero_grads()
    xTg, _ = tape.rollout(dev(sc.x0), dev(sc.v0))
    loss, adj, adj_c, _ = gs.loss_rgb(xTg, _itris(sc.tris), dev(col), cg, sg, dev(target))
    ax0g, av0g = tape.backward(adj_x_T=adj)
    assert rel_inf(host(loss), np.array([L])) <= 1e-3
    assert rel_inf(host(adj_c), gc[None]) <= 2e-3
    assert rel_inf(host(av0g), av0) <= 2e-3 and rel_inf(host(ax0g), ax0) <= 2e-3
    assert rel_inf(host(m.param_grads("tri_mu")), o.grads("tri_mu")) <= 2e-3


@pytest.mark.parametrize("plan", [gs.GS_PLAN_RESIDENT, gs.GS_PLAN_STREAMING])
def test_solid_pixels_to_parameters_gradient_through_the_rollout(plan):
    """The deformable-solid loop of the paper (material parameters and masses of an FEM solid from images):
    unroll the falling, bouncing box of config 0 (small), draw the BOUNDARY FACES of its tet mesh at x_T, pixelwise MSE against
    a target silhouette, and back through rasteriser and physics: dL/dmu, dL/dlambda, dL/dk_damp per tet, dL/dm per particle,
    dL/dx0, dL/dv0 against the two oracles chained the same way, on both plans."""
    sc = scenes.make_scene(0, small=True)
    T = sc.n_substeps
    faces = scenes.boundary_faces(sc.tets)
    th = 0.5
    R = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]])
    cam_args = (R, -R @ sc.x0[0].astype(np.float64).mean(0) + np.array([0.0, 0.05, 1.2]), 2.0, 2.0, 96, 80, 1e-3)
    co, cg = ro.Camera(*cam_args), gs.make_camera(*cam_args)
    o = orc.Oracle(sc)
    rollo = o.rollout(sc.x0, sc.v0, T, rec_times=[T])
    xT = rollo["xT"]
    target = ro.silhouette(xT[0] * np.array([1.05, 0.9, 1.0]) + np.array([0.02, 0.0, 0.01]), faces, co).astype(np.float32)[None]
    L, gx = ro.silhouette_loss_and_grad(xT[0], faces, co, target[0].astype(np.float64))
    assert L > 1e-4 and np.abs(gx).max() > 0
    o.zero_grads()
    ax0, av0 = o.rollout_backward(rollo, [T], gx[None, None])
    m = gs.Model(sc, plan=plan)
    assert m.plan == plan
    tape = m.tape(T)
    m.zero_grads()
    xTg, _ = tape.rollout(dev(sc.x0), dev(sc.v0))
    loss, adj, _ = gs.loss_silhouette(xTg, _itris(faces), cg, dev(target))
    ax0g, av0g = tape.backward(adj_x_T=adj)
    assert m.check_finite() == -1
    assert rel_inf(host(loss), np.array([L])) <= 1e-3
    assert rel_inf(host(av0g), av0) <= 2e-3 and rel_inf(host(ax0g), ax0) <= 2e-3
    for g in ("tet_mu", "tet_lambda", "tet_damp", "mass"):
        assert np.abs(o.grads(g)).max() > 0
        assert rel_inf(host(m.param_grads(g)), o.grads(g)) <= 2e-3, g
