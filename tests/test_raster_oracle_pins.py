"""Pins of the soft-silhouette oracle (oracle/raster_oracle.py; reading A22) against what
SPEC.md:240-251 and the mathematics fix.  No GPU."""
import numpy as np

from oracle import raster_oracle as ro


def _cam(W=32, H=24, sigma=1e-3, fx=1.0, fy=1.0, t=(0.0, 0.0, 5.0)):
    return ro.Camera(np.eye(3), t, fx, fy, W, H, sigma)


def test_projection_closed_forms():
    """a point on the optical axis -> NDC (0, 0); a point at the right edge of a 90-degree frustum
    (fx = 1 / tan(pi/4) = 1) at depth z -> u = +1; a square of half-size 1 at z = 5 -> corners at (+-0.2, +-0.2)."""
    cam = _cam(t=(0.0, 0.0, 0.0))
    ndc, z = ro.project(np.array([[0.0, 0.0, 3.0], [2.5, 0.0, 2.5], [1.0, -1.0, 5.0], [-1.0, 1.0, 5.0]]), cam)
    assert np.allclose(ndc[0], 0) and z[0] == 3.0
    assert np.allclose(ndc[1], [1.0, 0.0])
    assert np.allclose(ndc[2], [0.2, -0.2]) and np.allclose(ndc[3], [-0.2, 0.2])
    # rotation + translation: camera at (0, 0, -4) looking along +z after a quarter turn about y
    R = np.array([[0.0, 0.0, -1.0], [0.0, 1.0, 0.0], [1.0, 0.0, 0.0]])
    cam2 = ro.Camera(R, (0.0, 0.0, 4.0), 2.0, 2.0, 8, 8, 1e-3)
    ndc2, z2 = ro.project(np.array([[1.0, 0.5, 0.25]]), cam2)
    assert np.allclose(z2, [5.0]) and np.allclose(ndc2, [[2.0 * -0.25 / 5.0, 2.0 * 0.5 / 5.0]])


def test_silhouette_values_the_spec_fixes():
    """SPEC.md:251 examples: no triangles -> 0 everywhere; a pixel centre exactly on an edge -> D = sigmoid(0) = 1/2; a
    large triangle with a small sigma -> >= 0.999 inside; agreement with the hard point-in-triangle test as sigma -> 0."""
    cam = _cam(W=4, H=4, sigma=1e-2)
    x = np.array([[-20.0, -10.0, 0.0], [20.0, -10.0, 0.0], [0.0, 30.0, 0.0]])  # covers the whole image (NDC [-1, 1]^2)
    assert np.all(ro.silhouette(x, np.zeros((0, 3), int), cam) == 0)
    # pixel (i=2, j=1) has its centre at (u, v) = (0.25, -0.25): put an edge through it (the line v = -0.25, at z = 5 -> y = -1.25)
    xe = np.array([[-10.0, -1.25, 0.0], [10.0, -1.25, 0.0], [0.0, 10.0, 0.0]])
    S = ro.silhouette(xe, [[0, 1, 2]], cam)
    assert abs(S[1, 2] - 0.5) < 1e-12 and S[2, 2] > 0.99 and S[0, 2] < 0.01
    big = ro.silhouette(x, [[0, 1, 2]], _cam(W=4, H=4, sigma=1e-5))
    assert big.min() >= 0.999
    rng = np.random.default_rng(7)
    xr = np.concatenate([rng.uniform(-4, 4, (30, 2)), rng.uniform(-0.5, 0.5, (30, 1))], 1)
    tris = rng.integers(0, 30, (12, 3))
    tris = tris[(tris[:, 0] != tris[:, 1]) & (tris[:, 1] != tris[:, 2]) & (tris[:, 0] != tris[:, 2])]
    camr = _cam(W=48, H=48, sigma=1e-7)
    soft, hard = ro.silhouette(xr, tris, camr), ro.hard_silhouette(xr, tris, camr)
    assert ((soft > 0.5) == hard).mean() >= 0.999
    # winding does not matter; a triangle behind the near plane is not drawn
    assert np.allclose(ro.silhouette(xe, [[0, 2, 1]], cam), S)
    xb = xe.copy(); xb[2, 2] = -10.0
    assert np.all(ro.silhouette(xb, [[0, 1, 2]], cam) == 0)


def test_silhouette_bounds_and_union():
    """0 <= S <= 1; S of a mesh >= S of any sub-mesh (1 - prod is monotone); two copies of a triangle give 1 - (1 - D)^2."""
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.uniform(-3, 3, (12, 2)), rng.uniform(-0.3, 0.3, (12, 1))], 1)
    tris = np.array([[0, 1, 2], [3, 4, 5], [6, 7, 8], [9, 10, 11], [0, 4, 8]])
    cam = _cam(sigma=3e-3)
    S = ro.silhouette(x, tris, cam)
    assert S.min() >= 0 and S.max() <= 1
    for j in range(len(tris)):
        assert np.all(S >= ro.silhouette(x, tris[j:j + 1], cam) - 1e-15)
    D = ro.silhouette(x, tris[:1], cam)
    assert np.allclose(ro.silhouette(x, tris[[0, 0]], cam), 1 - (1 - D) ** 2, atol=1e-15)


def test_silhouette_loss_gradient_vs_fd():
    """dL/dx of the pixelwise MSE (hand-written chain rule) against central finite differences, camera rotated and
    off-axis, overlapping triangles, sigma wide enough that many pixels sit on the sigmoid's slope."""
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(-2.5, 2.5, (9, 2)), rng.uniform(-0.4, 0.4, (9, 1))], 1)
    tris = np.array([[0, 1, 2], [2, 3, 4], [4, 5, 6], [6, 7, 8], [1, 5, 8]])
    th = 0.3
    R = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]]) @ np.array([[1, 0, 0], [0, np.cos(0.2), -np.sin(0.2)], [0, np.sin(0.2), np.cos(0.2)]])
    cam = ro.Camera(R, (0.2, -0.1, 6.0), 1.7, 1.9, 40, 30, 2e-2)
    target = ro.silhouette(x + 0.15 * rng.normal(size=x.shape), tris, cam)
    L, g = ro.silhouette_loss_and_grad(x, tris, cam, target)
    assert L > 0 and np.abs(g).max() > 0
    eps = 1e-6
    fd = np.zeros_like(x)
    for i in range(x.shape[0]):
        for r in range(3):
            d = np.zeros_like(x); d[i, r] = eps
            fd[i, r] = (ro.silhouette_loss_and_grad(x + d, tris, cam, target)[0] - ro.silhouette_loss_and_grad(x - d, tris, cam, target)[0]) / (2 * eps)
    assert np.abs(g - fd).max() <= 1e-6 * np.abs(fd).max()
    # and L is what its definition says
    assert abs(L - ((ro.silhouette(x, tris, cam) - target) ** 2).mean()) <= 1e-18
