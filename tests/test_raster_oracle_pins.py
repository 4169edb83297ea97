"""Pins of the soft-silhouette oracle (oracle/raster_oracle.py; reading A22) against what
SPEC.md:240-251 and the mathematics fix.  No GPU."""
import numpy as np

from oracle import raster_oracle as ro
from paper_2104_02646_b200 import scenes


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


# ------------------------------------------------------------------------------------------ colour channel (reading A22b)
def _sh(gamma=0.05, eps=1e-3, far=10.0, bg=(0.1, 0.2, 0.3)):
    return ro.Shading(gamma, eps, far, bg)


def test_rgb_values_the_definition_fixes():
    """no triangles -> rgb = background; one fronto-parallel triangle of one colour: the two-term softmax in
    closed form, with D = 1 deep inside and D = 1/2 at a pixel centre on an edge; a triangle farther than the cut
    (s < -40 sigma) leaves the pixel at the background exactly."""
    cam = _cam(W=4, H=4, sigma=1e-4)
    sh = _sh()
    bg = sh.background
    x = np.array([[-20.0, -10.0, 0.0], [20.0, -10.0, 0.0], [0.0, 30.0, 0.0]])
    col = np.tile([0.9, 0.5, 0.2], (3, 1))
    I0 = ro.rgb(x, np.zeros((0, 3), int), col, cam, sh)
    assert all(np.all(I0[c] == bg[c]) for c in range(3))
    zbar = (sh.far - 5.0) / (sh.far - cam.near)
    a, b = np.exp(zbar / sh.gamma), np.exp(sh.eps / sh.gamma)
    I = ro.rgb(x, [[0, 1, 2]], col, cam, sh)
    for c in range(3):
        assert np.allclose(I[c], (a * col[0, c] + b * bg[c]) / (a + b), rtol=1e-12)
    xe = np.array([[-10.0, -1.25, 0.0], [10.0, -1.25, 0.0], [0.0, 10.0, 0.0]])  # edge through the centre of pixel (i=2, j=1)
    Ie = ro.rgb(xe, [[0, 1, 2]], col, _cam(W=4, H=4, sigma=1e-2), sh)
    for c in range(3):
        assert abs(Ie[c, 1, 2] - (0.5 * a * col[0, c] + b * bg[c]) / (0.5 * a + b)) < 1e-12
    # the row below the edge is 0.5 NDC away: s = -0.25 < -40 * 1e-4 -> not in the sum at all
    If = ro.rgb(xe, [[0, 1, 2]], col, cam, sh)
    assert all(np.all(If[c, 0, :] == bg[c]) for c in range(3))


def test_rgb_barycentric_interpolation_and_clamping():
    """With the background weight at zero (eps / gamma = -inf in effect) one triangle's pixel is its own C_j: an affine
    colour field over the vertices is reproduced at every interior pixel (wrong vertex / weight pairing fails), any vertex
    order gives the same image, and an exterior pixel beyond the edge opposite vertex k gets none of vertex k's colour."""
    cam = _cam(W=16, H=12, sigma=5e-2)
    sh = _sh(eps=-1e4)
    x = np.array([[-3.5, -3.0, 0.3], [4.0, -2.0, -0.2], [0.5, 3.5, 0.1]])
    ndc, _ = ro.project(x, cam)
    A, b0 = np.array([[0.3, -0.2], [0.1, 0.4], [-0.25, 0.15]]), np.array([0.5, 0.4, 0.6])
    col = ndc @ A.T + b0
    I = ro.rgb(x, [[0, 1, 2]], col, cam, sh)
    pu, pv = ro.pixel_centres(cam)
    inside = ro.hard_silhouette(x, [[0, 1, 2]], cam)
    assert inside.sum() > 20
    for c in range(3):
        assert np.allclose(I[c][inside], (A[c, 0] * pu + A[c, 1] * pv + b0[c])[inside], atol=1e-12)
    for perm in ([1, 2, 0], [2, 1, 0]):
        assert np.allclose(ro.rgb(x, [perm], col, cam, sh), I, atol=1e-13)
    rgbc = np.eye(3)
    Ic = ro.rgb(x, [[0, 1, 2]], rgbc, cam, sh)
    lam, _ = ro._bary(pu, pv, ndc)
    for k in range(3):
        beyond = lam[k] < 0
        assert beyond.any() and np.all(Ic[k][beyond] == 0.0)
    assert np.allclose(Ic.sum(0), 1.0, atol=1e-13)  # the clamped weights are renormalised


def test_rgb_depth_softmax_limits():
    """Two fronto-parallel triangles over the same pixels: gamma -> 0 shows the nearer one, gamma -> infinity the plain mean
    of the two and the background (all D = 1); the image is a convex combination of the colours throughout."""
    cam = _cam(W=6, H=6, sigma=1e-6)
    x = np.array([[-20.0, -10.0, 0.0], [20.0, -10.0, 0.0], [0.0, 30.0, 0.0], [-20.0, -10.0, 1.0], [20.0, -10.0, 1.0], [0.0, 30.0, 1.0]])
    col = np.array([[1.0, 0.0, 0.0]] * 3 + [[0.0, 1.0, 0.0]] * 3)
    tris = [[3, 4, 5], [0, 1, 2]]
    near = ro.rgb(x, tris, col, cam, _sh(gamma=1e-4))
    assert np.allclose(near[0], 1.0, atol=1e-12) and np.allclose(near[1], 0.0, atol=1e-12)
    flat = ro.rgb(x, tris, col, cam, _sh(gamma=1e9))
    for c, want in enumerate([(1.0 + 0.1) / 3, (1.0 + 0.2) / 3, 0.3 / 3]):
        assert np.allclose(flat[c], want, atol=1e-8)
    mid = ro.rgb(x, tris, col, cam, _sh(gamma=0.05))
    zb = [(10.0 - 5.0) / (10.0 - cam.near), (10.0 - 6.0) / (10.0 - cam.near)]
    wts = np.array([np.exp(zb[0] / 0.05), np.exp(zb[1] / 0.05), np.exp(1e-3 / 0.05)])
    for c, cols in enumerate([(1.0, 0.0, 0.1), (0.0, 1.0, 0.2), (0.0, 0.0, 0.3)]):  # (near, far, background) per channel
        assert np.allclose(mid[c], (wts * np.array(cols)).sum() / wts.sum(), rtol=1e-12)
    rng = np.random.default_rng(11)
    xr = np.concatenate([rng.uniform(-3, 3, (12, 2)), rng.uniform(-0.5, 0.5, (12, 1))], 1)
    cr = rng.uniform(0.2, 0.9, (12, 3))
    Ir = ro.rgb(xr, [[0, 1, 2], [3, 4, 5], [6, 7, 8], [9, 10, 11]], cr, _cam(sigma=3e-3), _sh())
    assert Ir.min() >= 0.1 - 1e-12 and Ir.max() <= 0.9 + 1e-12


def test_rgb_loss_gradients_vs_fd():
    """dL/dx and dL/dcolours of the pixelwise RGB MSE (hand-written chain rule through coverage, depth softmax and the
    clamped barycentrics) against central differences: rotated off-axis camera (vertex depths differ), overlapping
    triangles, many exterior pixels inside the 40 sigma cut."""
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(-2.5, 2.5, (9, 2)), rng.uniform(-0.4, 0.4, (9, 1))], 1)
    tris = np.array([[0, 1, 2], [2, 3, 4], [4, 5, 6], [6, 7, 8], [1, 5, 8]])
    th = 0.3
    R = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]]) @ np.array([[1, 0, 0], [0, np.cos(0.2), -np.sin(0.2)], [0, np.sin(0.2), np.cos(0.2)]])
    cam = ro.Camera(R, (0.2, -0.1, 6.0), 1.7, 1.9, 40, 30, 2e-2)
    sh = _sh()
    col = rng.uniform(0, 1, (9, 3))
    target = ro.rgb(x + 0.15 * rng.normal(size=x.shape), tris, rng.uniform(0, 1, (9, 3)), cam, sh)
    L, gx, gc = ro.rgb_loss_and_grads(x, tris, col, cam, sh, target)
    assert abs(L - ((ro.rgb(x, tris, col, cam, sh) - target) ** 2).mean()) <= 1e-18
    f = lambda xx, cc: ro.rgb_loss_and_grads(xx, tris, cc, cam, sh, target)[0]
    eps = 1e-6
    fdx, fdc = np.zeros_like(x), np.zeros_like(col)
    for i in range(9):
        for r in range(3):
            d = np.zeros_like(x); d[i, r] = eps
            fdx[i, r] = (f(x + d, col) - f(x - d, col)) / (2 * eps)
            fdc[i, r] = (f(x, col + d) - f(x, col - d)) / (2 * eps)
    assert np.abs(gx).max() > 0 and np.abs(gx - fdx).max() <= 1e-6 * np.abs(fdx).max()
    assert np.abs(gc).max() > 0 and np.abs(gc - fdc).max() <= 1e-6 * np.abs(fdc).max()
    # depth matters: the gradient with respect to a pure camera-depth shift of one triangle is not zero
    assert np.abs(gx @ R[2]).max() > 1e-6


def test_rgb_slivers_and_hidden_triangles_are_skipped():
    """A collinear triangle (no barycentrics) and one with a vertex behind the near plane add nothing to the colour image."""
    cam = _cam(W=12, H=10, sigma=1e-2)
    x = np.array([[-2.0, -1.5, 0.0], [2.0, -1.0, 0.2], [0.0, 2.0, -0.1], [1.0, -1.25, 0.1], [0.3, 0.2, -9.0]])
    col = np.random.default_rng(2).uniform(0, 1, (5, 3))
    base = ro.rgb(x, [[0, 1, 2]], col, cam, _sh())
    assert np.abs(base - _sh().background[:, None, None]).max() > 0.1
    x[3] = 0.25 * x[0] + 0.75 * x[1]  # on the segment 0-1, hence collinear in the image too
    assert np.array_equal(ro.rgb(x, [[0, 1, 2], [0, 3, 1], [0, 1, 4]], col, cam, _sh()), base)


def test_boundary_faces_of_a_tet_mesh_and_its_silhouette():
    """scenes.boundary_faces (topology only): one tet -> its four faces; the 4 x 4 x 4-cell box -> 6 x 16 x 2 = 192 triangles
    forming a closed surface (every edge in exactly two faces), all on the box's boundary; and the silhouette drawn from them is
    that of ALL tet faces (interior faces project inside the outline: same hard silhouette as sigma -> 0)."""
    assert sorted(map(sorted, scenes.boundary_faces(np.array([[0, 1, 2, 3]])).tolist())) == [[0, 1, 2], [0, 1, 3], [0, 2, 3], [1, 2, 3]]
    sc = scenes.make_scene(0, small=True)
    f = scenes.boundary_faces(sc.tets)
    assert f.shape == (192, 3)
    edges = {}
    for t in f.tolist():
        for a, b in ((t[0], t[1]), (t[1], t[2]), (t[2], t[0])):
            edges[tuple(sorted((a, b)))] = edges.get(tuple(sorted((a, b))), 0) + 1
    assert set(edges.values()) == {2}
    x = sc.x_rest.astype(np.float64)
    lo, hi = x.min(0), x.max(0)
    on_boundary = (np.isclose(x, lo) | np.isclose(x, hi)).any(1)
    assert on_boundary[f].all() and not on_boundary.all()
    all_faces = np.array([[t[i] for i in idx] for t in sc.tets.tolist() for idx in ((1, 2, 3), (0, 3, 2), (0, 1, 3), (0, 2, 1))])
    th = 0.5
    R = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]])
    cam = ro.Camera(R, -R @ x.mean(0) + np.array([0.0, 0.0, 1.5]), 2.0, 2.0, 40, 40, 1e-7)
    assert np.array_equal(ro.hard_silhouette(x, f, cam), ro.hard_silhouette(x, all_faces, cam))
    assert 0.1 < ro.hard_silhouette(x, f, cam).mean() < 0.9
