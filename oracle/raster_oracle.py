"""fp64 oracle of the soft silhouette rasteriser and its adjoint.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle.py): imported only by tests/, smoke() and bench.py's CPU leg.
Shares no code with paper_2104_02646_b200/csrc.

What it follows.  PAPER.md:168-172 (section 2.2): the renderers "replace discontinuous triangle mesh edges with smooth
sigmoids ... blurring triangle edges into semi-transparent boundaries".  The paper prints no formula; reading A22 takes the
SoftRas silhouette as SPEC.md:251 states it:
    per pixel p and triangle j:  D_j(p) = sigmoid(delta_j(p) d^2(p, boundary of triangle j) / sigma)
                                 delta = +1 inside, -1 outside, d = Euclidean distance in NDC
    silhouette                   S(p) = 1 - prod_j (1 - D_j(p))
    loss ("pixelwise MSE")   L = mean_p (S(p) - S*(p))^2
Camera: pinhole, p_cam = R x + t, visible iff z_cam > near, NDC (u, v) = (fx X / Z, fy Y / Z); pixel (i, j) of
a W x H image has its centre at u = 2 (i + 1/2) / W - 1, v = 2 (j + 1/2) / H - 1.  A triangle with a vertex at z_cam <=
near is not drawn.  Plain loops over triangles, numpy over pixels.
"""
from __future__ import annotations

import numpy as np


class Camera:
    def __init__(self, R, t, fx, fy, width, height, sigma, near=1e-3):
        self.R, self.t = np.asarray(R, np.float64).reshape(3, 3), np.asarray(t, np.float64).reshape(3)
        self.fx, self.fy, self.W, self.H, self.sigma, self.near = float(fx), float(fy), int(width), int(height), float(sigma), float(near)


def project(x, cam):
    """x [N,3] -> (ndc [N,2], z [N])"""
    pc = x @ cam.R.T + cam.t
    z = pc[:, 2]
    zs = np.where(z > cam.near, z, 1.0)
    return np.stack([cam.fx * pc[:, 0] / zs, cam.fy * pc[:, 1] / zs], 1), z


def pixel_centres(cam):
    u = 2.0 * (np.arange(cam.W) + 0.5) / cam.W - 1.0
    v = 2.0 * (np.arange(cam.H) + 0.5) / cam.H - 1.0
    return np.meshgrid(u, v)  # [H,W] each


def _seg(pu, pv, a, b):
    """squared distance of every pixel to segment ab, the closest-point parameter t and the offset p - c"""
    ab = b - a
    den = ab @ ab
    t = np.zeros_like(pu) if den == 0.0 else np.clip(((pu - a[0]) * ab[0] + (pv - a[1]) * ab[1]) / den, 0.0, 1.0)
    du, dv = pu - (a[0] + t * ab[0]), pv - (a[1] + t * ab[1])
    return du * du + dv * dv, t, du, dv


def _tri_terms(pu, pv, q):
    """q [3,2] NDC vertices -> (signed squared distance s = delta d^2, index of the closest edge, t, du, dv of that edge)"""
    d2 = [None] * 3
    for k in range(3):
        d2[k] = _seg(pu, pv, q[k], q[(k + 1) % 3])
    best = np.argmin(np.stack([d[0] for d in d2]), 0)
    pick = lambda i: np.choose(best, [d2[0][i], d2[1][i], d2[2][i]])
    dd, t, du, dv = pick(0), pick(1), pick(2), pick(3)
    e = [(q[(k + 1) % 3][0] - q[k][0]) * (pv - q[k][1]) - (q[(k + 1) % 3][1] - q[k][1]) * (pu - q[k][0]) for k in range(3)]
    inside = ((e[0] > 0) & (e[1] > 0) & (e[2] > 0)) | ((e[0] < 0) & (e[1] < 0) & (e[2] < 0))
    return np.where(inside, dd, -dd), best, t, du, dv


def _sigmoid(a):
    return 0.5 * (1.0 + np.tanh(0.5 * a))


def silhouette(x, tris, cam):
    ndc, z = project(np.asarray(x, np.float64), cam)
    pu, pv = pixel_centres(cam)
    keep = np.ones_like(pu)
    for tr in np.asarray(tris):
        if (z[tr] <= cam.near).any():
            continue
        s, *_ = _tri_terms(pu, pv, ndc[tr])
        keep = keep * (1.0 - _sigmoid(s / cam.sigma))
    return 1.0 - keep


def silhouette_loss_and_grad(x, tris, cam, target):
    """L = mean_p (S - S*)^2 and dL/dx [N,3], the chain rule written out by hand:
       dL/dS = 2 (S - S*) / (W H);  dS/dD_j = prod_{i != j} (1 - D_i);  dD/ds = D (1 - D) / sigma;
       ds/d(endpoints of the closest edge a, b) = delta (-2 (1 - t) (p - c), -2 t (p - c)), c = a + t (b - a);
       d(u, v)/d(p_cam) = [[fx / Z, 0, -fx X / Z^2], [0, fy / Z, -fy Y / Z^2]];  dp_cam/dx = R."""
    x = np.asarray(x, np.float64)
    tris = np.asarray(tris)
    ndc, z = project(x, cam)
    pu, pv = pixel_centres(cam)
    drawn = [j for j, tr in enumerate(tris) if not (z[tr] <= cam.near).any()]
    terms = [_tri_terms(pu, pv, ndc[tris[j]]) for j in drawn]
    one_minus = [1.0 - _sigmoid(tm[0] / cam.sigma) for tm in terms]
    # prod over the OTHER triangles by prefix and suffix products (no division by 1 - D, which may underflow)
    pre = [np.ones_like(pu)]
    for om in one_minus:
        pre.append(pre[-1] * om)
    suf = [np.ones_like(pu)]
    for om in reversed(one_minus):
        suf.append(suf[-1] * om)
    suf = suf[::-1]
    S = 1.0 - pre[-1]
    L = ((S - target) ** 2).mean()
    gS = 2.0 * (S - target) / S.size
    g_ndc = np.zeros_like(ndc)
    for n_, j in enumerate(drawn):
        tr = tris[j]
        s_, best, t, du, dv = terms[n_]
        D = 1.0 - one_minus[n_]
        others = pre[n_] * suf[n_ + 1]
        gs = gS * others * D * (1.0 - D) / cam.sigma  # dL/ds per pixel
        sign = np.where(s_ >= 0, 1.0, -1.0)
        for k in range(3):
            m = best == k
            wa, wb = -2.0 * (1.0 - t) * sign * gs * m, -2.0 * t * sign * gs * m
            a, b = tr[k], tr[(k + 1) % 3]
            g_ndc[a] += [(wa * du).sum(), (wa * dv).sum()]
            g_ndc[b] += [(wb * du).sum(), (wb * dv).sum()]
    pc = x @ cam.R.T + cam.t
    gx = np.zeros_like(x)
    for i in range(x.shape[0]):
        X, Y, Z = pc[i]
        if Z <= cam.near:
            continue
        gpc = np.array([g_ndc[i, 0] * cam.fx / Z, g_ndc[i, 1] * cam.fy / Z, -(g_ndc[i, 0] * cam.fx * X + g_ndc[i, 1] * cam.fy * Y) / (Z * Z)])
        gx[i] = cam.R.T @ gpc
    return L, gx


def hard_silhouette(x, tris, cam):
    """reference of the sigma -> 0 limit: plain point-in-triangle test at the pixel centres (SPEC.md:251 example)"""
    ndc, z = project(np.asarray(x, np.float64), cam)
    pu, pv = pixel_centres(cam)
    out = np.zeros_like(pu, dtype=bool)
    for tr in np.asarray(tris):
        if (z[tr] <= cam.near).any():
            continue
        s, *_ = _tri_terms(pu, pv, ndc[tr])
        out |= s > 0
    return out
