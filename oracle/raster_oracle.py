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


# ------------------------------------------------------------------------------------------ colour channel (reading A22b)
# "color = depth-softmax aggregation over triangles with weights proportional to D_j exp(zbar_j / gamma) plus a
# background term, normalized (SoftRas-style); per-triangle color from barycentric interpolation of shaded vertex colors,
# barycentrics clamped for exterior pixels".  The paper prints none of it ("only colour" shading);
# reading A22b fixes what SPEC.md leaves open:
#   lam_k(p)   screen-space (NDC) barycentric coordinates of pixel centre p in triangle j, k = 0, 1, 2
#   w_k        = clip(lam_k, 0, 1) / sum_i clip(lam_i, 0, 1)                       ("clamped for exterior pixels")
#   z_j(p)     = sum_k w_k Z_k (camera depths),  zbar_j = (far - z_j) / (far - near)  (nearer = larger)
#   C_j(p)     = sum_k w_k c_k  (vertex colours c_k in R^3: the "only colour" shading of PAPER.md:495, no lighting)
#   I(p)       = (sum_j D_j e^{zbar_j / gamma} C_j + e^{eps / gamma} C_b) / (sum_j D_j e^{zbar_j / gamma} + e^{eps / gamma})
# the sums over the drawn triangles that are not slivers (|2 area| > 1e-5 x the squared longest edge, in NDC: a collinear
# triangle has no barycentrics, and the threshold sits where fp32 and fp64 still agree on which side a triangle is) whose
# signed squared distance s_j(p) >= -40 sigma (beyond that
# D_j < e^-40; the cut is part of the definition, as SoftRas's distance threshold is).  Loss: pixelwise MSE over the three
# channels, L = mean_{p, c} (I_c(p) - I*_c(p))^2.
K_CULL = 40.0
SLIVER = 1e-5


class Shading:
    def __init__(self, gamma, eps, far, background):
        self.gamma, self.eps, self.far = float(gamma), float(eps), float(far)
        self.background = np.asarray(background, np.float64).reshape(3)


def _edge_functions(pu, pv, q):
    """e_k(p) = cross(q_{k+1} - q_k, p - q_k): twice the signed area of (q_k, q_{k+1}, p); their sum is twice the triangle's"""
    return [(q[(k + 1) % 3][0] - q[k][0]) * (pv - q[k][1]) - (q[(k + 1) % 3][1] - q[k][1]) * (pu - q[k][0]) for k in range(3)]


def _bary(pu, pv, q):
    """raw barycentrics lam [3][H,W] (lam_k is the weight of vertex k: the area opposite to it) and twice the signed area"""
    e = _edge_functions(pu, pv, q)
    A2 = e[0] + e[1] + e[2]  # constant over the image
    return [e[1] / A2, e[2] / A2, e[0] / A2], A2


def _rgb_terms(x, tris, cam, sh):
    """per contributing triangle: everything the image and its adjoint need"""
    ndc, z = project(x, cam)
    pu, pv = pixel_centres(cam)
    out = []
    for j, tr in enumerate(np.asarray(tris)):
        if (z[tr] <= cam.near).any():
            continue
        q = ndc[tr]
        A2c = (q[1][0] - q[0][0]) * (q[2][1] - q[0][1]) - (q[1][1] - q[0][1]) * (q[2][0] - q[0][0])
        if abs(A2c) <= SLIVER * max(((q[(k + 1) % 3] - q[k]) ** 2).sum() for k in range(3)):
            continue
        s, best, t, du, dv = _tri_terms(pu, pv, q)
        on = s >= -K_CULL * cam.sigma
        lam, A2 = _bary(pu, pv, q)
        u = [np.clip(l, 0.0, 1.0) for l in lam]
        su = u[0] + u[1] + u[2]
        w = [uk / su for uk in u]
        zj = w[0] * z[tr[0]] + w[1] * z[tr[1]] + w[2] * z[tr[2]]
        zbar = (sh.far - zj) / (sh.far - cam.near)
        a = s / cam.sigma
        logD = -np.logaddexp(0.0, -a)
        logit = np.where(on, logD + zbar / sh.gamma, -np.inf)
        out.append(dict(j=j, tr=tr, q=q, s=s, best=best, t=t, du=du, dv=dv, on=on, lam=lam, A2=A2, su=su, w=w, zbar=zbar, D=_sigmoid(a), logit=logit))
    return out, ndc, z, pu, pv


def rgb(x, tris, colours, cam, sh):
    """image [3][H][W]"""
    x, colours = np.asarray(x, np.float64), np.asarray(colours, np.float64)
    terms, ndc, z, pu, pv = _rgb_terms(x, tris, cam, sh)
    m = np.full_like(pu, sh.eps / sh.gamma)
    for tm in terms:
        m = np.maximum(m, tm["logit"])
    ab = np.exp(sh.eps / sh.gamma - m)
    den = ab.copy()
    num = [ab * sh.background[c] for c in range(3)]
    for tm in terms:
        aj = np.exp(tm["logit"] - m)
        den += aj
        for c in range(3):
            Cj = sum(tm["w"][k] * colours[tm["tr"][k], c] for k in range(3))
            num[c] = num[c] + aj * Cj
    return np.stack([n / den for n in num])


def rgb_loss_and_grads(x, tris, colours, cam, sh, target):
    """L = mean (I - I*)^2 over pixels and channels; returns (L, dL/dx [N,3], dL/dcolours [N,3]).  Chain rule by hand:
       W = sum_j a_j + a_b, a_j = D_j e^{zbar_j / gamma}:  dI_c/da_j = (C_jc - I_c) / W,  dI_c/dC_jc = a_j / W;
       da_j/ds_j = a_j (1 - D_j) / sigma  (s_j through the closest edge, as in the silhouette);
       da_j/dzbar_j = a_j / gamma,  zbar = (far - sum_k w_k Z_k) / (far - near);
       w = u / sum u, u_k = clip(lam_k, 0, 1) (derivative 1 strictly inside (0, 1), else 0);
       lam = (e_1, e_2, e_0) / (e_0 + e_1 + e_2), e_k = cross(q_{k+1} - q_k, p - q_k);
       then d(u, v, Z)/dx through the projection."""
    x, colours = np.asarray(x, np.float64), np.asarray(colours, np.float64)
    tris = np.asarray(tris)
    terms, ndc, z, pu, pv = _rgb_terms(x, tris, cam, sh)
    m = np.full_like(pu, sh.eps / sh.gamma)
    for tm in terms:
        m = np.maximum(m, tm["logit"])
    ab = np.exp(sh.eps / sh.gamma - m)
    Wt = ab.copy()
    num = [ab * sh.background[c] for c in range(3)]
    for tm in terms:
        tm["a"] = np.exp(tm["logit"] - m)
        tm["C"] = [sum(tm["w"][k] * colours[tm["tr"][k], c] for k in range(3)) for c in range(3)]
        Wt += tm["a"]
        for c in range(3):
            num[c] = num[c] + tm["a"] * tm["C"][c]
    I = np.stack([n / Wt for n in num])
    L = ((I - target) ** 2).mean()
    gI = 2.0 * (I - target) / I.size
    g_ndc, g_z, g_col = np.zeros_like(ndc), np.zeros_like(z), np.zeros_like(colours)
    for tm in terms:
        tr, a, w, q = tm["tr"], tm["a"], tm["w"], tm["q"]
        g_a = sum(gI[c] * (tm["C"][c] - I[c]) for c in range(3)) / Wt
        gC = [gI[c] * a / Wt for c in range(3)]
        # through the coverage: closest edge of the triangle
        gs = g_a * a * (1.0 - tm["D"]) / cam.sigma
        sign = np.where(tm["s"] >= 0, 1.0, -1.0)
        for k in range(3):
            mk = tm["best"] == k
            wa, wb = -2.0 * (1.0 - tm["t"]) * sign * gs * mk, -2.0 * tm["t"] * sign * gs * mk
            g_ndc[tr[k]] += [(wa * tm["du"]).sum(), (wa * tm["dv"]).sum()]
            g_ndc[tr[(k + 1) % 3]] += [(wb * tm["du"]).sum(), (wb * tm["dv"]).sum()]
        # through depth and colour: the clamped, renormalised barycentrics
        g_zj = -(g_a * a / sh.gamma) / (sh.far - cam.near)
        g_w = [g_zj * z[tr[k]] + sum(gC[c] * colours[tr[k], c] for c in range(3)) for k in range(3)]
        for k in range(3):
            g_z[tr[k]] += (g_zj * w[k]).sum()
            for c in range(3):
                g_col[tr[k], c] += (gC[c] * w[k]).sum()
        dot = g_w[0] * w[0] + g_w[1] * w[1] + g_w[2] * w[2]
        g_lam = [np.where((tm["lam"][k] > 0.0) & (tm["lam"][k] < 1.0), (g_w[k] - dot) / tm["su"], 0.0) for k in range(3)]
        g_A2 = -(g_lam[0] * tm["lam"][0] + g_lam[1] * tm["lam"][1] + g_lam[2] * tm["lam"][2]) / tm["A2"]
        # lam_0 = e_1 / A2, lam_1 = e_2 / A2, lam_2 = e_0 / A2;  A2 = e_0 + e_1 + e_2
        g_e = [g_lam[2] / tm["A2"] + g_A2, g_lam[0] / tm["A2"] + g_A2, g_lam[1] / tm["A2"] + g_A2]
        for k in range(3):
            qa, qb = q[k], q[(k + 1) % 3]
            # e_k = (qb_u - qa_u)(p_v - qa_v) - (qb_v - qa_v)(p_u - qa_u)
            g_ndc[tr[k]] += [(g_e[k] * (qb[1] - pv)).sum(), (g_e[k] * (pu - qb[0])).sum()]
            g_ndc[tr[(k + 1) % 3]] += [(g_e[k] * (pv - qa[1])).sum(), (g_e[k] * -(pu - qa[0])).sum()]
    pc = x @ cam.R.T + cam.t
    gx = np.zeros_like(x)
    for i in range(x.shape[0]):
        X, Y, Z = pc[i]
        if Z <= cam.near:
            continue
        gpc = np.array([g_ndc[i, 0] * cam.fx / Z, g_ndc[i, 1] * cam.fy / Z, -(g_ndc[i, 0] * cam.fx * X + g_ndc[i, 1] * cam.fy * Y) / (Z * Z) + g_z[i]])
        gx[i] = cam.R.T @ gpc
    return L, gx, g_col
