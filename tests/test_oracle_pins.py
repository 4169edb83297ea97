"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU).

P1 Listing 1 / free fall      P2 zero force at rest + rigid rotations    P3 f = -grad U (central FD)
P4 momentum                   P5 invariance / equivariance               P6 contact values
P7 step Jacobian^T vs FD      P8 rollout adjoint vs FD <= 1e-5           P9 checkpoint == full tape bit-for-bit
P10 damping dissipates        + rest quantities, small-strain linearisation, linearity in the cotangent
Chosen so that a dropped term, a wrong sign/index or a transposed operand fails at least one.
"""
import os

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2104_02646_b200 import scenes



GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        out[k] = np.array([float(t) for t in v])
    return out


def _rot(rng):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q *= np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def _free(sc):
    """no gravity, contact plane far away, no air"""
    sc.gravity = (0.0, 0.0, 0.0)
    sc.plane_d = -1e6
    sc.k_drag, sc.k_lift = 0 * sc.k_drag, 0 * sc.k_lift
    return sc


def _mixed_scene(rng, **kw):
    """small mixed mesh: 1 hex cell (5 tets) + a 3x3 cloth patch (8 triangles, 8 hinges)."""
    xs, tets = scenes.hex_grid_tets(1, 1, 1, 0.1, origin=(0.0, 0.05, 0.0))
    xc, tris, hinges = scenes.cloth_grid(3, 3, 0.05, origin=(0.3, 0.03, 0.0))
    x = np.concatenate([xs, xc])
    n0 = xs.shape[0]
    M, Mt = tets.shape[0], tris.shape[0]
    args = dict(
        mass=rng.uniform(0.05, 0.2, x.shape[0]), mu=rng.uniform(5e3, 2e4, M), lam=rng.uniform(5e3, 2e4, M),
        damp=rng.uniform(0.5, 2.0, M), tri_mu=rng.uniform(5e2, 2e3, Mt), tri_lam=rng.uniform(5e2, 2e3, Mt),
        tri_damp=rng.uniform(0.5, 2.0, Mt), kb=rng.uniform(5, 20, hinges.shape[0]),
        k_drag=0.3, k_lift=0.2, wind=(0.5, -0.2, 0.3),  # lift / drag of the air on the cloth patch (reading A21)
    )
    args.update(kw)
    return scenes.custom_scene(x, tets=tets, tris=tris + n0, hinges=hinges + n0, **args)


SCALAR_GROUPS = ("ke", "kd", "kf", "mu_c", "k_drag", "k_lift")  # one value per environment
ABS_STEP = ("gravity", "hinge_theta0")       # parameters whose value may be 0: absolute FD steps


def _param(sc, o, g):
    """(analytic gradient, base value) of parameter group g as flat fp64 arrays of equal shape."""
    if g == "gravity":  # one vector shared by all environments; the oracle keeps dL/dg per environment
        return o.grads(g).sum(0).copy(), np.asarray(sc.gravity, np.float64)
    if g == "hinge_theta0":  # rest angles (derived from x_rest; one array shared by all environments)
        return o.grads(g).sum(0).copy(), o.rest()["theta0"].copy()
    scalar = g in SCALAR_GROUPS
    an = (o.grads(g)[:, 0] if scalar else o.grads(g)[0]).copy()
    base = getattr(sc, g).astype(np.float64)
    return an, (base if g == "hinge_kb" or scalar else base[0])  # k_b is one array shared by all environments


# ---------------------------------------------------------------- P1 integrate
def test_p1_listing1_golden():
    g = _gold("listing1_integrate.txt")
    for pinned, kx, kv in ((0, "x1", "v1"), (1, "x1_pinned", "v1_pinned")):
        sc = scenes.custom_scene(g["x0"][None], mass=g["mass"][0], dt=g["dt"][0], ke=500.0, kd=0.0, kf=0.0, pinned=[pinned])
        o = orc.Oracle(sc)
        assert np.allclose(o.forces(g["x0"], g["v0"])[0, 0], g["f0"], atol=1e-12)
        x1, v1 = o.step(g["x0"], g["v0"])
        assert np.allclose(v1[0, 0], g[kv], atol=1e-12)
        assert np.allclose(x1[0, 0], g[kx], atol=1e-12)


def test_p1_free_fall_closed_form_and_adjoint():
    T, dt = 50, 1.0 / 1920.0
    x0 = np.array([[0.3, 5.0, -0.2], [1.0, 7.0, 2.0]])
    v0 = np.array([[0.1, 0.4, -0.3], [0.0, -0.2, 0.5]])
    sc = scenes.custom_scene(x0, v0=v0, dt=dt, pinned=[0, 1])
    o = orc.Oracle(sc)
    ro = o.rollout(sc.x0, sc.v0, T)
    g = np.array(sc.gravity)
    x0f, v0f = sc.x0.astype(np.float64)[0], sc.v0.astype(np.float64)[0]
    # x_T = x0 + v0 T dt + g dt^2 T(T+1)/2 for the free particle; pinned: x0 + v0 T dt, v unchanged
    assert np.allclose(ro["xT"][0, 0], x0f[0] + v0f[0] * T * dt + g * dt * dt * T * (T + 1) / 2, atol=1e-13)
    assert np.allclose(ro["xT"][0, 1], x0f[1] + v0f[1] * T * dt, atol=1e-13)
    assert np.allclose(ro["vT"][0, 1], v0f[1], atol=0)
    # d(final height)/d(initial vertical velocity) = T dt exactly
    cot = np.zeros((1, 1, 2, 3)); cot[0, 0, 0, 1] = 1.0
    ax0, av0 = o.rollout_backward(ro, [T], cot)
    assert abs(av0[0, 0, 1] - T * dt) < 1e-15 and abs(ax0[0, 0, 1] - 1.0) < 1e-15
    assert np.all(o.grads("mass") == 0)  # free fall does not depend on mass (A11)
    # dL/dg (Table 5): from the closed form, d(x_T,y of the free particle)/dg_y = dt^2 T (T+1)/2; the
    # pinned particle ignores gravity; the other components of the cotangent are zero
    gg = o.grads("gravity")[0]
    assert abs(gg[1] - dt * dt * T * (T + 1) / 2) < 1e-15 and gg[0] == 0 and gg[2] == 0
    # with a cotangent on the final VELOCITY of the free particle: d(v_T)/dg = T dt
    o.zero_grads()
    avT = np.zeros((1, 2, 3)); avT[0, 0, 2] = 1.0; avT[0, 1, 2] = 5.0
    o.rollout_backward(ro, [T], 0 * cot, adj_vT=avT)
    assert np.allclose(o.grads("gravity")[0], [0.0, 0.0, T * dt], atol=1e-15)


# ---------------------------------------------------------------- rest quantities
def test_rest_quantities():
    sc = scenes.box_scene(cells=(3, 2, 4), h=0.1)
    r = orc.Oracle(sc).rest()
    assert abs(r["tet_V"].sum() - 0.3 * 0.2 * 0.4) < 1e-6 * 0.024  # 5-tet split fills the box (A12)
    assert r["tet_V"].min() > 0.1**3 / 6 * (1 - 1e-5)
    cs = scenes.cloth_scene(n=7, h=0.02)
    rc = orc.Oracle(cs).rest()
    assert abs(rc["tri_A"].sum() - (6 * 0.02) ** 2) < 1e-6 * 0.0144  # inputs are fp32-rounded (A19)
    assert np.allclose(rc["theta0"], 0.0, atol=1e-6)  # flat sheet (A5/A13)
    assert set(np.round(rc["l0"] / 0.02, 4)) <= {1.0, round(np.sqrt(2), 4)}
    # B is the inverse of the rest edge matrix: F(rest) = I
    x = cs.x_rest.astype(np.float64)
    for e in (0, 5, 11):
        t = cs.tris[e]
        e1, e2 = x[t[1]] - x[t[0]], x[t[2]] - x[t[0]]
        F = np.stack([e1, e2], 1) @ rc["tri_B"][e]
        assert np.allclose(F.T @ F, np.eye(2), atol=1e-6)


def test_invalid_mesh_rejected():
    x = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1.0]])
    with pytest.raises(ValueError):
        orc.Oracle(scenes.custom_scene(x, tets=[[0, 2, 1, 3]]))  # inverted
    with pytest.raises(ValueError):
        orc.Oracle(scenes.custom_scene(x, tets=[[0, 1, 2, 7]]))  # index out of range


# ---------------------------------------------------------------- P2 rest + rotations
def test_p2_zero_force_at_rest_and_rigid_rotations():
    rng = np.random.default_rng(2)
    sc = _free(_mixed_scene(rng, damp=0.0, tri_damp=0.0))
    o = orc.Oracle(sc)
    x = sc.x_rest.astype(np.float64)
    scale = 1e4 * 0.1**2  # mu * h^2: natural force scale
    for mask in (orc.TETS, orc.TRIS, orc.HINGES):
        assert np.abs(o.forces(x, mask=mask)).max() < 1e-9 * scale
    for _ in range(5):
        R, t = _rot(rng), rng.normal(size=3)
        xr = x @ R.T + t
        for mask in (orc.TETS, orc.TRIS, orc.HINGES):
            assert np.abs(o.forces(xr, mask=mask)).max() < 1e-9 * scale
    # A1 closed form: with SPEC's alpha = 1 + mu/lambda the rest stress would be -mu/4 != 0; ours is 0 for any mu, lambda


# ---------------------------------------------------------------- P3 f = -grad U
@pytest.mark.parametrize("mask", [orc.TETS, orc.TRIS, orc.HINGES])
def test_p3_force_is_minus_energy_gradient(mask):
    rng = np.random.default_rng(3)
    sc = _free(_mixed_scene(rng))
    o = orc.Oracle(sc)
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (sc.n_particles, 3))
    f = o.forces(x, mask=mask)[0]  # v = 0: no damping force
    eps = 1e-6
    g = np.zeros_like(f)
    for i in range(x.shape[0]):
        for r in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, r] += eps; xm[i, r] -= eps
            g[i, r] = (o.energy(xp, mask)[0] - o.energy(xm, mask)[0]) / (2 * eps)
    assert np.abs(f).max() > 1e-3
    assert np.abs(f + g).max() <= 2e-7 * np.abs(f).max()


# ---------------------------------------------------------------- small-strain linearisation
def test_small_strain_matches_linear_elasticity():
    g = _gold("smith_linearisation.txt")
    mu, lam = 1.3e4, 2.1e4
    X = np.array([[0, 0, 0], [0.1, 0, 0], [0, 0.1, 0], [0, 0, 0.1]], dtype=np.float64)
    sc = _free(scenes.custom_scene(X, tets=[[0, 1, 2, 3]], mu=mu, lam=lam, damp=0.0))
    o = orc.Oracle(sc)
    rng = np.random.default_rng(4)
    a = rng.normal(size=(3, 3)); eps = 1e-7 * (a + a.T)
    x = sc.x_rest.astype(np.float64) @ (np.eye(3) + eps).T
    f = o.forces(x, mask=orc.TETS)[0]
    mu_l, lam_l = g["mu_lin_over_mu"][0] * mu, lam + g["lambda_lin_minus_lambda_over_mu"][0] * mu
    sigma = 2 * mu_l * eps + lam_l * np.trace(eps) * np.eye(3)
    Xd = sc.x_rest.astype(np.float64)
    Dm = (Xd[1:] - Xd[0]).T
    V = np.linalg.det(Dm) / 6
    H = -V * sigma @ np.linalg.inv(Dm).T
    fl = np.stack([-H.sum(1), H[:, 0], H[:, 1], H[:, 2]])
    assert np.abs(f - fl).max() <= 1e-5 * np.abs(fl).max()


# ---------------------------------------------------------------- P4 momentum, P5 invariance, P10 dissipation
def test_p4_internal_forces_have_zero_net_force_and_torque():
    rng = np.random.default_rng(5)
    sc = _free(_mixed_scene(rng))
    o = orc.Oracle(sc)
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (sc.n_particles, 3))
    v = rng.normal(size=x.shape)
    for mask in (orc.TETS, orc.TRIS, orc.HINGES):
        f = o.forces(x, v, mask=mask)[0]
        s = np.abs(f).max()
        assert s > 1e-3
        assert np.abs(f.sum(0)).max() < 1e-11 * s
        assert np.abs(np.cross(x, f).sum(0)).max() < 1e-11 * s


def test_p4_rollout_conserves_linear_and_angular_momentum():
    rng = np.random.default_rng(6)
    sc = _free(_mixed_scene(rng))
    o = orc.Oracle(sc)
    m = sc.mass.astype(np.float64)[0][:, None]
    x0 = sc.x_rest.astype(np.float64) + 0.005 * rng.uniform(-1, 1, (sc.n_particles, 3))
    v0 = 0.3 * rng.normal(size=x0.shape)
    ro = o.rollout(x0, v0, 200, rec_times=[0, 100, 200], want_rec_v=True)
    p = [(m * ro["rec_v"][k, 0]).sum(0) for k in range(3)]
    # semi-implicit Euler: L_{t+1} = sum m x_{t+1} x v_{t+1} = sum m (x_t + dt v+) x v+ = sum m x_t x v+, and
    # sum x_t x f_t = 0, so the discrete angular momentum is conserved exactly too
    Lm = [np.cross(ro["rec_x"][k, 0], m * ro["rec_v"][k, 0]).sum(0) for k in range(3)]
    for k in (1, 2):
        assert np.abs(p[k] - p[0]).max() < 1e-12 * np.abs(m * v0).sum()
        assert np.abs(Lm[k] - Lm[0]).max() < 1e-12 * np.abs(m * v0).sum()
    assert np.abs(ro["rec_x"][2] - ro["rec_x"][0]).max() > 1e-3  # something moved


def test_p5_translation_invariance_rotation_equivariance():
    rng = np.random.default_rng(7)
    sc = _free(_mixed_scene(rng))
    o = orc.Oracle(sc)
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (sc.n_particles, 3))
    v = rng.normal(size=x.shape)
    f = o.forces(x, v, mask=orc.TETS | orc.TRIS | orc.HINGES)[0]
    R, t = _rot(rng), rng.normal(size=3)
    f_t = o.forces(x + t, v + 0.7, mask=orc.TETS | orc.TRIS | orc.HINGES)[0]  # uniform velocity shift: no damping change
    f_r = o.forces(x @ R.T, v @ R.T, mask=orc.TETS | orc.TRIS | orc.HINGES)[0]
    s = np.abs(f).max()
    assert np.abs(f_t - f).max() < 1e-9 * s
    assert np.abs(f_r - f @ R.T).max() < 1e-9 * s


def test_p10_damping_dissipates_and_ignores_rigid_motion():
    rng = np.random.default_rng(8)
    sc = _free(_mixed_scene(rng))
    o = orc.Oracle(sc)
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (sc.n_particles, 3))
    for _ in range(5):
        v = rng.normal(size=x.shape)
        fd = o.forces(x, v, mask=orc.TETS | orc.TRIS)[0] - o.forces(x, 0 * v, mask=orc.TETS | orc.TRIS)[0]
        assert (fd * v).sum() < 0
    w = rng.normal(size=3)
    v_rigid = np.cross(w, x) + rng.normal(size=3)  # rigid spin + translation: zero strain rate (A3)
    fd = o.forces(x, v_rigid, mask=orc.TETS | orc.TRIS)[0] - o.forces(x, 0 * x, mask=orc.TETS | orc.TRIS)[0]
    assert np.abs(fd).max() < 1e-9 * np.abs(o.forces(x, mask=orc.TETS | orc.TRIS)).max()


# ---------------------------------------------------------------- P6 contact
def test_p6_contact_golden_values():
    for line in open(os.path.join(GOLD, "contact_spec.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        y, v, (ke, kd, kf, muc), exp = float(t[1]), [float(a) for a in t[2:5]], [float(a) for a in t[5:9]], [float(a) for a in t[9:12]]
        sc = scenes.custom_scene(np.array([[0.0, y, 0.0]]), ke=ke, kd=kd, kf=kf, mu_c=muc)
        f = orc.Oracle(sc).forces(sc.x0, np.array(v), mask=orc.CONTACT)[0, 0]
        assert np.allclose(f, exp, atol=1e-6), (t[0], f)  # 1e-6: y = -0.01 is fp32-rounded by the generator


def test_p6_contact_invariants():
    rng = np.random.default_rng(9)
    n = 400
    x = np.stack([rng.normal(size=n), rng.uniform(-0.02, 0.005, n), rng.normal(size=n)], 1)
    v = rng.normal(size=(n, 3)) * np.where(rng.random(n) < 0.5, 1e-3, 3.0)[:, None]
    sc = scenes.custom_scene(x, ke=1e4, kd=10.0, kf=50.0, mu_c=0.5)
    f = orc.Oracle(sc).forces(sc.x0, v, mask=orc.CONTACT)[0]
    xd = sc.x0.astype(np.float64)[0]
    fn, ft = f[:, 1], f[:, [0, 2]]
    assert np.all(fn >= 0)  # no adhesion (A7)
    assert np.all(f[xd[:, 1] >= 0] == 0)
    assert np.all(np.linalg.norm(ft, axis=1) <= 0.5 * fn * (1 + 1e-12) + 1e-15)  # Coulomb cone (A8)
    vt = v[:, [0, 2]]
    act = xd[:, 1] < 0
    assert np.all((ft * vt).sum(1)[act] <= 0)  # friction opposes sliding
    stick = act & (50.0 * np.linalg.norm(vt, axis=1) < 0.5 * fn)
    assert stick.sum() > 10 and (act & ~stick).sum() > 10  # both regimes exercised
    assert np.allclose(ft[stick], -50.0 * vt[stick], rtol=1e-12)


# ---------------------------------------------------------------- P7 one-substep Jacobian^T vs central FD
def _contact_state(sc, rng):
    x = sc.x_rest.astype(np.float64) + 0.004 * rng.uniform(-1, 1, (sc.n_particles, 3))
    x[:, 1] -= x[:, 1].min() + 0.004  # a few particles below the plane
    v = 0.2 * rng.normal(size=x.shape)
    below = np.where(x[:, 1] < 0)[0]
    v[below[::2]] *= 1e-3  # stick
    v[below[1::2], 0] += 2.0  # slip
    v[below[::3], 1] = -0.3  # approaching: damping branch
    return x, v, below


def test_p7_step_adjoint_is_transposed_jacobian():
    rng = np.random.default_rng(10)
    sc = _mixed_scene(rng, pinned=[0] * 16 + [1], dt=1.0 / 1920.0)
    o = orc.Oracle(sc)
    x, v, below = _contact_state(sc, rng)
    assert len(below) >= 3
    N = sc.n_particles
    bx, bv = rng.normal(size=(N, 3)), rng.normal(size=(N, 3))
    ax, av = o.step_adjoint(x, v, bx, bv)

    def phi(xx, vv):
        xo, vo = o.step(xx, vv)
        return (xo[0] * bx).sum() + (vo[0] * bv).sum()

    eps = 1e-7
    gx, gv = np.zeros((N, 3)), np.zeros((N, 3))
    for i in range(N):
        for r in range(3):
            d = np.zeros((N, 3)); d[i, r] = eps
            gx[i, r] = (phi(x + d, v) - phi(x - d, v)) / (2 * eps)
            gv[i, r] = (phi(x, v + d) - phi(x, v - d)) / (2 * eps)
    assert np.abs(ax[0] - gx).max() <= 1e-6 * np.abs(gx).max()
    assert np.abs(av[0] - gv).max() <= 1e-6 * np.abs(gv).max()


@pytest.mark.parametrize("group", list(orc.GROUPS))
def test_p7_step_param_gradients_vs_fd(group):
    rng = np.random.default_rng(11)
    sc = _mixed_scene(rng)
    o = orc.Oracle(sc)
    x, v, _ = _contact_state(sc, rng)
    N = sc.n_particles
    bx, bv = rng.normal(size=(N, 3)), rng.normal(size=(N, 3))
    o.zero_grads()
    o.step_adjoint(x, v, bx, bv)
    scalar = group in SCALAR_GROUPS
    g, base = _param(sc, o, group)
    fd = np.zeros_like(base)
    for e in range(base.size):
        # one substep is piecewise LINEAR in the contact parameters (within a friction regime), so their central
        # difference is exact for any step that keeps the regimes; a larger step keeps round-off out of the tiny
        # stick-friction terms
        # (the substep is also exactly affine in mu, lambda, k_damp, k_b -- the stress is linear in them -- so the larger
        # step is exact for those groups too and keeps round-off of the O(1) functional out of their small gradients)
        affine = scalar or group.startswith(("tet_", "tri_")) or group == "hinge_kb"
        h = (1e-3 if affine else 1e-6) * (base[e] if group not in ABS_STEP else 1.0)
        vals = []
        for s in (+1, -1):
            p = base.copy(); p[e] += s * h
            o.set_params(group, p)
            xo, vo = o.step(x, v)
            vals.append((xo[0] * bx).sum() + (vo[0] * bv).sum())
        fd[e] = (vals[0] - vals[1]) / (2 * h)
    o.set_params(group, base)
    assert np.abs(g).max() > 0
    assert np.abs(g - fd).max() <= 1e-6 * np.abs(fd).max()


@pytest.mark.parametrize("s", [0.8, 1.0, 1.25])
def test_uniform_stretch_closed_forms(s):
    """Closed forms of the elastic nodal forces under a uniform stretch x = s X (readings A1, A4).
    Corner tet with legs a: F = s I, I_C = 3 s^2, J = s^3, cof F = s^2 I, so P = p I with
    p = mu (1 - 1/(3 s^2 + 1)) s + (lambda (s^3 - 1) - 3 mu / 4) s^2 and H = -V P B^T = -(a^2 p / 6) I.
    Right triangle with legs a: F = s Q (Q the 3x2 rest frame), I_C = 2 s^2, J = s^2, dJ/dF = s Q, so P = p2 Q with
    p2 = s [mu (1 - 1/(2 s^2 + 1)) + lambda (s^2 - 1) - 2 mu / 3] and H = -A P B^T = -(a p2 / 2) Q.  Both vanish at s = 1."""
    a, mu, lam = 0.25, 1.25e4, 2.0e4  # exact in fp32 (inputs are rounded once, A19)
    X = np.array([[0, 0, 0], [a, 0, 0], [0, a, 0], [0, 0, a]], dtype=np.float64)
    sc = _free(scenes.custom_scene(X, tets=[[0, 1, 2, 3]], mu=mu, lam=lam, damp=0.0))
    f = orc.Oracle(sc).forces(s * X, mask=orc.TETS)[0]
    p = mu * (1 - 1 / (3 * s * s + 1)) * s + (lam * (s ** 3 - 1) - 0.75 * mu) * s * s
    want = np.vstack([np.full(3, a * a * p / 6), -a * a * p / 6 * np.eye(3)])
    assert np.abs(f - want).max() <= 1e-12 * max(abs(a * a * p / 6), 1.0)
    Xt = np.array([[0, 0, 0], [a, 0, 0], [0, 0, -a]], dtype=np.float64)  # legs along +x and -z: normal +y
    sc = _free(scenes.custom_scene(Xt, tris=[[0, 1, 2]], hinges=np.zeros((0, 4), np.int32), tri_mu=mu, tri_lam=lam, tri_damp=0.0))
    f = orc.Oracle(sc).forces(s * Xt, mask=orc.TRIS)[0]
    p2 = s * (mu * (1 - 1 / (2 * s * s + 1)) + lam * (s * s - 1) - 2 * mu / 3)
    f1, f2 = -(a * p2 / 2) * np.array([1.0, 0, 0]), -(a * p2 / 2) * np.array([0, 0, -1.0])
    want = np.vstack([-(f1 + f2), f1, f2])
    assert np.abs(f - want).max() <= 1e-12 * max(abs(a * p2 / 2), 1.0)


def test_uniform_expansion_rate_damping_closed_forms():
    """Damping force (reading A3: P_damp = k F sym(F^T Fdot)) for x = s X, v = r X: F = s I (or s Q), Fdot = r I (r Q),
    sym(F^T Fdot) = s r I, so P_damp = k s^2 r I: H = -(a^2 k s^2 r / 6) I for the corner tet, -(a k s^2 r / 2) Q for the
    right triangle; elastic part removed by differencing against v = 0."""
    a, mu, lam, k, s_, r = 0.25, 1.25e4, 2.0e4, 3.0, 1.125, 0.75
    X = np.array([[0, 0, 0], [a, 0, 0], [0, a, 0], [0, 0, a]], dtype=np.float64)
    o = orc.Oracle(_free(scenes.custom_scene(X, tets=[[0, 1, 2, 3]], mu=mu, lam=lam, damp=k)))
    fd = o.forces(s_ * X, v=r * X, mask=orc.TETS)[0] - o.forces(s_ * X, mask=orc.TETS)[0]
    c = a * a * k * s_ * s_ * r / 6
    assert np.abs(fd - np.vstack([np.full(3, c), -c * np.eye(3)])).max() <= 1e-10 * c  # difference of two O(1e3) forces
    Xt = np.array([[0, 0, 0], [a, 0, 0], [0, 0, -a]], dtype=np.float64)
    o = orc.Oracle(_free(scenes.custom_scene(Xt, tris=[[0, 1, 2]], hinges=np.zeros((0, 4), np.int32), tri_mu=mu, tri_lam=lam, tri_damp=k)))
    fd = o.forces(s_ * Xt, v=r * Xt, mask=orc.TRIS)[0] - o.forces(s_ * Xt, mask=orc.TRIS)[0]
    c = a * k * s_ * s_ * r / 2
    f1, f2 = -c * np.array([1.0, 0, 0]), -c * np.array([0, 0, -1.0])
    assert np.abs(fd - np.vstack([-(f1 + f2), f1, f2])).max() <= 1e-10 * c


@pytest.mark.parametrize("fold", [0.0, 0.3, -0.8, 2.0])
def test_hinge_force_closed_form_symmetric_fold(fold):
    """Worked example of PAPER.md:585-586 with readings A5, A6: a hinge whose edge (length L) lies on the z axis, both wings
    at distance h from it at mid-edge, rest shape flat, folded by the angle `fold`.  Then d_wing = n_hat / h (|n| = L h), so
    the wing forces have magnitude k_b L |sin(fold/2)| / h along their face normals, the edge vertices share the opposite
    force equally, and dL/dk_b of a substep is sum_i a_i.f_i / k_b (the force is linear in k_b)."""
    L, h, kb, dt, m = 0.5, 0.25, 7.0, 1.0 / 1920.0, 0.1  # L, h, k_b exact in fp32 (inputs are rounded once, A19)
    rest = np.array([[h, 0.0, L / 2], [-h, 0.0, L / 2], [0.0, 0.0, 0.0], [0.0, 0.0, L]])  # wing1, wing2, edge a, edge b
    sc = scenes.custom_scene(rest, tris=[[2, 3, 0], [3, 2, 1]], hinges=[[0, 1, 2, 3]], kb=kb, dt=dt, mass=m, gravity=(0.0, 0.0, 0.0), plane_d=-1e6)
    o = orc.Oracle(sc)
    x = rest.copy()
    x[1] = [-h * np.cos(fold), h * np.sin(fold), L / 2]  # rotate wing 2 about the edge
    f = o.forces(x, mask=orc.HINGES)[0]
    mag = kb * L * abs(np.sin(fold / 2)) / h
    assert abs(np.linalg.norm(f[0]) - mag) <= 1e-12 * max(mag, 1.0) and abs(np.linalg.norm(f[1]) - mag) <= 1e-12 * max(mag, 1.0)
    assert np.abs(f.sum(0)).max() <= 1e-12 * max(mag, 1.0)
    assert np.abs(f[2] - f[3]).max() <= 1e-12 * max(mag, 1.0)            # mid-edge wings: the edge vertices share equally
    if fold != 0.0:
        n1 = np.cross(x[0] - x[2], x[0] - x[3]); n1 /= np.linalg.norm(n1)
        assert abs(abs(f[0] @ n1) - mag) <= 1e-12 * mag                    # along the face normal
        # unfolding: the work of the wing forces along an opening motion of wing 2 is positive
        open_dir = np.array([h * np.sin(fold), h * np.cos(fold), 0.0]) * (-np.sign(fold))
        assert f[1] @ open_dir > 0
    # dL/dk_b of one substep by linearity of the force in k_b
    rng = np.random.default_rng(3)
    bx, bv = rng.normal(size=(4, 3)), rng.normal(size=(4, 3))
    v = np.zeros_like(x)
    o.zero_grads()
    o.step_adjoint(x, v, bx, bv)
    a = dt * (1.0 / float(sc.mass[0, 0])) * (bv + dt * bx)               # cotangent of the force
    want = (a * f).sum() / float(sc.hinge_kb[0])
    assert abs(o.grads("hinge_kb")[0, 0] - want) <= 1e-12 * max(abs(want), 1e-30)


def test_contact_parameter_gradients_closed_form():
    """Two free particles below the plane, no elements, one substep, L = bx.x+ + bv.v+ (A7, A8).
    Particle 0 slides fast and approaches (slip + normal damping), particle 1 creeps (stick).  With lam = bv + dt bx
    (cotangent of v+), w = 1/m:  dL/dk_e = sum w dt lam.(d f/d k_e) etc., written out by hand:
      slip : f = (-mu fn, fn, 0) for v_t along +x, fn = -k_e c - k_d v_n   ->  d/dk_e = -c (-mu, 1, 0), d/dk_d = -v_n (-mu, 1, 0),
             d/dmu = (-fn, 0, 0), d/dk_f = 0
      stick: f = (-k_f v_x, fn, -k_f v_z)                                  ->  d/dk_f = (-v_x, 0, -v_z), d/dk_e = -c (0, 1, 0), d/dmu = 0."""
    dt, m, ke, kd, kf, mu = 1.0 / 1920.0, 0.1, 1e4, 10.0, 50.0, 0.5
    x = np.array([[0.0, -0.010, 0.0], [1.0, -0.002, 0.0]])
    v = np.array([[3.0, -0.2, 0.0], [1e-3, 0.0, -2e-3]])
    sc = scenes.custom_scene(x, v0=v, dt=dt, mass=m, ke=ke, kd=kd, kf=kf, mu_c=mu)
    o = orc.Oracle(sc)
    x, v, m = sc.x0[0].astype(np.float64), sc.v0[0].astype(np.float64), float(sc.mass[0, 0])  # the fp32-rounded inputs (A19)
    bx = np.array([[0.3, -0.7, 0.2], [0.5, 0.4, -0.6]]); bv = np.array([[-0.2, 0.9, 0.1], [0.8, -0.3, 0.25]])
    o.zero_grads()
    o.step_adjoint(x, v, bx, bv)
    lam = bv + dt * bx
    w = 1.0 / m
    c0, vn0, c1 = x[0, 1], v[0, 1], x[1, 1]
    fn0 = -ke * c0 - kd * vn0
    assert mu * fn0 / 3.0 < kf            # particle 0 slips
    assert mu * (-ke * c1) / np.hypot(v[1, 0], v[1, 2]) >= kf   # particle 1 sticks
    want = dict(
        ke=w * dt * (lam[0] @ (-c0 * np.array([-mu, 1.0, 0.0])) + lam[1] @ (-c1 * np.array([0.0, 1.0, 0.0]))),
        kd=w * dt * (lam[0] @ (-vn0 * np.array([-mu, 1.0, 0.0]))),
        mu_c=w * dt * (lam[0] @ np.array([-fn0, 0.0, 0.0])),
        kf=w * dt * (lam[1] @ np.array([-v[1, 0], 0.0, -v[1, 2]])),
    )
    for k, val in want.items():
        got = o.grads(k)[0, 0]
        assert abs(got - val) <= 1e-12 * max(abs(val), 1e-30), (k, got, val)


def test_p7_conservative_forces_have_symmetric_jacobian():
    """Position-VJP of an elastic force equals its directional derivative (f(x+ea)-f(x-ea))/2e."""
    rng = np.random.default_rng(12)
    sc = _free(_mixed_scene(rng, damp=0.0, tri_damp=0.0))
    o = orc.Oracle(sc)
    N = sc.n_particles
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (N, 3))
    a = rng.normal(size=(N, 3))
    eps = 1e-6
    mask = orc.TETS | orc.TRIS | orc.HINGES
    jvp = (o.forces(x + eps * a, mask=mask)[0] - o.forces(x - eps * a, mask=mask)[0]) / (2 * eps)
    # step adjoint with bx = 0, bv = a / (dt w): adj_f = a, so ax = (df/dx)^T a
    w = 1.0 / sc.mass.astype(np.float64)[0][:, None]
    ax, _ = o.step_adjoint(x, np.zeros_like(x), np.zeros_like(x), a / (o.dt * w))
    assert np.abs(ax[0] - jvp).max() <= 1e-6 * np.abs(jvp).max()


# ---------------------------------------------------------------- P8 whole-rollout adjoint vs FD
def _rollout_loss(sc, o, x0, v0, T, lt, target, K=1):
    ro = o.rollout(x0, v0, T, K=K, rec_times=lt)
    L, cot = orc.loss_and_cotangents(sc.loss, ro["rec_x"], target)
    return L.sum(), ro, cot


@pytest.mark.parametrize("which", ["box", "cloth"])
def test_p8_rollout_adjoint_vs_central_fd(which):
    rng = np.random.default_rng(13)
    if which == "box":  # config-0-shaped: drops, hits the ground inside the window
        sc = scenes.box_scene(cells=(2, 2, 2), y0=0.004, n_substeps=160)
        sc.v0[:] = (0.4, -0.5, 0.2)
        sc.tet_mu[:] = rng.uniform(5e3, 2e4, sc.tet_mu.shape); sc.tet_lambda[:] = rng.uniform(5e3, 2e4, sc.tet_mu.shape)
        sc.mass[:] = rng.uniform(0.05, 0.2, sc.mass.shape)
        groups = ["tet_mu", "tet_lambda", "tet_damp", "mass", "ke", "kd", "mu_c"]
    else:  # config-1-shaped cloth with pins, bending, contact
        sc = scenes.cloth_scene(n=5, n_substeps=200, y0=0.003)
        sc.tri_mu[:] = rng.uniform(5e2, 2e3, sc.tri_mu.shape)
        groups = ["tri_mu", "tri_lambda", "tri_damp", "mass", "hinge_kb", "ke", "kd", "kf", "mu_c"]
    T, lt = sc.n_substeps, sc.loss_times()
    o = orc.Oracle(sc)
    x0, v0 = sc.x0.astype(np.float64), sc.v0.astype(np.float64)
    L, ro, cot = _rollout_loss(sc, o, x0, v0, T, lt, sc.target)
    assert (ro["xT"][0, :, 1] < 0).any()  # contact was active
    o.zero_grads()
    ax0, av0 = o.rollout_backward(ro, lt, cot)
    SCALAR = ("ke", "kd", "kf", "mu_c")
    grads = {g: (o.grads(g)[:, 0] if g in SCALAR else o.grads(g)[0]).copy() for g in groups}

    tol = 1e-5  # north_star check (c), on both scenes

    def check(an, fd_fun, scale):
        # "where a kink crossing spoils one FD step, repeat with two step sizes and take the consistent
        # pair".  A ladder of step sizes is walked and the entry passes only when TWO different step sizes both
        # reproduce the adjoint to `tol` (so they also agree with each other to 2 tol).  These scenes rest on the ground,
        # so |y| of some particle at some substep is as small as 1e-9: the loss is piecewise smooth with pieces that
        # small (forces are only C0; A20) and a central difference is only valid below the kink spacing,
        # while round-off of L spoils the smallest steps.  test_p8_smooth_regime_strict needs no ladder.
        hits = 0
        for h_rel in (1e-6, 1e-7, 1e-5, 1e-8, 1e-4, 1e-9, 1e-10, 1e-11):
            if abs(an - fd_fun(h_rel)) <= tol * scale:
                hits += 1
                if hits == 2:
                    return True
        return False

    for g in groups:
        base = getattr(sc, {"mass": "mass"}.get(g, g)).astype(np.float64)
        base = base if g == "hinge_kb" or g in SCALAR else base[0]
        scale = np.abs(grads[g]).max()
        if g in ("kf", "mu_c") and scale == 0:
            continue  # no particle in that friction regime over this rollout
        assert scale > 0
        idx = rng.choice(base.size, size=min(6, base.size), replace=False)
        for e in idx:
            if g == "mass" and sc.pinned[e]:
                assert grads[g][e] == 0
                continue

            def fd_fun(h_rel, e=e):
                h = h_rel * base[e]
                vals = []
                for s in (+1, -1):
                    p = base.copy(); p[e] += s * h
                    o.set_params(g, p)
                    vals.append(_rollout_loss(sc, o, x0, v0, T, lt, sc.target)[0])
                o.set_params(g, base)
                return (vals[0] - vals[1]) / (2 * h)

            assert check(grads[g][e], fd_fun, scale), (g, e)
    # state gradients
    for arr, an, nm in ((x0, ax0, "x0"), (v0, av0, "v0")):
        scale = np.abs(an).max()
        free = np.where(sc.pinned == 0)[0]
        for i in rng.choice(free, size=4, replace=False):
            r = int(rng.integers(3))

            def fd_fun(h_rel, i=i, r=r):
                h = h_rel * (0.01 if nm == "x0" else 1.0)
                vals = []
                for s in (+1, -1):
                    a = arr.copy(); a[0, i, r] += s * h
                    vals.append(_rollout_loss(sc, o, a if nm == "x0" else x0, a if nm == "v0" else v0, T, lt, sc.target)[0])
                return (vals[0] - vals[1]) / (2 * h)

            assert check(an[0, i, r], fd_fun, scale), (nm, i, r)


def test_p8_smooth_regime_strict():
    """No contact (airborne, tumbling, deformed mixed mesh with a pin): one fixed FD step must match to 1e-5."""
    rng = np.random.default_rng(16)
    sc = _mixed_scene(rng, pinned=[0] * 16 + [1], n_substeps=120)
    sc.plane_d = -1e6
    T = 120
    o = orc.Oracle(sc)
    x0 = sc.x_rest.astype(np.float64)[None] + 0.004 * rng.uniform(-1, 1, (1, sc.n_particles, 3))
    v0 = 0.3 * rng.normal(size=x0.shape); v0[0, 16] = 0
    tgt = x0.mean(1) + np.array([[0.1, -0.2, 0.05]])

    def loss(xa, va):
        ro = o.rollout(xa, va, T, rec_times=[T])
        L, cot = orc.loss_and_cotangents("final_centroid", ro["rec_x"], tgt)
        return L.sum(), ro, cot

    L, ro, cot = loss(x0, v0)
    o.zero_grads()
    ax0, av0 = o.rollout_backward(ro, [T], cot)
    for g in orc.GROUPS:
        an, base = _param(sc, o, g)
        for e in rng.choice(base.size, size=min(4, base.size), replace=False):
            if g == "mass" and sc.pinned[e]:
                assert an[e] == 0
                continue
            # (the air coefficients barely move this loss: |dL/dk| ~ 1e-8 against L ~ 0.05, so their step is larger to keep
            # the difference of the two losses above round-off)
            h = (1e-3 if g in ("k_drag", "k_lift") else 1e-5) * (base[e] if g not in ABS_STEP else 1.0)
            vals = []
            for sgn in (+1, -1):
                p = base.copy(); p[e] += sgn * h
                o.set_params(g, p)
                vals.append(loss(x0, v0)[0])
            o.set_params(g, base)
            assert abs(an[e] - (vals[0] - vals[1]) / (2 * h)) <= 1e-5 * np.abs(an).max(), (g, e)
    for nm, an, h in (("x0", ax0, 1e-7), ("v0", av0, 1e-6)):
        for i in rng.choice(sc.n_particles, size=5, replace=False):
            r = int(rng.integers(3))
            d = np.zeros_like(x0); d[0, i, r] = h
            fd = (loss(x0 + d, v0)[0] - loss(x0 - d, v0)[0]) / (2 * h) if nm == "x0" else (loss(x0, v0 + d)[0] - loss(x0, v0 - d)[0]) / (2 * h)
            assert abs(an[0, i, r] - fd) <= 1e-5 * np.abs(an).max(), (nm, i, r)


def test_p8_linear_in_cotangent_and_zero_cotangent():
    rng = np.random.default_rng(14)
    sc = scenes.box_scene(cells=(2, 1, 1), y0=0.002, n_substeps=40)
    o = orc.Oracle(sc)
    ro = o.rollout(sc.x0, sc.v0, 40)
    c1, c2 = rng.normal(size=(1, 1, sc.n_particles, 3)), rng.normal(size=(1, 1, sc.n_particles, 3))

    def run(c):
        o.zero_grads()
        ax, av = o.rollout_backward(ro, [40], c)
        return np.concatenate([ax.ravel(), av.ravel(), o.grads("tet_mu").ravel(), o.grads("mass").ravel()])

    r0 = run(0 * c1)
    assert np.all(r0 == 0)  # zero cotangent => zero gradient
    r1, r2, r12 = run(c1), run(c2), run(2.0 * c1 - 3.0 * c2)
    assert np.abs(r12 - (2.0 * r1 - 3.0 * r2)).max() <= 1e-12 * np.abs(r12).max()


# ---------------------------------------------------------------- P9 checkpointing
@pytest.mark.parametrize("K", [7, 32, 100])
def test_p9_checkpointed_backward_is_bitwise_full_tape(K):
    sc = scenes.hetero_solid_scene(cells=(2, 2, 2), y0=0.003, n_substeps=75)
    lt = sc.loss_times()
    o = orc.Oracle(sc)
    ref = scenes.rng_for(2, "misc").normal(size=(len(lt), 1, sc.n_particles, 3))
    outs = []
    for k in (1, K):
        o.zero_grads()
        ro = o.rollout(sc.x0, sc.v0, 75, K=k, rec_times=lt)
        L, cot = orc.loss_and_cotangents(sc.loss, ro["rec_x"], ref)
        ax0, av0 = o.rollout_backward(ro, lt, cot)
        outs.append((L, ax0, av0, o.grads("tet_mu"), o.grads("tet_lambda"), o.grads("tet_damp"), o.grads("mass")))
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------- losses
def test_loss_cotangents_vs_fd():
    rng = np.random.default_rng(15)
    for kind, tshape in (("final_centroid", (2, 3)), ("pos_mse_frames", (3, 2, 5, 3)), ("centroid_traj", (3, 2, 3))):
        n_t = 1 if kind == "final_centroid" else 3
        xs = rng.normal(size=(n_t, 2, 5, 3)); tg = rng.normal(size=tshape)
        L, cot = orc.loss_and_cotangents(kind, xs, tg)
        d = rng.normal(size=xs.shape); eps = 1e-6
        fd = (orc.loss_and_cotangents(kind, xs + eps * d, tg)[0].sum() - orc.loss_and_cotangents(kind, xs - eps * d, tg)[0].sum()) / (2 * eps)
        assert abs((cot * d).sum() - fd) <= 1e-8 * abs(fd)


def test_openmp_thread_count_does_not_change_results():
    sc = scenes.make_scene(3, small=True)
    sc.n_substeps = 20
    a = orc.Oracle(sc).rollout(sc.x0, sc.v0, 20)["xT"]
    sc1 = scenes.batched_sysid_scene(n_envs=1, n_substeps=20, y0=0.02)
    for k in ("tet_mu", "tet_lambda", "mass", "mu_c"):
        setattr(sc1, k, getattr(sc, k)[2:3])
    b = orc.Oracle(sc1).rollout(sc1.x0, sc1.v0, 20)["xT"]
    assert np.array_equal(a[2], b[0])  # env-parallel run == the same env alone (element-parallel run)


# ---------------------------------------------------------------- actuation
def test_actuation_closed_forms_tet_and_hinge():
    """alpha of (J - alpha)^2 is "a per-element actuation value that allows the element to expand and
    contract".  With reading A1, alpha = 1 + 3mu/(4 lambda) + act, at the rest shape F = I: P = -lambda act I, so the corner
    tet with legs a (B = I/a, V = a^3/6) gets H = -V P B^T = (a^2 lambda act / 6) I -- outward for act > 0 -- and the
    uniformly scaled shape x = s X is force-free where mu (1 - 1/(3s^2+1)) s + (lambda (s^3 - 1 - act) - 3mu/4) s^2 = 0.
    PAPER.md:585-586: f_b = k_b sin(phi/2 + alpha) d: on the symmetric fold of test_hinge_force_closed_form the wing force is
    k_b L |sin(theta/2 + alpha)| / h and vanishes at theta = -2 alpha ("flex inwards or outwards")."""
    a, mu, lam = 0.25, 1.25e4, 2.0e4
    X = np.array([[0, 0, 0], [a, 0, 0], [0, a, 0], [0, 0, a]], dtype=np.float64)
    o = orc.Oracle(_free(scenes.custom_scene(X, tets=[[0, 1, 2, 3]], mu=mu, lam=lam, damp=0.0)))
    for act in (0.125, -0.0625):
        o.set_act_current(tet_act=[act])
        f = o.forces(X, mask=orc.TETS)[0]
        c = a * a * lam * act / 6
        assert np.abs(f - np.vstack([np.full(3, -c), c * np.eye(3)])).max() <= 1e-12 * abs(c)
        lo, hi = 0.5, 2.0  # root of the rest-stability polynomial by bisection
        p = lambda s: mu * (1 - 1 / (3 * s * s + 1)) * s + (lam * (s ** 3 - 1 - act) - 0.75 * mu) * s * s
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if p(lo) * p(mid) > 0 else (lo, mid)
        s_eq = 0.5 * (lo + hi)
        assert (s_eq > 1) == (act > 0)
        assert np.abs(o.forces(s_eq * X, mask=orc.TETS)[0]).max() <= 1e-9 * abs(c)
    L, h, kb = 0.5, 0.25, 7.0
    rest = np.array([[h, 0.0, L / 2], [-h, 0.0, L / 2], [0.0, 0.0, 0.0], [0.0, 0.0, L]])
    oh = orc.Oracle(_free(scenes.custom_scene(rest, tris=[[2, 3, 0], [3, 2, 1]], hinges=[[0, 1, 2, 3]], kb=kb)))
    # rotating wing 2 by +fold about the edge (as in the test above) is a signed dihedral theta = -fold (A13 orientation)
    for alpha, fold in ((0.2, 0.3), (-0.15, 0.0), (0.1, 0.2)):
        oh.set_act_current(hinge_act=[alpha])
        x = rest.copy()
        x[1] = [-h * np.cos(fold), h * np.sin(fold), L / 2]
        f = oh.forces(x, mask=orc.HINGES)[0]
        mag = kb * L * abs(np.sin(-fold / 2 + alpha)) / h
        assert abs(np.linalg.norm(f[0]) - mag) <= 1e-12 * max(mag, 1.0) and abs(np.linalg.norm(f[1]) - mag) <= 1e-12 * max(mag, 1.0)
    assert np.abs(f).max() <= 1e-12  # the last case sits at theta = -2 alpha: the actuated rest angle


def test_actuation_forces_are_energy_gradients_and_conserve_momentum():
    """With random activations on every tet and hinge: f = -grad U still holds (P3; U carries act / alpha as in the
    oracle's header), internal forces still have zero net force and torque (P4)."""
    rng = np.random.default_rng(21)
    sc = _free(_mixed_scene(rng, damp=0.0, tri_damp=0.0))
    o = orc.Oracle(sc)
    o.set_act_current(tet_act=rng.uniform(-0.1, 0.1, sc.tets.shape[0]), hinge_act=rng.uniform(-0.3, 0.3, sc.hinges.shape[0]))
    N = sc.n_particles
    x = sc.x_rest.astype(np.float64) + 0.01 * rng.uniform(-1, 1, (N, 3))
    mask = orc.TETS | orc.HINGES
    f = o.forces(x, mask=mask)[0]
    eps, g = 1e-6, np.zeros((N, 3))
    for i in range(N):
        for r in range(3):
            d = np.zeros((N, 3)); d[i, r] = eps
            g[i, r] = -(o.energy(x + d, mask=mask)[0] - o.energy(x - d, mask=mask)[0]) / (2 * eps)
    assert np.abs(f - g).max() <= 1e-7 * np.abs(f).max()
    assert np.abs(f.sum(0)).max() <= 1e-10 * np.abs(f).max()
    assert np.abs(np.cross(x, f).sum(0)).max() <= 1e-10 * np.abs(f).max()


def test_actuation_gradients_vs_fd_step_and_rollout():
    """dL/d(act) per tet and per hinge: one substep against central FD (exact structure: P7), then a scheduled rollout
    (frames of 8 substeps, airborne so that FD is valid at one fixed step: P8 strict), then the checkpointed backward
    must reproduce the full-tape gradients bit for bit (P9) -- the replay has to reload each substep's frame."""
    rng = np.random.default_rng(22)
    sc = _mixed_scene(rng, n_substeps=40)
    sc.plane_d = -1e6
    o = orc.Oracle(sc)
    M, Mh, N = sc.tets.shape[0], sc.hinges.shape[0], sc.n_particles
    x = sc.x_rest.astype(np.float64)[None] + 0.004 * rng.uniform(-1, 1, (1, N, 3))
    v = 0.3 * rng.normal(size=x.shape)
    ta, ha = rng.uniform(-0.05, 0.05, (1, M)), rng.uniform(-0.2, 0.2, (1, Mh))
    bx, bv = rng.normal(size=(N, 3)), rng.normal(size=(N, 3))
    o.set_act_current(ta, ha)
    o.zero_grads()
    o.step_adjoint(x, v, bx, bv)
    gt, gh = o.act_grads_current()

    def phi():
        xo, vo = o.step(x, v)
        return (xo[0] * bx).sum() + (vo[0] * bv).sum()

    for arr, g, setter in ((ta, gt, lambda a: o.set_act_current(tet_act=a)), (ha, gh, lambda a: o.set_act_current(hinge_act=a))):
        assert np.abs(g).max() > 0
        for e in range(arr.shape[1]):
            vals = []
            for sgn in (+1, -1):
                p = arr.copy(); p[0, e] += sgn * 1e-6
                setter(p); vals.append(phi())
            setter(arr)
            assert abs(g[0, e] - (vals[0] - vals[1]) / 2e-6) <= 1e-6 * np.abs(g).max(), e
    # scheduled rollout: 5 frames of 8 substeps
    T, stride, F = 40, 8, 5
    st, sh = rng.uniform(-0.05, 0.05, (F, 1, M)), rng.uniform(-0.2, 0.2, (F, 1, Mh))
    tgt = x.mean(1) + np.array([[0.1, -0.2, 0.05]])

    def loss(st_, sh_, K=1):
        o.set_act_schedule(stride, st_, sh_)
        ro = o.rollout(x, v, T, K=K, rec_times=[T])
        L, cot = orc.loss_and_cotangents("final_centroid", ro["rec_x"], tgt)
        return L.sum(), ro, cot

    L0, ro, cot = loss(st, sh)
    o.zero_grads()
    ax0, _ = o.rollout_backward(ro, [T], cot)
    gst, gsh = o.act_schedule_grads()
    gmu = o.grads("tet_mu").copy()
    assert np.abs(gst[0]).max() > 0 and np.abs(gst[-1]).max() > 0 and np.abs(gsh).max() > 0
    for arr, g, which in ((st, gst, 0), (sh, gsh, 1)):
        for _ in range(6):
            f_, e = int(rng.integers(F)), int(rng.integers(arr.shape[2]))
            vals = []
            for sgn in (+1, -1):
                p = arr.copy(); p[f_, 0, e] += sgn * 1e-5
                vals.append(loss(p if which == 0 else st, p if which == 1 else sh)[0])
            assert abs(g[f_, 0, e] - (vals[0] - vals[1]) / 2e-5) <= 1e-5 * np.abs(g).max(), (which, f_, e)
    for K in (7, 16):
        _, rok, cotk = loss(st, sh, K=K)
        o.zero_grads()
        axk, _ = o.rollout_backward(rok, [T], cotk)
        gk_t, gk_h = o.act_schedule_grads()
        assert np.array_equal(axk, ax0) and np.array_equal(gk_t, gst) and np.array_equal(gk_h, gsh) and np.array_equal(o.grads("tet_mu"), gmu)
    # no schedule and zero current activation: the passive model of every other test
    o.set_act_schedule(1, None, None)
    o.set_act_current(np.zeros((1, M)), np.zeros((1, Mh)))
    o2 = orc.Oracle(sc)
    assert np.array_equal(o.step(x, v)[0], o2.step(x, v)[0])


# ---------------------------------------------------------------- lift / drag on cloth faces
def test_aero_closed_forms_and_dissipation():
    """PAPER.md:586 ("a lift/drag model that approximates the effect of the surrounding air on the surface of mesh") with
    reading A21: F = -A s (k_drag vb + k_lift (n.vb) n), s = |vb|, vb = mean vertex velocity - wind, shared equally by the
    three vertices.  Right triangle with legs a in the xz-plane (A = a^2/2, n = +y), elastic terms switched off:
      moving along its normal at speed u   ->  F = -A u^2 (k_drag + k_lift) n
      moving in its own plane at speed u   ->  F = -A u^2 k_drag t         (no pressure term: n.vb = 0)
      at rest in still air                 ->  F = 0
      at rest in a wind w                  ->  F = +A |w| (k_drag w + k_lift (n.w) n)
    and for any state F.vb = -A s (k_drag |vb|^2 + k_lift (n.vb)^2) <= 0: the air only dissipates."""
    a, kd_, kl_ = 0.25, 0.75, 0.5
    X = np.array([[0, 0, 0], [a, 0, 0], [0, 0, -a]], dtype=np.float64)  # normal +y
    A, n = a * a / 2, np.array([0.0, 1.0, 0.0])

    def force(v, wind=(0.0, 0.0, 0.0)):
        sc = scenes.custom_scene(X, tris=[[0, 1, 2]], hinges=np.zeros((0, 4), np.int32), tri_mu=0.0, tri_lam=1.0, tri_damp=0.0,
                                 k_drag=kd_, k_lift=kl_, wind=wind, gravity=(0, 0, 0), plane_d=-1e6)
        return orc.Oracle(sc).forces(X, v=np.broadcast_to(np.asarray(v, np.float64), (3, 3)), mask=orc.TRIS)[0]

    u = 1.5
    f = force(u * n)
    assert np.abs(f.sum(0) - (-A * u * u * (kd_ + kl_) * n)).max() <= 1e-12 and np.abs(f[0] - f[1]).max() == 0 and np.abs(f[0] - f[2]).max() == 0
    t = np.array([0.6, 0.0, -0.8])
    assert np.abs(force(u * t).sum(0) - (-A * u * u * kd_ * t)).max() <= 1e-12
    assert np.abs(force(np.zeros(3))).max() <= 1e-12  # eps = 1e-6 m/s regularisation: |F| <= A eps * 0 = 0 at vb = 0
    w = np.array([0.5, -0.25, 0.125])  # exact in fp32 (A19)
    assert np.abs(force(np.zeros(3), wind=tuple(w)).sum(0) - A * np.linalg.norm(w) * (kd_ * w + kl_ * (n @ w) * n)).max() <= 1e-9
    rng = np.random.default_rng(31)
    for _ in range(20):  # deformed, tumbling triangle: compare against the formula evaluated here and check dissipation
        x = X + 0.05 * rng.normal(size=(3, 3)); v = rng.normal(size=(3, 3))
        sc = scenes.custom_scene(X, tris=[[0, 1, 2]], hinges=np.zeros((0, 4), np.int32), tri_mu=0.0, tri_lam=1.0, tri_damp=0.0,
                                 k_drag=kd_, k_lift=kl_, gravity=(0, 0, 0), plane_d=-1e6)
        F = orc.Oracle(sc).forces(x, v=v, mask=orc.TRIS)[0].sum(0)
        vb = v.mean(0)
        assert F @ vb < 0
        c = np.cross(x[1] - x[0], x[2] - x[0]); Ac = 0.5 * np.linalg.norm(c); nc = c / np.linalg.norm(c)
        assert abs(F @ vb + Ac * np.linalg.norm(vb) * (kd_ * vb @ vb + kl_ * (nc @ vb) ** 2)) <= 1e-9
