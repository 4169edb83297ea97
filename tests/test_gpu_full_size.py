"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (plan AUTO).

configs 0, 1, 2   the whole rollout + loss + backward, every output element by element against the oracle.
config 3          the full 1024-environment launch; the oracle recomputes a seeded sample of environments one by
                  one (environments are independent).  The contact force of the method is discontinuous where an
                  approaching particle crosses the plane (f_n jumps by k_d |v_n|, reading A7 / A20), so an
                  environment whose trajectory passes within fp32 resolution of such a crossing has two valid
                  outcomes.  Those are recognised with the oracle alone -- its own result moves by more than the
                  tolerance under perturbations of the initial state of the size of fp32 rounding -- and excluded;
                  every other sampled environment must agree, and the excluded fraction is bounded.
config 4          one substep forward + adjoint at full size from a deformed state and a short airborne rollout, then
                  the FULL 256-substep rollout with the scene's own loss and the whole backward pass against the oracle
                  (~5 min of oracle on the box's host cores), every output element by element.

Relaxed branch (A20).  A gradient array may exceed 2e-3 only where the fp64 oracle's own answer moves by more
than that under fp32-sized perturbations of x0 (contact-rich rollouts: the penalty contact force is discontinuous), and
then only up to that spread.  Every use of the relaxed branch is recorded: the (config, array) pair must be listed in
tests/golden/parity_relaxed_allow.json (so the set cannot grow silently), it raises a warning that `pytest -q` prints
in its summary, and the measured errors / spreads are appended to $GS_PARITY_REPORT (default
gpurun_out/parity_report.jsonl).
"""
import copy
import json
import os
import warnings

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2104_02646_b200 import gradsim as gs
from paper_2104_02646_b200 import scenes

from gpu_util import dev, gpu_run_scene, host, rel_inf

pytestmark = pytest.mark.gpu

TOL_STEP, TOL_ROLLOUT, TOL_GRAD = 1e-5, 1e-3, 2e-3
STATE_GRADS = ("adj_x0", "adj_v0")
_HERE = os.path.dirname(os.path.abspath(__file__))
ALLOW = json.load(open(os.path.join(_HERE, "golden", "parity_relaxed_allow.json")))


def _report(record):
    """Append one JSON record to the parity report and surface it in the pytest summary."""
    path = os.environ.get("GS_PARITY_REPORT", os.path.join(os.path.dirname(_HERE), "gpurun_out", "parity_report.jsonl"))
    try:
        os.makedirs(os.path.dirname(path), exist_ok=True)
        with open(path, "a") as f:
            f.write(json.dumps(record) + "\n")
    except OSError:
        pass
    warnings.warn("parity report: " + json.dumps(record))


def _groups(sc):
    g = ["mass"]
    if sc.tets.shape[0]:
        g += ["tet_mu", "tet_lambda", "tet_damp"]
    if sc.tris.shape[0]:
        g += ["tri_mu", "tri_lambda", "tri_damp"]
    if sc.hinges.shape[0]:
        g += ["hinge_kb"]
    return g


def _fp32_noise(sc):
    """Amplitude of "fp32-sized" noise on x0: four ulps of the largest position coordinate of the scene (fp32 positions are
    rounded to half an ulp every substep and the roundings accumulate as a random walk until the first impact): 1.2e-7 m for
    config 1 (|x| <= 0.31 m), 9.5e-7 m for config 2 (|x| <= 2 m), 3.8e-6 m for config 4 (|x| <= 15.6 m)."""
    return 4.0 * float(np.spacing(np.float32(np.abs(sc.x0).max())))


def _oracle_spread(sc, ref, keys, draws=2):
    """How far the ORACLE's own outputs move (A18 norm) when x0 moves by fp32-sized seeded noise (_fp32_noise).  Contact is
    discontinuous where an approaching particle crosses the plane (f_n jumps by k_d |v_n|, A7 / A20), so a rollout
    with hundreds of particles on the ground has outputs that are only conditioned to this spread, for ANY fp32
    implementation: measured with the oracle alone, a 3e-8 m perturbation of config 1's x0 moves its fp64 dL/dm by 7 % and
    dL/dx0 by 10 % when it flips a contact branch, and by 3e-5 when it does not."""
    r = scenes.rng_for(sc.config, "misc", 4242)
    amp = _fp32_noise(sc)
    spread = {k: 0.0 for k in keys}
    for _ in range(draws):
        s2 = copy.copy(sc)
        s2.x0 = sc.x0.astype(np.float64) + amp * r.normal(size=sc.x0.shape)
        p = orc.run_scene(s2, target=ref["target"])
        for k in keys:
            spread[k] = max(spread[k], rel_inf(p[k], ref[k]))
    return spread


@pytest.mark.parametrize("config", [0, 1, 2])
def test_full_rollout_and_gradients(config):
    sc = scenes.make_scene(config)
    ref = orc.run_scene(sc)
    got = gpu_run_scene(sc, ref["target"])
    assert got["bad"] == -1
    ext = sc.extent()
    free_fall_vy = -9.8 * sc.n_substeps * sc.dt
    assert (np.abs(ref["vT"][..., 1] - free_fall_vy) > 0.5).any()  # the scene hit the ground: contact was exercised
    assert np.abs(got["xT"] - ref["xT"]).max() <= TOL_ROLLOUT * ext
    assert np.abs(got["rec_x"] - ref["rec_x"]).max() <= TOL_ROLLOUT * ext
    assert rel_inf(got["loss"], ref["loss"]) <= TOL_GRAD
    _compare_gradients(f"config{config}", sc, ref, got)


def _compare_gradients(tag, sc, ref, got, draws=None):
    """Every gradient array against the oracle at 2e-3 (A18 norm).  An array beyond that passes only through the relaxed
    branch (module docstring): it must be listed for this config in golden/parity_relaxed_allow.json, the oracle's own
    answer must be conditioned no better than the tolerance there (spread > 2e-3 under fp32-sized noise on x0, _fp32_noise) and the
    CUDA result no further from the oracle than twice what the oracle is from itself -- or the disagreement must be
    confined to at most 0.1 % of the array's entries (a local contact-branch flip).  Everything is recorded."""
    keys = list(STATE_GRADS) + ["g_" + g for g in _groups(sc)]
    errs = {k: rel_inf(got[k], ref[k]) for k in keys}
    for k in keys:
        assert np.abs(ref[k]).max() > 0, k
    late = [k for k in keys if errs[k] > TOL_GRAD]
    if draws is None:
        draws = 4 if sc.n_particles * sc.n_substeps < 2e6 else 2  # the spread is bimodal (a branch flips or not): more draws where they are cheap
    spread = _oracle_spread(sc, ref, late, draws=draws) if late else {}
    # share of an array's entries that are beyond the tolerance: a contact-branch flip of a few particles of a stiff
    # solid is a LOCAL event (its neighbours' entries move, nothing else does), on a cloth sheet it spreads everywhere
    frac = {k: float((np.abs(got[k] - ref[k]) > TOL_GRAD * np.abs(ref[k]).max()).mean()) for k in late}
    _report({"test": tag, "noise_on_x0_m": _fp32_noise(sc), "errors": errs, "relaxed": {k: {"error": errs[k], "oracle_spread": spread[k], "share_of_entries_beyond_tolerance": frac[k]} for k in late}})
    for k in late:
        assert k in ALLOW.get(tag, []), f"{tag}: {k} off by {errs[k]:.2e} and not in parity_relaxed_allow.json"
        ill_conditioned = spread[k] > TOL_GRAD and errs[k] <= 2.0 * spread[k]  # two draws of one distribution: a factor 2
        local = frac[k] <= 1e-3
        assert ill_conditioned or local, (tag, k, errs[k], spread[k], frac[k])


def _env_scene(sc, e):
    """environment e of a batched scene as a scene of its own (inputs only)."""
    s1 = copy.copy(sc)
    s1.n_envs = 1
    for k in ("x0", "v0", "mass", "tet_mu", "tet_lambda", "tet_damp", "tri_mu", "tri_lambda", "tri_damp", "ke", "kd", "kf", "mu_c", "k_drag", "k_lift"):
        setattr(s1, k, getattr(sc, k)[e:e + 1])
    s1.truth = {k: v[e:e + 1] for k, v in sc.truth.items()}
    return s1


C3_KEYS = ("loss", "adj_x0", "adj_v0", "g_tet_mu", "g_tet_lambda", "g_tet_damp", "g_mass")


def _env_metrics(a, ref, ext):
    """(rollout error / extent, worst gradient error) of one environment: the loss, dL/dx0, dL/dv0 and the per-tet /
    per-particle gradient ARRAYS (A18 norm per array), plus the per-environment totals BASELINE.json configs[3] asks for"""
    ex = np.abs(a["xT"] - ref["xT"]).max() / ext
    eg = max(rel_inf(a[k], ref[k]) for k in C3_KEYS)
    for g in ("tet_mu", "tet_lambda", "mass"):
        eg = max(eg, abs(a["g_" + g].sum() - ref["g_" + g].sum()) / abs(ref["g_" + g].sum()))
    return ex, eg


# Measured in round 2 (gpurun_out/parity_report.jsonl, summarised in DESIGN.md A20): 16 of these 128 environments
# (12.5 %) sit at a contact discontinuity -- their ORACLE gradients move by 2 .. 235 tolerances under 1e-6 m
# perturbations of x0 -- now that every per-tet / per-particle array is compared, not only the totals.  The cap leaves
# room for two more; the property is the workload's (a box bouncing on a penalty plane for 1300 substeps), not the GPU's.
C3_SAMPLE, C3_MAX_AMBIGUOUS = 128, 18


def test_config3_full_batch_sampled_environments():
    sc = scenes.make_scene(3)
    assert sc.n_envs == 1024 and sc.n_substeps == 1920
    # targets of the whole batch from the oracle's truth rollouts (forward only, ~10 s on 8 threads)
    target = orc.truth_targets(sc)
    got = gpu_run_scene(sc, target)
    assert got["bad"] == -1
    assert np.isfinite(got["loss"]).all() and np.isfinite(got["g_tet_mu"]).all()
    ext = sc.extent() / 1.0
    sample = scenes.rng_for(3, "misc", 11).choice(sc.n_envs, size=C3_SAMPLE, replace=False)
    ambiguous, worst = [], (0.0, 0.0)
    for e in sample:
        s1 = _env_scene(sc, int(e))
        ref = orc.run_scene(s1, target=target[:, e:e + 1])
        a = {k: got[k][e:e + 1] for k in ("xT",) + C3_KEYS}
        ex, eg = _env_metrics(a, ref, ext)
        if ex <= TOL_ROLLOUT and eg <= TOL_GRAD:
            worst = (max(worst[0], ex), max(worst[1], eg))
            continue
        # disagreement: is the oracle's own answer stable under fp32-sized perturbations of the initial state?
        # (free fall from y ~ 0.5-0.9 m in fp32: ulp 6e-8 per substep over ~600 substeps -> ~1e-6 m at landing)
        r = scenes.rng_for(3, "misc", 1000 + int(e))
        spread = 0.0
        for _ in range(6):
            s2 = copy.copy(s1)
            s2.x0 = s1.x0.astype(np.float64) + 1e-6 * r.normal(size=s1.x0.shape)
            p = orc.run_scene(s2, target=target[:, e:e + 1])
            px, pg = _env_metrics(p, ref, ext)
            spread = max(spread, px / TOL_ROLLOUT, pg / TOL_GRAD)
        assert spread > 0.5, f"env {e}: GPU off by ({ex:.1e}, {eg:.1e}) while the oracle is stable there (spread {spread:.2f})"
        ambiguous.append({"env": int(e), "rollout_err": ex, "grad_err": eg, "oracle_spread_in_tolerances": spread})
    _report({"test": "config3", "sampled": len(sample), "compared": len(sample) - len(ambiguous), "worst_rollout": worst[0], "worst_grad": worst[1],
             "at_contact_discontinuity": ambiguous})
    assert len(ambiguous) <= C3_MAX_AMBIGUOUS


def test_config4_full_size_substep_and_short_rollout():
    sc = scenes.make_scene(4)
    assert sc.tets.shape[0] == 1_000_000 and sc.tris.shape[0] == 522_242 and sc.n_particles == 476_365
    ext = sc.extent()
    x, v = scenes.perturbed_state(sc, amp_x=0.05, amp_v=0.3)
    o = orc.Oracle(sc)
    m = gs.Model(sc)
    # one substep, every particle
    xo, vo = o.step(x, v)
    xg, vg = m.step_forward(dev(x), dev(v))
    assert m.check_finite() == -1
    assert np.abs(host(xg) - xo).max() <= TOL_STEP * ext
    assert rel_inf(host(vg), vo) <= 1e-4
    r = scenes.rng_for(4, "misc", 3)
    bx, bv = r.normal(size=x.shape).astype(np.float32), r.normal(size=x.shape).astype(np.float32)
    o.zero_grads()
    ax, av = o.step_adjoint(x, v, bx, bv)
    m.zero_grads()
    axg, avg = m.step_backward(dev(x), dev(v), dev(bx), dev(bv))
    assert rel_inf(host(axg), ax) <= TOL_GRAD and rel_inf(host(avg), av) <= TOL_GRAD
    for g in _groups(sc):
        assert rel_inf(host(m.param_grads(g)), o.grads(g)) <= TOL_GRAD, g
    # short rollout through tape + backward with the config's own loss, from the same deformed state lifted 5 cm
    # off the ground: with 272k particles at the plane a 12-substep window is certain to put some of them within
    # fp32 resolution of the contact discontinuity (A20); contact at full size is covered by the substep above
    s2 = copy.copy(sc)
    xa = x.copy()
    xa[..., 1] += 0.05
    s2.x0, s2.v0, s2.n_substeps, s2.frame_stride = xa, v, 12, 12
    ref = orc.run_scene(s2)
    got = gpu_run_scene(s2, ref["target"], model=m)
    assert got["bad"] == -1
    assert np.abs(got["xT"] - ref["xT"]).max() <= TOL_ROLLOUT * ext
    for k in ["adj_x0", "adj_v0"] + ["g_" + g for g in _groups(sc)]:
        assert rel_inf(got[k], ref[k]) <= TOL_GRAD, k
    # entry points interleaved on one model at full size (the forward kernel's tile queues are re-zeroed by the
    # particle kernel of every substep, whichever call launched it): two single steps == a 2-substep rollout, up to
    # the order of the atomic sums
    x1, v1 = m.step_forward(dev(x), dev(v))
    x2, v2 = m.step_forward(x1, v1)
    xT, vT = m.tape(2).rollout(dev(x), dev(v))
    assert np.abs(host(x2) - host(xT)).max() <= 1e-6 * ext
    assert rel_inf(host(v2), host(vT)) <= 1e-5


def test_config4_full_rollout_vs_oracle():
    """The whole config-4 workload exactly as bench.py times it (1M tets + 522k triangles + 782k hinges, 256 substeps,
    full tape, the scene's own final-position loss, backward pass) against the oracle, element by element:
    xT <= 1e-3 extent, loss and every parameter gradient <= 2e-3 (north_star).  ~5 min of oracle on 16 host cores."""
    sc = scenes.make_scene(4)
    assert sc.n_substeps == 256 and sc.loss == "pos_mse_frames" and sc.loss_times() == [256]
    ref = orc.run_scene(sc)
    got = gpu_run_scene(sc, ref["target"])
    assert got["bad"] == -1
    ext = sc.extent()
    # both bodies reached the ground inside the rollout (impact ~ substep 123; the sheet is in its first rebound at
    # T): nearly every particle's final velocity is far from free fall, i.e. contact is exercised at full size
    free_fall_vy = -9.8 * sc.n_substeps * sc.dt
    assert (np.abs(ref["vT"][..., 1] - free_fall_vy) > 0.5).sum() > 300_000
    assert np.abs(got["xT"] - ref["xT"]).max() <= TOL_ROLLOUT * ext
    assert rel_inf(got["vT"], ref["vT"]) <= 1e-2  # velocities are not part of the stated tolerances: sanity bound
    assert rel_inf(got["loss"], ref["loss"]) <= TOL_GRAD
    # the 1M-tet solid and the sheet do not interact (A16): the solid's share of every per-particle array is held to 2e-3
    # flat (norm of its own slice); the relaxed branch below is needed by the sheet's entries only (and by dL/dk_damp of the
    # few tets next to a bottom particle whose contact branch flipped)
    Ns = int(sc.tets.max()) + 1
    solid = {k: rel_inf(got[k][:, :Ns], ref[k][:, :Ns]) for k in ("adj_x0", "adj_v0", "g_mass")}
    _report({"test": "config4_solid_particles", "errors": solid, "relaxed": {}})
    for k, e in solid.items():
        assert e <= TOL_GRAD, (k, e)
    _compare_gradients("config4", sc, ref, got, draws=1)


def test_config4_full_rollout_properties():
    """The full 256-substep rollout at full size (too long for the oracle): properties that hold at any size."""
    sc = scenes.make_scene(4)
    m = gs.Model(sc)
    tape = m.tape(sc.n_substeps, 1)
    x0, v0 = dev(sc.x0), dev(sc.v0)
    xT, vT = tape.rollout(x0, v0)
    assert m.check_finite() == -1
    xT = host(xT)
    # nothing tunnels through the ground: penalty equilibrium depth is m g / k_e ~ 1e-4 .. 2e-3 m here
    assert xT[..., 1].min() > -0.05
    # both bodies came down and reached the plane
    assert (xT[..., 1] < 1e-3).sum() > 10_000
    # horizontal momentum only changes through friction: the solid started at rest and must not drift
    Ns = (sc.mass[0] == 0.1).sum()
    assert np.abs(xT[0, :, 0].mean() - sc.x0[0, :, 0].astype(np.float64).mean()) < 1e-3
    # backward with a zero cotangent gives exactly zero everywhere (linearity)
    m.zero_grads()
    z = dev(np.zeros_like(sc.x0))
    ax0, av0 = tape.backward(adj_x_T=z)
    assert float(ax0.abs().max()) == 0.0 and float(av0.abs().max()) == 0.0
    assert float(m.param_grads("tet_mu").abs().max()) == 0.0
    # and is linear in the cotangent: backward(2c) == 2 backward(c) up to atomics' summation order
    c = dev(scenes.rng_for(4, "misc", 9).normal(size=sc.x0.shape).astype(np.float32))
    m.zero_grads()
    a1, _ = tape.backward(adj_x_T=c)
    g1 = m.param_grads("tet_mu").clone()
    m.zero_grads()
    a2, _ = tape.backward(adj_x_T=2 * c)
    g2 = m.param_grads("tet_mu")
    assert rel_inf(host(a2), 2 * host(a1)) <= 1e-4
    assert rel_inf(host(g2), 2 * host(g1)) <= 1e-4


@pytest.mark.parametrize("n,T", [(32, 512), (512, 96)])
def test_contact_rich_rollout_with_smooth_contact_is_strict(n, T):
    """A contact-rich scene whose contact force is SMOOTH, held to the stated tolerances with no relaxed branch (ADVICE
    round 1).  The sheet starts in resting contact at the equilibrium penetration c = -m g / k_e = -9.8e-5 m with seeded
    in-plane velocities (0.1 m/s) and 1e-3 m/s of vertical noise (oscillation amplitude 3e-6 m: no particle ever leaves the
    plane), with k_d = 0 (no normal damping, whose switch at v_n = 0 is a kink of the force) and mu_c = 1e3 (always the stick
    branch: f_f = -k_f v_t).  Then f_contact = -k_e c n - k_f v_t on every particle at every substep, linear in the state,
    and the whole rollout is smooth: measured with the oracle alone, 1e-7 m of noise on x0 moves dL/dx0 by 5e-9 here, against
    21 % with k_d = 10 (every particle crosses v_n = 0 every ~19 substeps, and backpropagation through a kink of a C0
    force is discontinuous in the state: "these forces are only C0 continuous").  Compared strictly: xT, loss,
    dL/dx0, dL/dv0, dL/dm, dL/dk_e, dL/dk_f -- the contact adjoint carries all of them.  The elastic gradients are not
    compared here: stick friction freezes the sheet, so they are zero up to noise in the oracle itself (their strict
    comparisons are the airborne and small-variant tests).  32 x 32 over 512 substeps, and config 4's 512 x 512 sheet
    (262 144 particles) over 96 substeps."""
    sc = scenes.cloth_scene(config=1, n=n, n_substeps=T, y0=-0.1 * 9.8 / 1e4, pins=(n == 32))
    r = scenes.rng_for(1, "misc", 500 + n)
    v0 = r.normal(0.0, 0.1, sc.v0.shape)
    v0[..., 1] = r.normal(0.0, 1e-3, sc.v0.shape[:2])
    v0[:, sc.pinned.astype(bool)] = 0.0
    sc.v0 = v0.astype(np.float32)
    sc.kd[:] = 0.0
    sc.mu_c[:] = 1e3
    ref = orc.run_scene(sc)
    assert ref["xT"][..., 1].max() < 0 and np.abs(ref["g_kf"]).max() > 0 and np.abs(ref["g_mu_c"]).max() == 0  # in contact, stick only
    got = gpu_run_scene(sc, ref["target"])
    assert got["bad"] == -1
    assert np.abs(got["xT"] - ref["xT"]).max() <= TOL_ROLLOUT * sc.extent()
    assert rel_inf(got["loss"], ref["loss"]) <= TOL_GRAD
    errs = {k: rel_inf(got[k], ref[k]) for k in list(STATE_GRADS) + ["g_mass", "g_ke", "g_kf"]}
    _report({"test": f"smooth_contact_{n}x{n}", "errors": errs, "relaxed": {}})
    for k, e in errs.items():
        assert e <= TOL_GRAD, (k, e)
