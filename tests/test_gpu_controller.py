"""Parity of the MPC controller kernels (csrc/gs_controller.cu, through the C ABI) with the fp64 oracle
(oracle/controller_oracle.py; reading A23b), and the control loop of the paper's control-fem task in
state space: weights -> activation schedule -> rollout -> centre-of-mass loss -> backward -> dL/dW, against the oracles
chained the same way."""
import copy

import numpy as np
import pytest
import torch

from oracle import controller_oracle as co
from oracle import oracle as orc
from paper_2104_02646_b200 import gradsim as gs
from paper_2104_02646_b200 import scenes

from gpu_util import dev, gpu_run_scene, host, rel_inf

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("E,M,N,F", [(3, 37, 8, 11), (1, 1, 1, 1), (2, 300, 64, 200), (5, 1152, 8, 60)])
def test_controller_schedule_and_grads_match_the_oracle(E, M, N, F):
    """Random weights (pre-activations up to several units: tanh well into saturation for some elements), times up to
    omega t ~ 100 rad; sizes with a ragged last CTA, a signal table larger than one staging round (64 x 200), and the
    paper's control-fem shape (1152 tets, 8 signals).  act <= 1e-5 absolute, dL/dW <= 1e-4 (A18 norm)."""
    r = np.random.default_rng(100 + N)
    W = r.normal(0, 0.8, (E, M, N)).astype(np.float32)
    frame_dt, omega, amp = 0.0137, 37.0, 0.3
    act = host(gs.controller_schedule(dev(W), F, frame_dt, omega, amp))
    ref = co.schedule(W, F, frame_dt, omega, amp)
    assert act.shape == ref.shape == (F, E, M)
    assert np.abs(ref).max() > 0.1 * amp or F == 1
    assert np.abs(act - ref).max() <= 1e-5
    g_act = r.normal(size=(F, E, M)).astype(np.float32)
    gW = host(gs.controller_grads(dev(W), dev(g_act), frame_dt, omega, amp))
    gref = co.grads(W, g_act, frame_dt, omega, amp)
    assert rel_inf(gW, gref) <= 1e-4 or np.abs(gref).max() == 0


def test_controller_error_paths():
    W = dev(np.zeros((1, 2, 3), np.float32))
    L = gs.lib()
    out = torch.zeros((4, 1, 2), dtype=torch.float32, device="cuda:0")
    assert L.gs_controller_schedule(4, 1, 2, 3, 1.0, 0.0, 1.0, gs._dp(W), gs._dp(out), gs._stream()) == gs.GS_EINVAL   # frame_dt
    assert L.gs_controller_schedule(4, 1, 2, 0, 1.0, 0.1, 1.0, gs._dp(W), gs._dp(out), gs._stream()) == gs.GS_EINVAL   # no signals
    assert L.gs_controller_schedule(4, 1, 2, 3, 1.0, 0.1, 1.0, None, gs._dp(out), gs._stream()) == gs.GS_EINVAL        # null weights
    assert L.gs_controller_grads(4, 1, 2, 3, 1.0, 0.1, 1.0, gs._dp(W), gs._dp(out), None, gs._stream()) == gs.GS_EINVAL
    assert b"controller" in L.gs_last_error()


@pytest.mark.parametrize("config,plan", [(0, gs.GS_PLAN_STREAMING), (3, gs.GS_PLAN_RESIDENT)])
def test_control_loop_gradient_of_the_weights(config, plan):
    """control-fem in state space (actuate a tet mesh towards a target, centre-of-mass loss): the
    controller's weights produce the per-tet activation schedule on the device, the rollout runs under it, and dL/dW comes
    back through the physics adjoint and the controller adjoint; the oracles are chained the same way on the host."""
    sc = copy.copy(scenes.make_scene(config, small=True))
    E, M, N, F, stride = sc.n_envs, sc.tets.shape[0], 8, 6, 16
    frame_dt, omega, amp = stride * sc.dt, 2.0 * np.pi * 4.0, 0.05
    W = scenes.rng_for(config, "misc", 97).normal(0, 0.7, (E, M, N)).astype(np.float32)
    # oracle chain
    sc.act = dict(stride=stride, tet=co.schedule(W, F, frame_dt, omega, amp).astype(np.float32), hinge=None)
    ref = orc.run_scene(sc)
    gW_ref = co.grads(W, ref["g_act_tet"], frame_dt, omega, amp)
    assert np.abs(gW_ref).max() > 0
    # CUDA chain: the schedule never leaves the device
    sg = copy.copy(sc)
    sg.act = None
    m = gs.Model(sg, plan=plan)
    m.actuation(F, stride)
    Wd = dev(W)
    m.set_actuation("tet", gs.controller_schedule(Wd, F, frame_dt, omega, amp))
    got = _run_with_model(sg, ref["target"], m)
    assert m.plan == plan and got["bad"] == -1
    assert np.abs(got["xT"] - ref["xT"]).max() <= 1e-3 * sc.extent()
    gW = host(gs.controller_grads(Wd, m.actuation_grads("tet"), frame_dt, omega, amp))
    assert rel_inf(gW, gW_ref) <= 2e-3


def _run_with_model(sc, target, m):
    """gpu_run_scene on a model whose schedule is already attached (gpu_run_scene would attach sc.act itself)"""
    return gpu_run_scene(sc, target, model=m)
