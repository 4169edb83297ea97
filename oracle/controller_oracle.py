"""fp64 oracle of the open-loop MPC controller that produces the activation schedule (SURVEY.md 8(f) NEXT-1 "the
sinusoid -> FC -> tanh controller as a consumer").

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle.py): imported only by tests/.  Shares no code with
paper_2104_02646_b200/csrc.

What it follows.  PAPER.md:777 (appendix "MPC Controller Architecture"): "With simulation time t as input we generate N
phase-shifted sinusoidal signals which are passed to a fully-connected layer (zero-bias), and a final activation layer.  The
output is a vector of per-element activation values"; "one fully connected layer and a tanh activation ... 8
time-varying sinusoidal signals".  The paper gives neither the frequency nor the phases; reading A23b:
    s_i(t)   = sin(omega t + 2 pi i / N),  i = 0 .. N-1                  (equally spaced phases)
    act_e(t) = A tanh(sum_i W[e, i] s_i(t))                              (A = 1 is the paper's form)
evaluated at the start time t_f = f frame_dt of every frame of the piecewise-constant schedule (reading A23), for every
environment on its own weights.  dL/dW[e, i] = sum_f dL/dact_e(t_f) A (1 - tanh^2(y_e(t_f))) s_i(t_f).
"""
from __future__ import annotations

import numpy as np


def signals(n_signals, omega, t):
    """[N] phase-shifted sinusoids at time t"""
    return np.sin(omega * t + 2.0 * np.pi * np.arange(n_signals) / n_signals)


def schedule(W, n_frames, frame_dt, omega, amplitude=1.0):
    """W [E, M, N] -> act [F, E, M]"""
    W = np.asarray(W, np.float64)
    act = np.zeros((n_frames,) + W.shape[:2])
    for f in range(n_frames):
        act[f] = amplitude * np.tanh(W @ signals(W.shape[2], omega, f * frame_dt))
    return act


def grads(W, g_act, frame_dt, omega, amplitude=1.0):
    """dL/dW [E, M, N] from dL/dact [F, E, M]"""
    W, g_act = np.asarray(W, np.float64), np.asarray(g_act, np.float64)
    gW = np.zeros_like(W)
    for f in range(g_act.shape[0]):
        s = signals(W.shape[2], omega, f * frame_dt)
        th = np.tanh(W @ s)
        gW += (g_act[f] * amplitude * (1.0 - th * th))[:, :, None] * s[None, None, :]
    return gW
