"""Pins of the controller oracle (oracle/controller_oracle.py; reading A23b).  No GPU."""
import numpy as np

from oracle import controller_oracle as co


def test_signals_closed_forms():
    """N equally phase-shifted sinusoids: the first is sin(omega t); N = 4 gives (sin, cos, -sin, -cos); for N >= 2 they
    sum to zero at every time and sum s_i^2 = N / 2 for N >= 3 (roots of unity)."""
    t, om = 0.37, 5.0
    assert abs(co.signals(1, om, t)[0] - np.sin(om * t)) < 1e-15
    s4 = co.signals(4, om, t)
    assert np.allclose(s4, [np.sin(om * t), np.cos(om * t), -np.sin(om * t), -np.cos(om * t)], atol=1e-15)
    for n in (2, 3, 8, 13):
        s = co.signals(n, om, t)
        assert abs(s.sum()) < 1e-14
        if n >= 3:
            assert abs((s * s).sum() - n / 2) < 1e-13


def test_schedule_closed_forms():
    """W = 0 -> no actuation; equal weights on all signals -> tanh(0) = 0; a single weight on signal 0 -> A tanh(w sin(omega
    f frame_dt)); frame 0 sits at t = 0; the layer has no bias (act is odd in W)."""
    E, M, N, F = 2, 3, 8, 5
    assert np.all(co.schedule(np.zeros((E, M, N)), F, 0.1, 3.0) == 0)
    assert np.abs(co.schedule(np.full((E, M, N), 0.7), F, 0.1, 3.0)).max() < 1e-15
    W = np.zeros((E, M, N)); W[1, 2, 0] = 1.3
    a = co.schedule(W, F, 0.1, 3.0, amplitude=0.25)
    assert np.allclose(a[:, 1, 2], 0.25 * np.tanh(1.3 * np.sin(3.0 * 0.1 * np.arange(F))), atol=1e-15)
    assert np.all(a[:, 0] == 0) and np.all(a[0] == 0)
    Wr = np.random.default_rng(0).normal(size=(E, M, N))
    assert np.allclose(co.schedule(-Wr, F, 0.1, 3.0), -co.schedule(Wr, F, 0.1, 3.0), atol=1e-15)
    assert np.abs(co.schedule(50 * Wr, F, 0.1, 3.0, amplitude=0.3)).max() <= 0.3  # tanh saturates at the amplitude


def test_grads_vs_finite_differences():
    rng = np.random.default_rng(1)
    E, M, N, F = 2, 4, 5, 7
    W, c = rng.normal(size=(E, M, N)), rng.normal(size=(F, E, M))
    L = lambda w: (c * co.schedule(w, F, 0.05, 11.0, 0.4)).sum()
    g = co.grads(W, c, 0.05, 11.0, 0.4)
    fd = np.zeros_like(W)
    for idx in np.ndindex(W.shape):
        d = np.zeros_like(W); d[idx] = 1e-6
        fd[idx] = (L(W + d) - L(W - d)) / 2e-6
    assert np.abs(g - fd).max() <= 1e-8 * np.abs(fd).max()
