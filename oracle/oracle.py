"""ctypes wrapper + fp64 losses for the CPU oracle (oracle/gs_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  May be imported only by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
Imports nothing from paper_2104_02646_b200 (scene objects are passed in by the caller
and read by attribute).

Losses (SURVEY.md 8(c) "Losses"; BASELINE.json configs; PAPER.md:365 COM-based loss):
  final_centroid  L_e = || c(x_T) - c* ||^2,                       c(x) = mean_i x_i
  pos_mse_frames  L   = 1/(n_t N) sum_f sum_i || x_i(t_f) - x_i^ref(t_f) ||^2
  centroid_traj   L_e = 1/n_t sum_f || c_e(t_f) - c*_e(t_f) ||^2
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gs_oracle.c")
_LIB = os.path.join(_HERE, "libgs_oracle.so")

TETS, TRIS, HINGES, CONTACT, ALL = 1, 2, 4, 8, 15
GROUPS = {"tet_mu": 0, "tet_lambda": 1, "tet_damp": 2, "tri_mu": 3, "tri_lambda": 4, "tri_damp": 5, "mass": 6, "hinge_kb": 7,
          "ke": 8, "kd": 9, "kf": 10, "mu_c": 11, "gravity": 12, "hinge_theta0": 13, "k_drag": 14, "k_lift": 15}


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) -fopenmp; rebuilt when the source is newer than the .so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_last_error.restype = C.c_char_p
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _i(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """One model (mesh + parameters) in fp64.  State arrays are [E, N, 3] float64."""

    def __init__(self, sc):
        L = lib()
        self.E, self.N = int(sc.n_envs), int(sc.x_rest.shape[0])
        self.M, self.Mt, self.Mh = int(sc.tets.shape[0]), int(sc.tris.shape[0]), int(sc.hinges.shape[0])
        E = self.E

        def full(a, n):
            if n == 0:
                return np.zeros((E, 0))
            return _d(np.broadcast_to(_d(a).reshape(-1, n), (E, n)))

        args = [
            _d(sc.x_rest), full(sc.mass, self.N), np.ascontiguousarray(sc.pinned, dtype=np.uint8),
            _i(sc.tets), full(sc.tet_mu, self.M), full(sc.tet_lambda, self.M), full(sc.tet_damp, self.M),
            _i(sc.tris), full(sc.tri_mu, self.Mt), full(sc.tri_lambda, self.Mt), full(sc.tri_damp, self.Mt),
            _i(sc.hinges), _d(sc.hinge_kb),
        ]
        g, n = _d(sc.gravity), _d(sc.plane_n)
        sc_e = [_d(np.broadcast_to(_d(a).ravel(), (E,))) for a in (sc.ke, sc.kd, sc.kf, sc.mu_c)]
        self._keep = args + [g, n] + sc_e
        h = L.orc_create(
            C.c_int(self.N), C.c_int(self.M), C.c_int(self.Mt), C.c_int(self.Mh), C.c_int(E),
            *[_p(a) for a in args], _p(g), C.c_double(float(sc.dt)), _p(n), C.c_double(float(sc.plane_d)),
            C.c_double(float(sc.radius)), *[_p(a) for a in sc_e],
        )
        if not h:
            raise ValueError("oracle: invalid mesh: " + L.orc_last_error().decode())
        self.h = C.c_void_p(h)
        self.dt = float(sc.dt)
        # lift / drag of the air (reading A21): optional scene attributes, zero when absent
        for g, code in (("k_drag", 14), ("k_lift", 15)):
            val = getattr(sc, g, None)
            if val is not None:
                assert L.orc_set_params(self.h, C.c_int(code), _p(_d(np.broadcast_to(_d(val).ravel(), (E,))))) == 0
        if getattr(sc, "wind", None) is not None:
            assert L.orc_set_params(self.h, C.c_int(16), _p(_d(sc.wind))) == 0

    def __del__(self):
        if getattr(self, "h", None) is not None and _lib is not None:
            _lib.orc_destroy(self.h)
            self.h = None

    # ---- shapes
    def _shape(self):
        return (self.E, self.N, 3)

    def _st(self, a):
        a = _d(a).reshape(self._shape())
        return a

    # ---- per-term evaluation (pins)
    def forces(self, x, v=None, mask=ALL):
        x = self._st(x)
        v = np.zeros_like(x) if v is None else self._st(v)
        f = np.zeros_like(x)
        lib().orc_forces(self.h, _p(x), _p(v), _p(f), C.c_int(mask))
        return f

    def energy(self, x, mask=TETS | TRIS | HINGES):
        x = self._st(x)
        U = np.zeros(self.E)
        lib().orc_energy(self.h, _p(x), C.c_int(mask), _p(U))
        return U

    def rest(self):
        tb, tv = np.zeros((self.M, 3, 3)), np.zeros(self.M)
        rb, ra = np.zeros((self.Mt, 2, 2)), np.zeros(self.Mt)
        th, l0 = np.zeros(self.Mh), np.zeros(self.Mh)
        lib().orc_get_rest(self.h, _p(tb), _p(tv), _p(rb), _p(ra), _p(th), _p(l0))
        return dict(tet_B=tb, tet_V=tv, tri_B=rb, tri_A=ra, theta0=th, l0=l0)

    # ---- parameters / gradients
    def set_params(self, group, values):
        n = {0: self.M, 1: self.M, 2: self.M, 3: self.Mt, 4: self.Mt, 5: self.Mt, 6: self.N, 7: self.Mh, 12: 3, 13: self.Mh}.get(GROUPS[group], 1)
        a = _d(np.broadcast_to(_d(values).reshape(-1, n), (self.E, n)))
        assert lib().orc_set_params(self.h, C.c_int(GROUPS[group]), _p(a)) == 0

    def grads(self, group):
        n = {0: self.M, 1: self.M, 2: self.M, 3: self.Mt, 4: self.Mt, 5: self.Mt, 6: self.N, 7: self.Mh, 12: 3, 13: self.Mh}.get(GROUPS[group], 1)
        out = np.zeros((self.E, n))
        assert lib().orc_get_grads(self.h, C.c_int(GROUPS[group]), _p(out)) == 0
        return out

    def contact_abs_sums(self):
        """[E, 4] diagnostic: sum of |term| behind the totals dL/d(k_e, k_d, k_f, mu_c) -- how far each total cancels."""
        out = np.zeros((self.E, 4))
        assert lib().orc_get_grads(self.h, C.c_int(100), _p(out)) == 0
        return out

    # ---- actuation: current values for single substeps, schedules for rollouts
    def set_act_current(self, tet_act=None, hinge_act=None):
        t = None if tet_act is None else _d(np.broadcast_to(_d(tet_act).reshape(-1, self.M), (self.E, self.M)))
        h = None if hinge_act is None else _d(np.broadcast_to(_d(hinge_act).reshape(-1, self.Mh), (self.E, self.Mh)))
        lib().orc_set_act_current(self.h, _p(t), _p(h))

    def act_grads_current(self):
        gt, gh = np.zeros((self.E, self.M)), np.zeros((self.E, self.Mh))
        lib().orc_get_act_grads_current(self.h, _p(gt), _p(gh))
        return gt, gh

    def set_act_schedule(self, stride, tet=None, hinge=None):
        """tet [F, E, M], hinge [F, E, Mh] (either None): frame f holds during substeps [f stride, (f+1) stride)."""
        F = 0
        t = h = None
        if tet is not None:
            t = _d(tet); F = t.shape[0]; assert t.shape == (F, self.E, self.M)
        if hinge is not None:
            h = _d(hinge); assert F in (0, h.shape[0]); F = h.shape[0]; assert h.shape == (F, self.E, self.Mh)
        self._sched = (F, t is not None, h is not None)
        lib().orc_set_act_schedule(self.h, C.c_int(F), C.c_int(int(stride)), _p(t), _p(h))

    def act_schedule_grads(self):
        F, ht, hh = getattr(self, "_sched", (0, False, False))
        gt = np.zeros((F, self.E, self.M)) if ht else None
        gh = np.zeros((F, self.E, self.Mh)) if hh else None
        lib().orc_get_act_schedule_grads(self.h, _p(gt), _p(gh))
        return gt, gh

    def zero_grads(self):
        lib().orc_zero_grads(self.h)

    # ---- substep
    def step(self, x, v):
        x, v = self._st(x), self._st(v)
        xo, vo = np.zeros_like(x), np.zeros_like(v)
        lib().orc_step(self.h, _p(x), _p(v), _p(xo), _p(vo))
        return xo, vo

    def step_adjoint(self, x, v, bx, bv):
        x, v, bx, bv = self._st(x), self._st(v), self._st(bx), self._st(bv)
        ax, av = np.zeros_like(x), np.zeros_like(v)
        lib().orc_step_adjoint(self.h, _p(x), _p(v), _p(bx), _p(bv), _p(ax), _p(av))
        return ax, av

    # ---- rollout
    def rollout(self, x0, v0, T, K=1, rec_times=(), want_rec_v=False):
        x0, v0 = self._st(x0), self._st(v0)
        n_ck = (T + K - 1) // K
        ck_x, ck_v = np.zeros((n_ck,) + self._shape()), np.zeros((n_ck,) + self._shape())
        rt = _i(sorted(rec_times))
        rec_x = np.zeros((len(rt),) + self._shape())
        rec_v = np.zeros((len(rt),) + self._shape()) if want_rec_v else None
        xT, vT = np.zeros_like(x0), np.zeros_like(v0)
        lib().orc_rollout(
            self.h, C.c_int(T), C.c_int(K), _p(x0), _p(v0), _p(ck_x), _p(ck_v), C.c_int(len(rt)), _p(rt),
            _p(rec_x), _p(rec_v), _p(xT), _p(vT),
        )
        return dict(ck_x=ck_x, ck_v=ck_v, rec_t=rt, rec_x=rec_x, rec_v=rec_v, xT=xT, vT=vT, T=T, K=K)

    def rollout_backward(self, ro, loss_times, loss_ax, adj_vT=None):
        lt = _i(loss_times)
        la = _d(loss_ax).reshape((len(lt),) + self._shape())
        assert np.all(np.diff(lt) > 0) and (len(lt) == 0 or (lt[0] >= 1 and lt[-1] <= ro["T"]))
        avT = None if adj_vT is None else self._st(adj_vT)
        ax0, av0 = np.zeros(self._shape()), np.zeros(self._shape())
        lib().orc_rollout_backward(
            self.h, C.c_int(ro["T"]), C.c_int(ro["K"]), _p(ro["ck_x"]), _p(ro["ck_v"]), C.c_int(len(lt)), _p(lt),
            _p(la), _p(avT), _p(ax0), _p(av0),
        )
        return ax0, av0


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(C.c_int(int(n)))


# ------------------------------------------------------------------ losses (fp64 numpy)
def loss_and_cotangents(kind, xs, target):
    """xs: [n_t, E, N, 3] states at the loss times.  Returns (L [E], dL/dxs [n_t, E, N, 3]).

    final_centroid: n_t == 1, target [E, 3]
    pos_mse_frames: target [n_t, E, N, 3]
    centroid_traj:  target [n_t, E, 3]
    """
    xs = _d(xs)
    n_t, E, N, _ = xs.shape
    if kind == "final_centroid":
        assert n_t == 1
        c = xs[0].mean(axis=1)  # [E,3]
        dlt = c - _d(target).reshape(E, 3)
        L = (dlt**2).sum(-1)
        cot = np.broadcast_to((2.0 * dlt / N)[None, :, None, :], xs.shape).copy()
        return L, cot
    if kind == "pos_mse_frames":
        dlt = xs - _d(target).reshape(xs.shape)
        L = (dlt**2).sum(axis=(0, 2, 3)) / (n_t * N)
        return L, 2.0 * dlt / (n_t * N)
    if kind == "centroid_traj":
        c = xs.mean(axis=2)  # [n_t,E,3]
        dlt = c - _d(target).reshape(n_t, E, 3)
        L = (dlt**2).sum(axis=(0, 2)) / n_t
        cot = np.broadcast_to((2.0 * dlt / (n_t * N))[:, :, None, :], xs.shape).copy()
        return L, cot
    raise ValueError(kind)


def truth_targets(sc):
    """Targets of configs 2 and 3: the oracle's own rollout with the scene's truth-stream parameters
    (guess -> unroll -> compare with the observed trajectory)."""
    import copy

    if sc.target is not None:  # seeded targets (final_centroid [E,3]; final-state position loss [1,E,N,3])
        return _d(sc.target)
    tsc = copy.copy(sc)
    for k, val in sc.truth.items():
        setattr(tsc, k, val)
    o = Oracle(tsc)
    ro = o.rollout(sc.x0, sc.v0, sc.n_substeps, K=max(1, sc.n_substeps), rec_times=sc.loss_times())
    if sc.loss == "pos_mse_frames":
        return ro["rec_x"]
    return ro["rec_x"].mean(axis=2)


def run_scene(sc, target=None, K=None):
    """Forward rollout + loss + backward for a whole scene.  Returns final state, loss, dL/dx0, dL/dv0 and
    every parameter gradient, all fp64."""
    o = Oracle(sc)
    if target is None:
        target = truth_targets(sc)
    act = getattr(sc, "act", None)  # optional actuation schedule: dict(stride=, tet=[F,E,M] or None, hinge=[F,E,Mh] or None)
    if act:
        o.set_act_schedule(act["stride"], act.get("tet"), act.get("hinge"))
    K = sc.checkpoint_every if K is None else K
    lt = sc.loss_times()
    ro = o.rollout(sc.x0, sc.v0, sc.n_substeps, K=K, rec_times=lt)
    L, cot = loss_and_cotangents(sc.loss, ro["rec_x"], target)
    ax0, av0 = o.rollout_backward(ro, lt, cot)
    out = dict(xT=ro["xT"], vT=ro["vT"], loss=L, adj_x0=ax0, adj_v0=av0, rec_x=ro["rec_x"], target=target)
    for g in GROUPS:
        out["g_" + g] = o.grads(g)
    out["contact_abs"] = o.contact_abs_sums()
    if act:
        out["g_act_tet"], out["g_act_hinge"] = o.act_schedule_grads()
    return out
