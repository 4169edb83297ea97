"""Thin ctypes binding of libgradsim.so (include/gradsim.h).  Argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; torch is used for device
memory (workspace, tape, state tensors) and for the stream handle.  There is NO CPU fallback:
if the library is missing or no CUDA device is present the calls raise.

The module-level ``gs_*`` functions have the C names and take raw pointers; ``Model`` / ``Tape``
wrap them for torch tensors ([E, N, 3] float32 cuda, caller's particle order).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgradsim.so")

GS_OK, GS_EINVAL, GS_EMESH, GS_ENOMEM, GS_ECUDA, GS_ENONFINITE, GS_ESTATE = 0, -1, -2, -3, -4, -5, -6
GROUPS = {"tet_mu": 0, "tet_lambda": 1, "tet_damp": 2, "tri_mu": 3, "tri_lambda": 4, "tri_damp": 5, "mass": 6, "hinge_kb": 7,
          "ke": 8, "kd": 9, "kf": 10, "mu_c": 11, "gravity": 12, "hinge_theta0": 13, "k_drag": 14, "k_lift": 15, "wind": 16}
ACT_KINDS = {"tet": 0, "hinge": 1}
GS_ELEM_PER_ENV, GS_MASS_PER_ENV, GS_CONTACT_PER_ENV = 1, 2, 4
GS_PLAN_AUTO, GS_PLAN_STREAMING, GS_PLAN_RESIDENT = 0, 1, 2
LOSS_KINDS = {"final_centroid": 0, "pos_mse_frames": 1, "centroid_traj": 2}

_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)
_bp = C.POINTER(C.c_uint8)


class gs_model_desc(C.Structure):
    _fields_ = [
        ("n_particles", C.c_int32), ("n_tets", C.c_int32), ("n_tris", C.c_int32), ("n_hinges", C.c_int32), ("n_envs", C.c_int32),
        ("x_rest", _fp), ("mass", _fp), ("pinned", _bp),
        ("tets", _ip), ("tet_mu", _fp), ("tet_lambda", _fp), ("tet_damp", _fp),
        ("tris", _ip), ("tri_mu", _fp), ("tri_lambda", _fp), ("tri_damp", _fp),
        ("hinges", _ip), ("hinge_kb", _fp),
        ("param_layout", C.c_uint32),
        ("gravity", C.c_float * 3), ("dt", C.c_float),
        ("plane_n", C.c_float * 3), ("plane_d", C.c_float), ("particle_radius", C.c_float),
        ("ke", _fp), ("kd", _fp), ("kf", _fp), ("mu_c", _fp),
        ("plan", C.c_int32),
        ("k_drag", _fp), ("k_lift", _fp), ("wind", C.c_float * 3),
    ]


class gs_camera(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float), ("width", C.c_int32), ("height", C.c_int32),
                ("sigma", C.c_float), ("near_z", C.c_float)]


def make_camera(R, t, fx, fy, width, height, sigma, near_z=1e-3):
    c = gs_camera()
    c.R = (C.c_float * 9)(*[float(v) for v in np.asarray(R, np.float64).reshape(9)])
    c.t = (C.c_float * 3)(*[float(v) for v in np.asarray(t, np.float64).reshape(3)])
    c.fx, c.fy, c.width, c.height, c.sigma, c.near_z = float(fx), float(fy), int(width), int(height), float(sigma), float(near_z)
    return c


class gs_shading(C.Structure):
    _fields_ = [("gamma", C.c_float), ("eps", C.c_float), ("far_z", C.c_float), ("background", C.c_float * 3)]


def make_shading(gamma, eps, far_z, background):
    s = gs_shading()
    s.gamma, s.eps, s.far_z = float(gamma), float(eps), float(far_z)
    s.background = (C.c_float * 3)(*[float(v) for v in np.asarray(background, np.float64).reshape(3)])
    return s


# name -> (restype, argtypes); the list tests/test_abi.py checks against include/gradsim.h
_vp, _sz, _int = C.c_void_p, C.c_size_t, C.c_int
_descp = C.POINTER(gs_model_desc)
SIGNATURES = {
    "gs_model_workspace_bytes": (_sz, [_descp]),
    "gs_model_create": (_int, [_descp, _vp, _sz, _vp, C.POINTER(_vp)]),
    "gs_model_destroy": (None, [_vp]),
    "gs_model_plan": (_int, [_vp]),
    "gs_model_info": (_int, [_vp, _ip, _ip, _ip]),
    "gs_set_params": (_int, [_vp, _int, _vp, _vp]),
    "gs_actuation_bytes": (_sz, [_vp, _int]),
    "gs_actuation_create": (_int, [_vp, _int, _int, _vp, _sz, _vp]),
    "gs_set_actuation": (_int, [_vp, _int, _vp, _vp]),
    "gs_actuation_grads": (_int, [_vp, _int, _vp, _vp]),
    "gs_set_actuation_frame": (_int, [_vp, _int]),
    "gs_step_forward": (_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "gs_step_backward": (_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "gs_tape_bytes": (_sz, [_vp, _int, _int]),
    "gs_tape_create": (_int, [_vp, _int, _int, _vp, _sz, C.POINTER(_vp)]),
    "gs_tape_destroy": (None, [_vp]),
    "gs_rollout": (_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "gs_tape_read": (_int, [_vp, _vp, _int, _vp, _vp, _vp]),
    "gs_rollout_backward": (_int, [_vp, _vp, _int, _int, _vp, _vp, _vp, _vp, _vp, _vp]),
    "gs_request_grads": (_int, [_vp, _int, _int]),
    "gs_set_deterministic": (_int, [_vp, _int]),
    "gs_zero_grads": (_int, [_vp, _vp]),
    "gs_param_grads": (_int, [_vp, _int, _vp, _vp]),
    "gs_check_finite": (_int, [_vp, _vp, C.POINTER(_int)]),
    "gs_loss_centroid": (_int, [_int, _int, _vp, _vp, C.c_float, _int, _vp, _vp, _vp]),
    "gs_loss_pos": (_int, [_int, _int, _vp, _vp, C.c_float, _int, _vp, _vp, _vp]),
    "gs_loss_centroid_traj": (_int, [_vp, _vp, _int, _vp, _vp, _vp, _vp, _vp]),
    "gs_controller_schedule": (_int, [_int, _int, _int, _int, C.c_float, C.c_float, C.c_float, _vp, _vp, _vp]),
    "gs_controller_grads": (_int, [_int, _int, _int, _int, C.c_float, C.c_float, C.c_float, _vp, _vp, _vp, _vp]),
    "gs_raster_scratch_bytes": (_sz, [_int, _int, _int]),
    "gs_render_silhouette": (_int, [_int, _int, _vp, _int, _vp, C.POINTER(gs_camera), _vp, _vp, _sz, _vp]),
    "gs_loss_silhouette": (_int, [_int, _int, _vp, _int, _vp, C.POINTER(gs_camera), _vp, C.c_float, _int, _vp, _vp, _vp, _vp, _sz, _vp]),
    "gs_loss_silhouette_static": (_int, [_int, _int, _vp, _int, _vp, C.POINTER(gs_camera), _vp, C.c_float, _int, _vp, _vp, _vp, _vp]),
    "gs_raster_rgb_scratch_bytes": (_sz, [_int, _int, _int]),
    "gs_render_rgb": (_int, [_int, _int, _vp, _int, _vp, _vp, C.POINTER(gs_camera), C.POINTER(gs_shading), _vp, _vp, _sz, _vp]),
    "gs_loss_rgb": (_int, [_int, _int, _vp, _int, _vp, _vp, C.POINTER(gs_camera), C.POINTER(gs_shading), _vp, C.c_float, _int, _vp, _vp, _vp, _vp, _vp,
                           _sz, _vp]),
    "gs_host_scratch_bytes": (_sz, [_vp, _vp, _int, _int]),
    "gs_rollout_loss_backward_host": (_int, [_vp, _vp, _vp, _vp, _int, _int, _vp, _vp, _vp, _vp, _int, C.POINTER(_int), C.POINTER(_vp), _vp, _sz, _vp]),
    "gs_launch_count": (C.c_uint64, []),
    "gs_kernel_timing": (_int, [_vp, _int]),
    "gs_kernel_times": (_int, [_vp, _vp, _int, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]),
    "gs_last_error": (C.c_char_p, []),
    "gs_version": (C.c_char_p, []),
}

_lib = None


class GradSimError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gradsim error {code}: {msg}")
        self.code = code


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (python -m paper_2104_02646_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2104_02646_b200.build` "
                "(there is no CPU fallback for the gradSim hot path)"
            )
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc):
    if rc != GS_OK:
        raise GradSimError(rc, lib().gs_last_error().decode())
    return rc


def _make_gs(name):
    def call(*args):
        return getattr(lib(), name)(*args)

    call.__name__ = name
    call.__doc__ = f"Raw C call {name} (see include/gradsim.h)."
    return call


for _n in SIGNATURES:
    globals()[_n] = _make_gs(_n)


# ------------------------------------------------------------------------------------------ torch-facing wrappers
def _torch():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("gradsim needs a CUDA device (sm_100a); there is no CPU fallback")
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _dp(t):
    """device pointer of a torch tensor or None"""
    return None if t is None else C.c_void_p(t.data_ptr())


def _st(t, shape):
    torch = _torch()
    assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == tuple(shape), (t.shape, shape, t.dtype)
    return t


def _aligned_bytes(nbytes, device):
    """uint8 device block, 256-byte aligned (torch's caching allocator returns >= 512-byte aligned blocks)."""
    torch = _torch()
    t = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)
    assert t.data_ptr() % 256 == 0
    return t


def fill_desc(sc, plan=GS_PLAN_AUTO):
    """gs_model_desc from a scene object (attributes as paper_2104_02646_b200.scenes.Scene).  Returns
    (desc, keepalive list).  Parameter arrays are passed with the leading [E] axis when they have one."""
    keep = []

    def f(a):
        a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
        keep.append(a)
        return a.ctypes.data_as(_fp)

    def i(a):
        a = np.ascontiguousarray(np.asarray(a, dtype=np.int32))
        keep.append(a)
        return a.ctypes.data_as(_ip)

    E, N = int(sc.n_envs), int(sc.x_rest.shape[0])
    M, Mt, Mh = int(sc.tets.shape[0]), int(sc.tris.shape[0]), int(sc.hinges.shape[0])
    d = gs_model_desc()
    d.n_particles, d.n_tets, d.n_tris, d.n_hinges, d.n_envs = N, M, Mt, Mh, E
    d.x_rest = f(sc.x_rest)
    layout = 0
    mass = np.asarray(sc.mass, np.float32)
    if mass.ndim == 2:
        layout |= GS_MASS_PER_ENV
        mass = np.broadcast_to(mass, (E, N))
    d.mass = f(mass)
    pinned = np.ascontiguousarray(np.asarray(sc.pinned, np.uint8))
    keep.append(pinned)
    d.pinned = pinned.ctypes.data_as(_bp)
    per_env = any(np.asarray(a).ndim == 2 for a in (sc.tet_mu, sc.tri_mu))
    if per_env:
        layout |= GS_ELEM_PER_ENV

    def ep(a, n):
        a = np.asarray(a, np.float32)
        if n == 0:
            return f(np.zeros(1, np.float32))
        return f(np.broadcast_to(a.reshape(-1, n), (E, n)) if per_env else a.reshape(n))

    d.tets = i(sc.tets)
    d.tet_mu, d.tet_lambda, d.tet_damp = ep(sc.tet_mu, M), ep(sc.tet_lambda, M), ep(sc.tet_damp, M)
    d.tris = i(sc.tris)
    d.tri_mu, d.tri_lambda, d.tri_damp = ep(sc.tri_mu, Mt), ep(sc.tri_lambda, Mt), ep(sc.tri_damp, Mt)
    d.hinges = i(sc.hinges)
    d.hinge_kb = f(sc.hinge_kb)
    layout |= GS_CONTACT_PER_ENV
    for name in ("ke", "kd", "kf", "mu_c"):
        setattr(d, name, f(np.broadcast_to(np.asarray(getattr(sc, name), np.float32).ravel(), (E,))))
    for name in ("k_drag", "k_lift"):
        val = getattr(sc, name, None)
        setattr(d, name, f(np.broadcast_to(np.zeros(1, np.float32) if val is None else np.asarray(val, np.float32).ravel(), (E,))))
    d.wind = (C.c_float * 3)(*[float(g) for g in getattr(sc, "wind", (0.0, 0.0, 0.0))])
    d.param_layout = layout
    d.gravity = (C.c_float * 3)(*[float(g) for g in sc.gravity])
    d.dt = float(sc.dt)
    d.plane_n = (C.c_float * 3)(*[float(g) for g in sc.plane_n])
    d.plane_d = float(sc.plane_d)
    d.particle_radius = float(sc.radius)
    d.plan = int(plan)
    return d, keep


class Model:
    """One scene on the device.  Owns the torch block the library works in."""

    def __init__(self, sc, plan=GS_PLAN_AUTO, device="cuda:0"):
        torch = _torch()
        self.device = torch.device(device)
        L = lib()
        desc, keep = fill_desc(sc, plan)
        nbytes = L.gs_model_workspace_bytes(C.byref(desc))
        if nbytes == 0:
            raise GradSimError(GS_EINVAL, L.gs_last_error().decode())
        with torch.cuda.device(self.device):
            self.workspace = _aligned_bytes(nbytes, self.device)
            h = C.c_void_p()
            _check(L.gs_model_create(C.byref(desc), _dp(self.workspace), nbytes, _stream(), C.byref(h)))
        self.h = h
        self.E, self.N = int(sc.n_envs), int(sc.x_rest.shape[0])
        self.counts = {"tet": int(sc.tets.shape[0]), "tri": int(sc.tris.shape[0]), "hinge": int(sc.hinges.shape[0])}
        self.n_elements = sum(self.counts.values())
        self.plan = L.gs_model_plan(self.h)
        self._scratch = None
        self._act_mem, self.act_frames = None, 0
        self._want_gravity = False
        del keep

    def __del__(self):
        if getattr(self, "h", None) is not None and _lib is not None:
            _lib.gs_model_destroy(self.h)
            self.h = None

    def _shape(self):
        return (self.E, self.N, 3)

    def group_count(self, group):
        g = GROUPS[group] if isinstance(group, str) else int(group)
        if g in (12, 16):
            return 3  # gravity: dL/dg per environment; wind: one vector
        if g in (14, 15):
            return 1  # air coefficients: one value per environment
        if 8 <= g <= 11:
            return 1  # contact parameters: one value per environment
        return self.N if g == 6 else (self.counts["hinge"] if g in (7, 13) else (self.counts["tet"] if g < 3 else self.counts["tri"]))

    def new_state(self):
        return _torch().empty(self._shape(), dtype=_torch().float32, device=self.device)

    def step_forward(self, x, v, x_out=None, v_out=None):
        x, v = _st(x, self._shape()), _st(v, self._shape())
        x_out = self.new_state() if x_out is None else _st(x_out, self._shape())
        v_out = self.new_state() if v_out is None else _st(v_out, self._shape())
        _check(lib().gs_step_forward(self.h, _dp(x), _dp(v), _dp(x_out), _dp(v_out), _stream()))
        return x_out, v_out

    def step_backward(self, x, v, adj_x_out, adj_v_out):
        sh = self._shape()
        ax, av = self.new_state(), self.new_state()
        _check(lib().gs_step_backward(self.h, _dp(_st(x, sh)), _dp(_st(v, sh)), _dp(_st(adj_x_out, sh)), _dp(_st(adj_v_out, sh)), _dp(ax), _dp(av), _stream()))
        return ax, av

    def set_params(self, group, values):
        n = self.group_count(group)
        _check(lib().gs_set_params(self.h, GROUPS[group], _dp(_st(values, (self.E, n))), _stream()))

    # ---- actuation inputs: a schedule of n_frames frames of frame_stride substeps
    def actuation(self, n_frames, frame_stride=1):
        """Attach an all-zero activation schedule (n_frames = 0 detaches).  The model keeps the torch block alive."""
        L = lib()
        if n_frames == 0:
            _check(L.gs_actuation_create(self.h, 0, 1, None, 0, _stream()))
            self._act_mem, self.act_frames = None, 0
            return
        nbytes = L.gs_actuation_bytes(self.h, int(n_frames))
        mem = _aligned_bytes(nbytes, self.device)
        _check(L.gs_actuation_create(self.h, int(n_frames), int(frame_stride), _dp(mem), nbytes, _stream()))
        self._act_mem, self.act_frames = mem, int(n_frames)

    def set_actuation(self, kind, values):
        n = self.counts[kind]
        _check(lib().gs_set_actuation(self.h, ACT_KINDS[kind], _dp(_st(values, (self.act_frames, self.E, n))), _stream()))

    def actuation_grads(self, kind):
        torch = _torch()
        out = torch.zeros((self.act_frames, self.E, self.counts[kind]), dtype=torch.float32, device=self.device)
        if out.numel():
            _check(lib().gs_actuation_grads(self.h, ACT_KINDS[kind], _dp(out), _stream()))
        return out

    def set_actuation_frame(self, frame):
        _check(lib().gs_set_actuation_frame(self.h, int(frame)))

    def set_deterministic(self, enable=True):
        _check(lib().gs_set_deterministic(self.h, int(bool(enable))))

    def request_grads(self, group, enable=True):
        _check(lib().gs_request_grads(self.h, GROUPS[group], int(bool(enable))))
        self._want_gravity = bool(enable)

    def zero_grads(self):
        _check(lib().gs_zero_grads(self.h, _stream()))

    def param_grads(self, group):
        torch = _torch()
        n = self.group_count(group)
        out = torch.zeros((self.E, n), dtype=torch.float32, device=self.device)
        if n:
            _check(lib().gs_param_grads(self.h, GROUPS[group], _dp(out), _stream()))
        return out

    def check_finite(self):
        bad = C.c_int(-1)
        rc = lib().gs_check_finite(self.h, _stream(), C.byref(bad))
        if rc not in (GS_OK, GS_ENONFINITE):
            _check(rc)
        return bad.value

    def tape(self, n_substeps, checkpoint_every=1):
        return Tape(self, n_substeps, checkpoint_every)

    def rollout_loss_backward_host(self, tape, h_x0, h_v0, h_target, groups=(), loss="final_centroid", frame_stride=1):
        """bench.py's e2e leg: HOST (pinned torch CPU tensors) in, HOST out, ONE C call.  loss / frame_stride /
        h_target as gs_rollout_loss_backward_host documents them.  The returned pinned tensors are owned by the model
        and overwritten by the next call."""
        torch = _torch()
        L = lib()
        kind = LOSS_KINDS[loss]
        need = L.gs_host_scratch_bytes(self.h, tape.h, kind, int(frame_stride))
        if need == 0:
            raise GradSimError(GS_EINVAL, "bad loss arguments")
        if self._scratch is None or self._scratch.numel() < need:
            self._scratch = _aligned_bytes(need, self.device)
        E, N = self.E, self.N
        gl = [GROUPS[g] for g in groups]
        key = tuple(gl)
        if getattr(self, "_host_out", None) is None or self._host_out[0] != key:
            # pinned result buffers are allocated once and reused (page-locking 20+ MB per call costs milliseconds)
            bufs = dict(
                loss=torch.empty(E, dtype=torch.float32).pin_memory(),
                adj_x0=torch.empty((E, N, 3), dtype=torch.float32).pin_memory(),
                adj_v0=torch.empty((E, N, 3), dtype=torch.float32).pin_memory(),
            )
            gb = [torch.empty((E, self.group_count(g)), dtype=torch.float32).pin_memory() for g in groups]
            self._host_out = (key, bufs, gb)
        out = dict(self._host_out[1])
        gbuf = self._host_out[2]
        garr = (C.c_int * max(len(gl), 1))(*gl)
        gptr = (C.c_void_p * max(len(gl), 1))(*[b.data_ptr() for b in gbuf])
        assert h_target.dtype == torch.float32 and h_target.is_contiguous() and not h_target.is_cuda
        _check(L.gs_rollout_loss_backward_host(
            self.h, tape.h, C.c_void_p(h_x0.data_ptr()), C.c_void_p(h_v0.data_ptr()), kind, int(frame_stride), C.c_void_p(h_target.data_ptr()),
            C.c_void_p(out["loss"].data_ptr()), C.c_void_p(out["adj_x0"].data_ptr()), C.c_void_p(out["adj_v0"].data_ptr()),
            len(gl), garr, gptr, _dp(self._scratch), self._scratch.numel(), _stream()))
        for g, b in zip(groups, gbuf):
            out["g_" + g] = b
        return out


class Tape:
    """On-device state tape of one rollout."""

    def __init__(self, model: Model, n_substeps: int, checkpoint_every: int = 1):
        torch = _torch()
        L = lib()
        self.model, self.T, self.K = model, int(n_substeps), int(checkpoint_every)
        nbytes = L.gs_tape_bytes(model.h, self.T, self.K)
        if nbytes == 0:
            raise GradSimError(GS_EINVAL, "bad tape arguments")
        with torch.cuda.device(model.device):
            self.mem = _aligned_bytes(nbytes, model.device)
        h = C.c_void_p()
        _check(L.gs_tape_create(model.h, self.T, self.K, _dp(self.mem), nbytes, C.byref(h)))
        self.h = h
        self.nbytes = nbytes

    def __del__(self):
        if getattr(self, "h", None) is not None and _lib is not None:
            _lib.gs_tape_destroy(self.h)
            self.h = None

    def rollout(self, x0, v0, want_final=True):
        m = self.model
        sh = m._shape()
        xT = m.new_state() if want_final else None
        vT = m.new_state() if want_final else None
        _check(lib().gs_rollout(m.h, self.h, _dp(_st(x0, sh)), _dp(_st(v0, sh)), _dp(xT), _dp(vT), _stream()))
        return xT, vT

    def read(self, substep, want_v=True):
        m = self.model
        x = m.new_state()
        v = m.new_state() if want_v else None
        _check(lib().gs_tape_read(m.h, self.h, int(substep), _dp(x), _dp(v), _stream()))
        return x, v

    def loss_centroid_traj(self, frame_stride, targets, want_adj=True):
        """gs_loss_centroid_traj: (loss [E], dL/dx of the frames [n_t, E, N, 3]) from the tape of the last rollout."""
        torch = _torch()
        m = self.model
        n_t = self.T // int(frame_stride)
        loss = torch.zeros(m.E, dtype=torch.float32, device=m.device)
        adj = torch.empty((n_t,) + m._shape(), dtype=torch.float32, device=m.device) if want_adj else None
        _check(lib().gs_loss_centroid_traj(m.h, self.h, int(frame_stride), _dp(_st(targets, (n_t, m.E, 3))), _dp(loss), _dp(adj), _dp(m.new_state()), _stream()))
        return loss, adj

    def backward(self, adj_x_T=None, adj_v_T=None, adj_x_frames=None, frame_stride=1, want_out=True):
        m = self.model
        sh = m._shape()
        n_frames = 0
        if adj_x_frames is not None:
            n_frames = int(adj_x_frames.shape[0])
            _st(adj_x_frames, (n_frames,) + sh)
        ax0 = m.new_state() if want_out else None
        av0 = m.new_state() if want_out else None
        _check(lib().gs_rollout_backward(
            m.h, self.h, n_frames, int(frame_stride), _dp(adj_x_frames),
            _dp(None if adj_x_T is None else _st(adj_x_T, sh)), _dp(None if adj_v_T is None else _st(adj_v_T, sh)),
            _dp(ax0), _dp(av0), _stream()))
        return ax0, av0


def loss_centroid(x, target, scale=1.0, loss=None, accumulate=False, want_adj=True):
    torch = _torch()
    E, N, _ = x.shape
    loss = torch.zeros(E, dtype=torch.float32, device=x.device) if loss is None else loss
    adj = torch.empty_like(x) if want_adj else None
    _check(lib().gs_loss_centroid(E, N, _dp(x), _dp(_st(target, (E, 3))), float(scale), int(accumulate), _dp(loss), _dp(adj), _stream()))
    return loss, adj


def loss_pos(x, ref, scale=1.0, loss=None, accumulate=False, want_adj=True):
    torch = _torch()
    E, N, _ = x.shape
    loss = torch.zeros(E, dtype=torch.float32, device=x.device) if loss is None else loss
    adj = torch.empty_like(x) if want_adj else None
    _check(lib().gs_loss_pos(E, N, _dp(x), _dp(_st(ref, (E, N, 3))), float(scale), int(accumulate), _dp(loss), _dp(adj), _stream()))
    return loss, adj


# ------------------------------------------------------------------------------------------ soft silhouette rasteriser
def _raster_args(x, tris):
    torch = _torch()
    E, N, _ = x.shape
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
    assert tris.is_cuda and tris.dtype == torch.int32 and tris.is_contiguous() and tris.ndim == 2 and tris.shape[1] == 3
    nbytes = lib().gs_raster_scratch_bytes(E, N, int(tris.shape[0]))
    return E, N, int(tris.shape[0]), _aligned_bytes(nbytes, x.device), nbytes


def render_silhouette(x, tris, cam):
    """x [E, N, 3] cuda fp32, tris [Mt, 3] cuda int32, cam a gs_camera -> silhouette images [E, H, W]."""
    torch = _torch()
    E, N, Mt, scratch, nbytes = _raster_args(x, tris)
    img = torch.empty((E, cam.height, cam.width), dtype=torch.float32, device=x.device)
    _check(lib().gs_render_silhouette(E, N, _dp(x), Mt, _dp(tris), C.byref(cam), _dp(img), _dp(scratch), nbytes, _stream()))
    return img


def loss_silhouette(x, tris, cam, target, scale=None, loss=None, accumulate=False, want_adj=True, want_image=False):
    """L_e (+)= scale sum_p (S_e(p) - target_e(p))^2 (scale defaults to 1 / (W H): the pixelwise mean) and dL/dx."""
    torch = _torch()
    E, N, Mt, scratch, nbytes = _raster_args(x, tris)
    scale = 1.0 / (cam.width * cam.height) if scale is None else float(scale)
    loss = torch.zeros(E, dtype=torch.float32, device=x.device) if loss is None else loss
    adj = torch.empty_like(x) if want_adj else None
    img = torch.empty((E, cam.height, cam.width), dtype=torch.float32, device=x.device) if want_image else None
    _check(lib().gs_loss_silhouette(E, N, _dp(x), Mt, _dp(tris), C.byref(cam), _dp(_st(target, (E, cam.height, cam.width))), scale, int(accumulate),
                                    _dp(loss), _dp(adj), _dp(img), _dp(scratch), nbytes, _stream()))
    return loss, adj, img


def _raster_rgb_args(x, tris, colour):
    torch = _torch()
    E, N, Mt, _, _ = _raster_args(x, tris)
    assert colour.is_cuda and colour.dtype == torch.float32 and colour.is_contiguous() and tuple(colour.shape) == (E, N, 3)
    nbytes = lib().gs_raster_rgb_scratch_bytes(E, N, Mt)
    return E, N, Mt, _aligned_bytes(nbytes, x.device), nbytes


def render_rgb(x, tris, colour, cam, shading):
    """x, colour [E, N, 3] cuda fp32, tris [Mt, 3] cuda int32 -> colour images [E, 3, H, W] (A22b)."""
    torch = _torch()
    E, N, Mt, scratch, nbytes = _raster_rgb_args(x, tris, colour)
    img = torch.empty((E, 3, cam.height, cam.width), dtype=torch.float32, device=x.device)
    _check(lib().gs_render_rgb(E, N, _dp(x), Mt, _dp(tris), _dp(colour), C.byref(cam), C.byref(shading), _dp(img), _dp(scratch), nbytes, _stream()))
    return img


def loss_rgb(x, tris, colour, cam, shading, target, scale=None, loss=None, accumulate=False, want_adj=True, want_adj_colour=True, want_image=False):
    """L_e (+)= scale sum_{p, c} (I_e(p, c) - target_e(p, c))^2 (scale defaults to 1 / (3 W H): the mean), dL/dx, dL/dcolour."""
    torch = _torch()
    E, N, Mt, scratch, nbytes = _raster_rgb_args(x, tris, colour)
    scale = 1.0 / (3 * cam.width * cam.height) if scale is None else float(scale)
    loss = torch.zeros(E, dtype=torch.float32, device=x.device) if loss is None else loss
    adj = torch.empty_like(x) if want_adj else None
    adj_c = torch.empty_like(colour) if want_adj_colour else None
    img = torch.empty((E, 3, cam.height, cam.width), dtype=torch.float32, device=x.device) if want_image else None
    _check(lib().gs_loss_rgb(E, N, _dp(x), Mt, _dp(tris), _dp(colour), C.byref(cam), C.byref(shading), _dp(_st(target, (E, 3, cam.height, cam.width))), scale,
                             int(accumulate), _dp(loss), _dp(adj), _dp(adj_c), _dp(img), _dp(scratch), nbytes, _stream()))
    return loss, adj, adj_c, img


# ------------------------------------------------------------------------------------------ MPC controller (A23b)
def controller_schedule(W, n_frames, frame_dt, omega, amplitude=1.0):
    """W [E, M, N] cuda fp32 -> activation schedule [F, E, M] (the array Model.set_actuation takes)."""
    torch = _torch()
    assert W.is_cuda and W.dtype == torch.float32 and W.is_contiguous() and W.ndim == 3
    E, M, N = W.shape
    act = torch.empty((int(n_frames), E, M), dtype=torch.float32, device=W.device)
    _check(lib().gs_controller_schedule(int(n_frames), E, M, N, float(omega), float(frame_dt), float(amplitude), _dp(W), _dp(act), _stream()))
    return act


def controller_grads(W, g_act, frame_dt, omega, amplitude=1.0):
    """dL/dW [E, M, N] from dL/dact [F, E, M] (what Model.actuation_grads returns)."""
    torch = _torch()
    E, M, N = W.shape
    F = int(g_act.shape[0])
    g_W = torch.empty_like(W)
    _check(lib().gs_controller_grads(F, E, M, N, float(omega), float(frame_dt), float(amplitude), _dp(W), _dp(_st(g_act, (F, E, M))), _dp(g_W), _stream()))
    return g_W


RASTER_STATIC_BYTES = 8 << 20  # GS_RASTER_STATIC_BYTES


def loss_silhouette_static(x, tris, cam, target, loss, adj=None, image=None, scale=None, accumulate=False):
    """gs_loss_silhouette_static: as loss_silhouette, with the scratch in the library's static device array.  Nothing is
    allocated, here either: the caller passes every output (loss [E]; adj [E, N, 3] and image [E, H, W] optional)."""
    torch = _torch()
    E, N, _ = x.shape
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
    assert tris.is_cuda and tris.dtype == torch.int32 and tris.is_contiguous() and tris.ndim == 2 and tris.shape[1] == 3
    scale = 1.0 / (cam.width * cam.height) if scale is None else float(scale)
    _check(lib().gs_loss_silhouette_static(E, N, _dp(x), int(tris.shape[0]), _dp(tris), C.byref(cam), _dp(_st(target, (E, cam.height, cam.width))), scale,
                                           int(accumulate), _dp(_st(loss, (E,))), _dp(adj if adj is None else _st(adj, (E, N, 3))),
                                           _dp(image if image is None else _st(image, (E, cam.height, cam.width))), _stream()))
    return loss, adj, image
