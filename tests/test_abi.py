"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol include/gradsim.h
declares; the Python binding declares a signature for each of them.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

from paper_2104_02646_b200 import build as gs_build
from paper_2104_02646_b200 import gradsim as gs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gradsim.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gs_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    return gs_build.build()


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for need in ("gs_model_create", "gs_step_forward", "gs_step_backward", "gs_rollout", "gs_rollout_backward", "gs_param_grads"):
        assert need in names


def test_library_exports_every_declared_symbol(lib_path):
    L = C.CDLL(lib_path)
    for name in _declared():
        assert hasattr(L, name), f"{name} declared in gradsim.h but not exported"


def test_binding_covers_every_declared_symbol(lib_path):
    assert sorted(gs.SIGNATURES) == _declared()
    L = gs.lib()
    assert L.gs_version().decode().startswith("gradsim-b200")
    assert L.gs_launch_count() >= 0


def test_desc_struct_matches_header_field_order():
    src = open(os.path.join(ROOT, "include", "gradsim.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} gs_model_desc;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(int32_t|uint32_t|uint8_t|float)\s*", "", decl)
        for part in decl.split(","):
            fields.append(re.sub(r"[\*\s]|\[\d+\]", "", part))
    assert fields == [f[0] for f in gs.gs_model_desc._fields_]


def _struct_fields(name):
    src = open(os.path.join(ROOT, "include", "gradsim.h")).read()
    body = re.search(r"typedef struct \{((?:(?!typedef struct).)*?)\} %s;" % name, src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        ctype = re.match(r"(const\s+)?(int32_t|uint32_t|uint8_t|float)", decl).group(2)
        decl = re.sub(r"^(const\s+)?(int32_t|uint32_t|uint8_t|float)\s*", "", decl)
        for part in decl.split(","):
            dim = re.search(r"\[(\d+)\]", part)
            fields.append((re.sub(r"[\*\s]|\[\d+\]", "", part), ctype, int(dim.group(1)) if dim else 0))
    return fields


@pytest.mark.parametrize("name,cls", [("gs_camera", gs.gs_camera), ("gs_shading", gs.gs_shading)])
def test_host_structs_of_the_rasteriser_match_the_header(name, cls):
    """field order, scalar type and array length of the HOST structs the rasteriser calls read"""
    ctype = {"float": C.c_float, "int32_t": C.c_int32}
    want = [(n, ctype[t] * d if d else ctype[t]) for n, t, d in _struct_fields(name)]
    assert [(f[0], f[1]) for f in cls._fields_] == want
    assert C.sizeof(cls) == sum(C.sizeof(t) for _, t in want)  # no padding: all members are 4-byte scalars


def test_param_group_enum_matches_binding():
    src = open(os.path.join(ROOT, "include", "gradsim.h")).read()
    body = re.search(r"enum gs_param_group \{(.*?)\};", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    enum = {k: int(v) for k, v in re.findall(r"(GS_[A-Z0-9_]+)\s*=\s*(\d+)", body)}
    names = {"GS_TET_MU": "tet_mu", "GS_TET_LAMBDA": "tet_lambda", "GS_TET_DAMP": "tet_damp", "GS_TRI_MU": "tri_mu", "GS_TRI_LAMBDA": "tri_lambda",
             "GS_TRI_DAMP": "tri_damp", "GS_MASS": "mass", "GS_HINGE_KB": "hinge_kb", "GS_CONTACT_KE": "ke", "GS_CONTACT_KD": "kd",
             "GS_CONTACT_KF": "kf", "GS_CONTACT_MUC": "mu_c", "GS_GRAVITY": "gravity", "GS_HINGE_THETA0": "hinge_theta0", "GS_AERO_DRAG": "k_drag", "GS_AERO_LIFT": "k_lift", "GS_WIND": "wind"}
    assert enum.pop("GS_NUM_GROUPS") == len(gs.GROUPS) == len(names)
    assert {names[k]: v for k, v in enum.items()} == gs.GROUPS


def test_argument_errors_without_a_device(lib_path):
    """Pure host-side argument checks return codes instead of crashing (no CUDA call is reached)."""
    L = gs.lib()
    assert L.gs_model_workspace_bytes(None) == 0
    out = C.c_void_p()
    assert L.gs_model_create(None, None, 0, None, C.byref(out)) == gs.GS_EINVAL
    assert b"desc" in L.gs_last_error()
    assert L.gs_tape_bytes(None, 10, 1) == 0
    assert L.gs_zero_grads(None, None) == gs.GS_EINVAL
    # rasteriser colour channel and controller: sizes and null arguments are rejected before any launch
    assert L.gs_raster_rgb_scratch_bytes(0, 10, 10) == 0 and L.gs_raster_rgb_scratch_bytes(2, 10, 0) > 0
    assert L.gs_render_rgb(1, 3, None, 1, None, None, None, None, None, None, 0, None) == gs.GS_EINVAL
    assert L.gs_controller_schedule(0, 1, 1, 8, 1.0, 0.1, 1.0, None, None, None) == gs.GS_EINVAL
    assert b"controller" in L.gs_last_error()
    assert L.gs_controller_grads(4, 1, 1, 8, 1.0, -0.1, 1.0, None, None, None, None) == gs.GS_EINVAL
    assert L.gs_step_forward(None, None, None, None, None, None) == gs.GS_EINVAL
    d = gs.gs_model_desc()
    d.n_particles, d.n_envs = 0, 1
    assert L.gs_model_workspace_bytes(C.byref(d)) == 0
    # round-2 entry points: null handles / bad sizes come back as codes
    assert L.gs_actuation_bytes(None, 4) == 0
    assert L.gs_actuation_create(None, 4, 8, None, 0, None) == gs.GS_EINVAL
    assert L.gs_set_actuation(None, 0, None, None) == gs.GS_EINVAL
    assert L.gs_actuation_grads(None, 0, None, None) == gs.GS_EINVAL
    assert L.gs_set_actuation_frame(None, 0) == gs.GS_EINVAL
    assert L.gs_request_grads(None, gs.GROUPS["gravity"], 1) == gs.GS_EINVAL
    assert L.gs_set_deterministic(None, 1) == gs.GS_EINVAL
    assert L.gs_loss_centroid_traj(None, None, 1, None, None, None, None, None) == gs.GS_EINVAL
    assert L.gs_host_scratch_bytes(None, None, 0, 1) == 0
    assert L.gs_raster_scratch_bytes(0, 10, 3) == 0 and L.gs_raster_scratch_bytes(1, 10, 3) > 0
    cam = gs.make_camera([1, 0, 0, 0, 1, 0, 0, 0, 1], [0, 0, 1], 1.0, 1.0, 8, 8, 1e-3)
    assert L.gs_render_silhouette(1, 4, None, 0, None, C.byref(cam), None, None, 0, None) == gs.GS_EINVAL  # image is null
    assert L.gs_loss_silhouette(1, 4, None, 0, None, C.byref(cam), None, 1.0, 0, None, None, None, None, 0, None) == gs.GS_EINVAL


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2104_02646_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "gs_oracle" not in txt and "libgs_oracle" not in txt, f
