"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is the ONLY code shared by the fp64 oracle (``oracle/``) and the CUDA
path (``paper_2104_02646_b200/csrc``).  It holds mesh topology and random draws
only -- none of the method's arithmetic (no B matrices, no forces, no energies):
both sides derive every rest-shape quantity from ``x_rest`` themselves.

Recipe (readings A9, A12-A17, A19):
numpy ``default_rng([1000 + config, stream])``, every array rounded to fp32 once
and the rounded values handed to both sides.

The paper's own meshes (beams, gear, cloth instances, PAPER.md:279, 364, 377,
468-474) are not available; these structured blocks / sheets stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

STREAMS = {"truth": 1, "guess": 2, "target": 3, "v0": 4, "misc": 5}


def rng_for(config: int, stream: str, salt: int = 0) -> np.random.Generator:
    return np.random.default_rng([1000 + config, STREAMS[stream], salt])


# ----------------------------------------------------------------------------
# topology
# ----------------------------------------------------------------------------
# hex corner numbering v0..v7 = (000,100,110,010,001,101,111,011)  (reading A12)
_HEX_CORNERS = np.array(
    [(0, 0, 0), (1, 0, 0), (1, 1, 0), (0, 1, 0), (0, 0, 1), (1, 0, 1), (1, 1, 1), (0, 1, 1)],
    dtype=np.int64,
)
_TETS_EVEN = np.array([(0, 1, 3, 4), (1, 2, 3, 6), (1, 4, 5, 6), (3, 4, 6, 7), (1, 3, 4, 6)])
_TETS_ODD = np.array([(0, 1, 2, 5), (0, 2, 3, 7), (0, 4, 5, 7), (2, 5, 6, 7), (0, 2, 5, 7)])


def hex_grid_tets(nx: int, ny: int, nz: int, h: float, origin=(0.0, 0.0, 0.0)):
    """nx*ny*nz hex cells of edge h, each split into 5 tets with alternating parity.

    Returns (x [N,3] float64, tets [M,4] int32).  Orientation is NOT fixed here;
    consumers validate det(D_m) > 0 and swap two vertices where needed (A12).
    Vertex id = (k*(ny+1) + j)*(nx+1) + i   (x fastest).
    """
    i, j, k = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), np.arange(nz + 1), indexing="ij")
    vid = (k * (ny + 1) + j) * (nx + 1) + i  # [nx+1, ny+1, nz+1]
    n = (nx + 1) * (ny + 1) * (nz + 1)
    x = np.zeros((n, 3))
    x[vid.ravel(), 0] = origin[0] + h * i.ravel()
    x[vid.ravel(), 1] = origin[1] + h * j.ravel()
    x[vid.ravel(), 2] = origin[2] + h * k.ravel()

    ci, cj, ck = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    ci, cj, ck = ci.ravel(), cj.ravel(), ck.ravel()
    # sort cells x-fastest so the caller's element order is the natural grid order
    order = np.lexsort((ci, cj, ck))
    ci, cj, ck = ci[order], cj[order], ck[order]
    corners = vid[
        ci[:, None] + _HEX_CORNERS[None, :, 0],
        cj[:, None] + _HEX_CORNERS[None, :, 1],
        ck[:, None] + _HEX_CORNERS[None, :, 2],
    ]  # [cells, 8]
    even = ((ci + cj + ck) % 2) == 0
    pat = np.where(even[:, None, None], _TETS_EVEN[None], _TETS_ODD[None])  # [cells,5,4]
    tets = np.take_along_axis(corners[:, None, :].repeat(5, 1), pat, axis=2).reshape(-1, 4)
    # orient positively (signed volume > 0) by swapping the last two vertices
    d = x[tets[:, 1:]] - x[tets[:, :1]]
    neg = np.linalg.det(d) < 0  # topology/orientation bookkeeping, not the method
    tets[neg, 2], tets[neg, 3] = tets[neg, 3].copy(), tets[neg, 2].copy()
    return x, tets.astype(np.int32)


def cloth_grid(n: int, m: int, h: float, origin=(0.0, 0.0, 0.0)):
    """n x m particle sheet in the xz-plane at height origin[1]; diagonal alternates
    with (i+j) parity (A13).  Vertex id = j*n + i.  Triangles are wound so that the
    face normal is +y.  Returns (x [N,3], tris [Mt,3] int32, hinges [Mh,4] int32)
    with hinge = (wing1, wing2, edge_a, edge_b), edge oriented as in its first triangle.
    """
    i, j = np.meshgrid(np.arange(n), np.arange(m), indexing="ij")
    vid = j * n + i
    x = np.zeros((n * m, 3))
    x[vid.ravel(), 0] = origin[0] + h * i.ravel()
    x[vid.ravel(), 1] = origin[1]
    x[vid.ravel(), 2] = origin[2] + h * j.ravel()
    tris = []
    for jj in range(m - 1):
        for ii in range(n - 1):
            a, b = jj * n + ii, jj * n + ii + 1
            c, d = (jj + 1) * n + ii + 1, (jj + 1) * n + ii
            # +y normal needs (z, x) orientation: a -> d -> c -> b is counter-clockwise seen from +y
            if (ii + jj) % 2 == 0:
                tris += [(a, d, c), (a, c, b)]
            else:
                tris += [(a, d, b), (b, d, c)]
    tris = np.asarray(tris, dtype=np.int32).reshape(-1, 3)
    return x, tris, hinges_from_tris(tris)


def hinges_from_tris(tris: np.ndarray) -> np.ndarray:
    """Interior edges shared by exactly two triangles -> (wing1, wing2, a, b)."""
    first = {}
    out = []
    for t, (p, q, r) in enumerate(np.asarray(tris).tolist()):
        for a, b, c in ((p, q, r), (q, r, p), (r, p, q)):
            key = (a, b) if a < b else (b, a)
            if key in first:
                a1, b1, c1 = first[key]
                out.append((c1, c, a1, b1))
            else:
                first[key] = (a, b, c)
    return np.asarray(out, dtype=np.int32).reshape(-1, 4)



def boundary_faces(tets: np.ndarray) -> np.ndarray:
    """Triangles of a tet mesh that belong to exactly one tet: the surface the rasteriser draws for a solid
    (include/gradsim.h, gs_render_silhouette: "the boundary faces of a tet mesh").  Topology only; [F,3] int32, in the
    order of first appearance, each face in the vertex order of its tet."""
    count, faces = {}, []
    for a, b, c, d in np.asarray(tets).tolist():
        for f in ((b, c, d), (a, d, c), (a, b, d), (a, c, b)):
            key = tuple(sorted(f))
            if key not in count:
                count[key] = 0
                faces.append((key, f))
            count[key] += 1
    return np.asarray([f for key, f in faces if count[key] == 1], dtype=np.int32).reshape(-1, 3)

# ----------------------------------------------------------------------------
# scene container
# ----------------------------------------------------------------------------
@dataclass
class Scene:
    name: str
    config: int
    n_envs: int
    x_rest: np.ndarray  # [N,3] f32
    x0: np.ndarray  # [E,N,3] f32
    v0: np.ndarray  # [E,N,3] f32
    mass: np.ndarray  # [E,N] f32
    pinned: np.ndarray  # [N] u8
    tets: np.ndarray  # [M,4] i32
    tet_mu: np.ndarray  # [E,M] f32
    tet_lambda: np.ndarray
    tet_damp: np.ndarray
    tris: np.ndarray  # [Mt,3]
    tri_mu: np.ndarray  # [E,Mt]
    tri_lambda: np.ndarray
    tri_damp: np.ndarray
    hinges: np.ndarray  # [Mh,4]
    hinge_kb: np.ndarray  # [Mh]
    ke: np.ndarray  # [E]
    kd: np.ndarray
    kf: np.ndarray
    mu_c: np.ndarray
    gravity: tuple = (0.0, -9.8, 0.0)
    dt: float = 1.0 / 1920.0
    plane_n: tuple = (0.0, 1.0, 0.0)
    plane_d: float = 0.0
    radius: float = 0.0
    n_substeps: int = 0
    checkpoint_every: int = 1  # 1 = full tape
    frame_stride: int = 32
    loss: str = "final_centroid"  # | "pos_mse_frames" | "centroid_traj"
    target: Optional[np.ndarray] = None  # final_centroid: [E,3]
    truth: dict = field(default_factory=dict)  # truth-stream parameters (configs 2, 3)
    k_drag: Optional[np.ndarray] = None  # [E] lift / drag of the air on the cloth faces (A21); None = zeros
    k_lift: Optional[np.ndarray] = None  # [E]
    wind: tuple = (0.0, 0.0, 0.0)
    act: Optional[dict] = None  # activation schedule: dict(stride=, tet=[F,E,M] or None, hinge=[F,E,Mh] or None)

    def __post_init__(self):
        if self.k_drag is None:
            self.k_drag = np.zeros(self.n_envs, np.float32)
        if self.k_lift is None:
            self.k_lift = np.zeros(self.n_envs, np.float32)

    @property
    def n_particles(self):
        return self.x_rest.shape[0]

    @property
    def n_elements(self):
        return self.tets.shape[0] + self.tris.shape[0] + self.hinges.shape[0]

    def extent(self) -> float:
        """Bounding-box diagonal of the initial scene (reading A18)."""
        lo = self.x0.reshape(-1, 3).min(0).astype(np.float64)
        hi = self.x0.reshape(-1, 3).max(0).astype(np.float64)
        return float(np.sqrt(((hi - lo) ** 2).sum()))

    def loss_times(self):
        """Substep indices t (state AFTER t substeps) at which the loss reads x."""
        T, s = self.n_substeps, self.frame_stride
        if self.loss == "final_centroid":
            return [T]
        times = list(range(s, T + 1, s))
        if self.loss == "pos_mse_frames" and (not times or times[-1] != T):
            times.append(T)
        return times


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _empty_elems():
    z = np.zeros((0,), np.float32)
    return dict(
        tets=np.zeros((0, 4), np.int32),
        tris=np.zeros((0, 3), np.int32),
        hinges=np.zeros((0, 4), np.int32),
        hinge_kb=z,
    )


def _contact(E, mu_c=0.5, ke=1e4, kd=10.0, kf=50.0):
    one = np.ones(E, np.float32)
    return dict(ke=_f32(ke * one), kd=_f32(kd * one), kf=_f32(kf * one), mu_c=_f32(mu_c * one))


def _bcast(E, n, val):
    return _f32(np.broadcast_to(np.asarray(val, np.float64), (E, n)))


def _final_centroid_target(config, x0):
    r = rng_for(config, "target")
    c0 = x0.astype(np.float64).mean(axis=1)  # [E,3]
    E = x0.shape[0]
    off = np.stack(
        [r.uniform(-0.2, 0.2, E), -r.uniform(0.2, 0.5, E), r.uniform(-0.2, 0.2, E)], axis=1
    )
    return _f32(c0 + off)


def _final_position_target(config, x0):
    """Seeded smooth, non-uniform per-particle target x_i* = x_i(0) + offset(x_i(0)) for the final-state
    position loss (shape [1,E,N,3]: one loss time).  A uniform offset would leave the gradient with respect to
    the elastic parameters of a free body at zero (momentum conservation), hence the spatial variation."""
    r = rng_for(config, "target")
    x = x0.astype(np.float64)
    a, b, c = r.uniform(0.02, 0.05, 3)
    k1, k2 = r.uniform(3.0, 6.0, 2)
    off = np.stack([a * np.sin(k1 * x[..., 2]), -0.05 - b * (1.0 + np.cos(k2 * x[..., 0])), c * np.cos(k1 * x[..., 0] + k2 * x[..., 2])], -1)
    return _f32((x + off)[None])


def box_scene(config=0, cells=(4, 4, 4), h=0.1, y0=0.5, n_substeps=1920, n_envs=1, origin_xz=(0.0, 0.0)):
    """Config 0: Neo-Hookean box dropped on the ground (BASELINE.json configs[0])."""
    nx, ny, nz = cells
    x, tets = hex_grid_tets(nx, ny, nz, h, origin=(origin_xz[0], y0, origin_xz[1]))
    N, M, E = x.shape[0], tets.shape[0], n_envs
    x = _f32(x)
    x0 = np.ascontiguousarray(np.broadcast_to(x, (E, N, 3))).copy()
    e = _empty_elems()
    z = np.zeros((E, 0), np.float32)
    sc = Scene(
        name=f"config{config}-box{nx}x{ny}x{nz}",
        config=config,
        n_envs=E,
        x_rest=x,
        x0=x0,
        v0=np.zeros_like(x0),
        mass=_bcast(E, N, 0.1),
        pinned=np.zeros(N, np.uint8),
        tets=tets,
        tet_mu=_bcast(E, M, 1e4),
        tet_lambda=_bcast(E, M, 1e4),
        tet_damp=_bcast(E, M, 1.0),
        tris=e["tris"],
        tri_mu=z,
        tri_lambda=z,
        tri_damp=z,
        hinges=e["hinges"],
        hinge_kb=e["hinge_kb"],
        n_substeps=n_substeps,
        loss="final_centroid",
        **_contact(E),
    )
    sc.target = _final_centroid_target(config, sc.x0)
    return sc


CLOTH_MASS = 0.1  # kg per particle (reading A15: lighter cloth makes the stick branch of friction unstable at this dt)


def cloth_scene(config=1, n=32, h=0.01, y0=0.02, n_substeps=512, pins=True, origin_xz=(0.0, 0.0)):
    """Config 1: cloth sheet, two corners pinned, seeded initial velocity (A15)."""
    x, tris, hinges = cloth_grid(n, n, h, origin=(origin_xz[0], y0, origin_xz[1]))
    N, Mt, Mh, E = x.shape[0], tris.shape[0], hinges.shape[0], 1
    x = _f32(x)
    pinned = np.zeros(N, np.uint8)
    if pins:
        pinned[0] = 1  # (i=0, j=0)
        pinned[(n - 1) * n] = 1  # (i=0, j=n-1)
    v0 = rng_for(config, "v0").normal(0.0, 0.01, size=(E, N, 3))
    v0[:, pinned.astype(bool)] = 0.0
    z = np.zeros((E, 0), np.float32)
    sc = Scene(
        name=f"config{config}-cloth{n}x{n}",
        config=config,
        n_envs=E,
        x_rest=x,
        x0=x[None].copy(),
        v0=_f32(v0),
        mass=_bcast(E, N, CLOTH_MASS),
        pinned=pinned,
        tets=np.zeros((0, 4), np.int32),
        tet_mu=z,
        tet_lambda=z,
        tet_damp=z,
        tris=tris,
        tri_mu=_bcast(E, Mt, 1e3),
        tri_lambda=_bcast(E, Mt, 1e3),
        tri_damp=_bcast(E, Mt, 1.0),
        hinges=hinges,
        hinge_kb=_f32(np.full(Mh, 10.0)),
        n_substeps=n_substeps,
        loss="final_centroid",
        **_contact(E),
    )
    sc.target = _final_centroid_target(config, sc.x0)
    return sc


def hetero_solid_scene(config=2, cells=(20, 10, 20), h=0.1, y0=0.1, n_substeps=2000, checkpoint_every=32):
    """Config 2: heterogeneous soft solid; per-tet lognormal mu, lambda; truth = second draw."""
    nx, ny, nz = cells
    x, tets = hex_grid_tets(nx, ny, nz, h, origin=(0.0, y0, 0.0))
    N, M, E = x.shape[0], tets.shape[0], 1
    x = _f32(x)
    g, t = rng_for(config, "guess"), rng_for(config, "truth")
    ln = np.log(1e4)
    mu_c = g.uniform(0.1, 0.9)
    z = np.zeros((E, 0), np.float32)
    e = _empty_elems()
    sc = Scene(
        name=f"config{config}-hetero{nx}x{ny}x{nz}",
        config=config,
        n_envs=E,
        x_rest=x,
        x0=x[None].copy(),
        v0=np.zeros((E, N, 3), np.float32),
        mass=_bcast(E, N, 0.1),
        pinned=np.zeros(N, np.uint8),
        tets=tets,
        tet_mu=_f32(g.lognormal(ln, 0.5, size=(E, M))),
        tet_lambda=_f32(g.lognormal(ln, 0.5, size=(E, M))),
        tet_damp=_bcast(E, M, 1.0),
        tris=e["tris"],
        tri_mu=z,
        tri_lambda=z,
        tri_damp=z,
        hinges=e["hinges"],
        hinge_kb=e["hinge_kb"],
        n_substeps=n_substeps,
        checkpoint_every=checkpoint_every,
        loss="pos_mse_frames",
        **_contact(E, mu_c=mu_c),
    )
    sc.truth = dict(
        tet_mu=_f32(t.lognormal(ln, 0.5, size=(E, M))), tet_lambda=_f32(t.lognormal(ln, 0.5, size=(E, M)))
    )
    return sc


def batched_sysid_scene(config=3, n_envs=1024, cells=(4, 4, 4), n_substeps=1920, y0=0.5):
    """Config 3: E copies of config 0's mesh, per-env mu, lambda, mass, mu_c; truth = second draw."""
    sc = box_scene(config=config, cells=cells, n_substeps=n_substeps, n_envs=n_envs, y0=y0)
    E, N, M = n_envs, sc.n_particles, sc.tets.shape[0]

    def draw(r):
        return dict(
            tet_mu=_f32(np.repeat(r.uniform(5e3, 5e4, (E, 1)), M, 1)),
            tet_lambda=_f32(np.repeat(r.uniform(5e3, 5e4, (E, 1)), M, 1)),
            mass=_f32(np.repeat(r.uniform(0.05, 0.2, (E, 1)), N, 1)),
            mu_c=_f32(r.uniform(0.1, 0.9, E)),
        )

    gd, td = draw(rng_for(config, "guess")), draw(rng_for(config, "truth"))
    sc.tet_mu, sc.tet_lambda, sc.mass, sc.mu_c = gd["tet_mu"], gd["tet_lambda"], gd["mass"], gd["mu_c"]
    sc.truth = td
    sc.name = f"config{config}-sysid-E{E}"
    sc.loss = "centroid_traj"
    sc.target = None
    return sc


def large_scene(config=4, solid_cells=(100, 20, 100), cloth_n=512, n_substeps=256):
    """Config 4: big homogeneous solid + big cloth sheet beside it, ground contact only (A16)."""
    nx, ny, nz = solid_cells
    xs, tets = hex_grid_tets(nx, ny, nz, 0.1, origin=(0.0, 0.02, 0.0))
    xc, tris, hinges = cloth_grid(cloth_n, cloth_n, 0.01, origin=(nx * 0.1 + 0.5, 0.02, 0.0))
    Ns = xs.shape[0]
    x = _f32(np.concatenate([xs, xc], 0))
    tris = (tris + Ns).astype(np.int32)
    hinges = (hinges + Ns).astype(np.int32)
    N, M, Mt, Mh, E = x.shape[0], tets.shape[0], tris.shape[0], hinges.shape[0], 1
    mass = np.concatenate([np.full(Ns, 0.1), np.full(N - Ns, CLOTH_MASS)])
    v0 = np.zeros((E, N, 3))
    # sigma = 0.1 m/s: with 0.01 the free sheet barely strains and its membrane gradients sit at the fp32 noise floor
    v0[:, Ns:] = rng_for(config, "v0").normal(0.0, 0.1, size=(E, N - Ns, 3))
    sc = Scene(
        name=f"config{config}-large-{M}tets-{Mt}tris",
        config=config,
        n_envs=E,
        x_rest=x,
        x0=x[None].copy(),
        v0=_f32(v0),
        mass=_f32(mass[None]),
        pinned=np.zeros(N, np.uint8),
        tets=tets,
        tet_mu=_bcast(E, M, 2e4),
        tet_lambda=_bcast(E, M, 2e4),
        tet_damp=_bcast(E, M, 1.0),
        tris=tris,
        tri_mu=_bcast(E, Mt, 1e3),
        tri_lambda=_bcast(E, Mt, 1e3),
        tri_damp=_bcast(E, Mt, 1.0),
        hinges=hinges,
        hinge_kb=_f32(np.full(Mh, 10.0)),
        n_substeps=n_substeps,
        loss="pos_mse_frames",  # one loss time, t = T: L = 1/N sum_i |x_i(T) - x_i*|^2
        frame_stride=n_substeps,
        **_contact(E),
    )
    sc.target = _final_position_target(config, sc.x0)
    return sc


def make_scene(config: int, small: bool = False) -> Scene:
    """BASELINE.json configs[config]; ``small=True`` gives a reduced variant with the same
    structure (several tiles + a ragged tail) that the oracle finishes in seconds.  The small variants
    start 2 cm above the ground so that the impact (substep ~123) falls inside their shorter rollouts."""
    if config == 0:
        return box_scene(n_substeps=256, y0=0.02) if small else box_scene()
    if config == 1:
        return cloth_scene(n=12, n_substeps=128) if small else cloth_scene()
    if config == 2:
        if small:
            return hetero_solid_scene(cells=(7, 3, 5), y0=0.02, n_substeps=420, checkpoint_every=32)
        return hetero_solid_scene()
    if config == 3:
        return batched_sysid_scene(n_envs=5, n_substeps=224, y0=0.02) if small else batched_sysid_scene()
    if config == 4:
        if small:
            return large_scene(solid_cells=(9, 3, 7), cloth_n=23, n_substeps=224)
        return large_scene()
    raise ValueError(f"unknown config {config}")


def perturbed_state(sc: Scene, amp_x=0.1, amp_v=0.5, seed=0):
    """A seeded deformed state near x0 (relative to the smallest rest edge) for one-substep
    parity tests, so that every force term is non-trivial.  Returns (x [E,N,3], v [E,N,3]) f32."""
    r = rng_for(sc.config, "misc", seed)
    edges = []
    for arr in (sc.tets, sc.tris):
        if arr.shape[0]:
            edges.append(np.linalg.norm(sc.x_rest[arr[:, 0]] - sc.x_rest[arr[:, 1]], axis=1).min())
    h = float(min(edges)) if edges else 1.0
    x = sc.x0.astype(np.float64) + amp_x * h * r.uniform(-1, 1, sc.x0.shape)
    v = sc.v0.astype(np.float64) + amp_v * r.uniform(-1, 1, sc.v0.shape)
    # push part of the scene through the ground so both contact branches are hit
    y = x[..., 1]
    x[..., 1] -= (y.min() + 0.3 * h) if (y.max() - y.min()) > h else np.median(y)
    v[:, sc.pinned.astype(bool)] = 0.0
    return _f32(x), _f32(v)


def custom_scene(x, tets=None, tris=None, hinges=None, n_envs=1, mass=0.1, mu=1e4, lam=1e4, damp=1.0,
                 tri_mu=1e3, tri_lam=1e3, tri_damp=1.0, kb=10.0, pinned=None, v0=None, x0=None, gravity=(0.0, -9.8, 0.0),
                 dt=1.0 / 1920.0, ke=1e4, kd=10.0, kf=50.0, mu_c=0.5, n_substeps=1, checkpoint_every=1,
                 plane_n=(0.0, 1.0, 0.0), plane_d=0.0, radius=0.0, name="custom", config=9, k_drag=0.0, k_lift=0.0, wind=(0.0, 0.0, 0.0)):
    """Free-form scene for unit tests.  Scalars broadcast; arrays are taken as given ([E,n] or [n])."""
    x = _f32(x)
    N, E = x.shape[0], n_envs
    tets = np.zeros((0, 4), np.int32) if tets is None else np.asarray(tets, np.int32).reshape(-1, 4)
    tris = np.zeros((0, 3), np.int32) if tris is None else np.asarray(tris, np.int32).reshape(-1, 3)
    if hinges is None:
        hinges = hinges_from_tris(tris) if tris.shape[0] else np.zeros((0, 4), np.int32)
    hinges = np.asarray(hinges, np.int32).reshape(-1, 4)
    M, Mt, Mh = tets.shape[0], tris.shape[0], hinges.shape[0]

    def en(val, n):
        a = np.asarray(val, np.float64)
        if a.ndim == 0:
            return _bcast(E, n, float(a))
        return _f32(np.broadcast_to(a.reshape(-1, n) if n else np.zeros((E, 0)), (E, n)))

    def e1(val):
        return _f32(np.broadcast_to(np.asarray(val, np.float64).ravel(), (E,)))

    x0 = np.broadcast_to(x, (E, N, 3)).copy() if x0 is None else _f32(x0).reshape(E, N, 3)
    v0 = np.zeros((E, N, 3), np.float32) if v0 is None else _f32(v0).reshape(E, N, 3)
    sc = Scene(
        name=name, config=config, n_envs=E, x_rest=x, x0=_f32(x0), v0=v0, mass=en(mass, N),
        pinned=np.zeros(N, np.uint8) if pinned is None else np.asarray(pinned, np.uint8),
        tets=tets, tet_mu=en(mu, M), tet_lambda=en(lam, M), tet_damp=en(damp, M),
        tris=tris, tri_mu=en(tri_mu, Mt), tri_lambda=en(tri_lam, Mt), tri_damp=en(tri_damp, Mt),
        hinges=hinges, hinge_kb=_f32(np.broadcast_to(np.asarray(kb, np.float64).ravel(), (Mh,))),
        ke=e1(ke), kd=e1(kd), kf=e1(kf), mu_c=e1(mu_c), gravity=tuple(gravity), dt=dt, plane_n=tuple(plane_n),
        plane_d=plane_d, radius=radius, n_substeps=n_substeps, checkpoint_every=checkpoint_every,
        k_drag=e1(k_drag), k_lift=e1(k_lift), wind=tuple(wind),
    )
    sc.target = _final_centroid_target(config, sc.x0)
    return sc
