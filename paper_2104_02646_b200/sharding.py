"""Multi-GPU: the batched-environment axis is the only axis of the path that shards without a per-substep exchange
(SURVEY.md 8(e)).  One process per GPU; every rank owns a contiguous block of environments,
runs its rollouts independently (no data-path collective) and the per-environment results (loss, 3 parameter
gradients per environment, ...) are gathered once at the end.

Host-side logic only -- no arithmetic of the method.  Works with any torch.distributed backend (nccl on GPUs,
gloo in the CPU tests).
"""
from __future__ import annotations

import copy

import numpy as np

# per-environment arrays of a scene (leading axis E)
_ENV_FIELDS = ("x0", "v0", "mass", "tet_mu", "tet_lambda", "tet_damp", "tri_mu", "tri_lambda", "tri_damp", "ke", "kd", "kf", "mu_c", "k_drag", "k_lift")


def env_block(n_envs: int, world: int, rank: int) -> tuple[int, int]:
    """[lo, hi) of the environments rank `rank` owns: contiguous blocks, sizes differ by at most one, the first
    n_envs % world ranks take the larger blocks.  Ranks beyond n_envs get an empty block."""
    if not (0 <= rank < world):
        raise ValueError(f"rank {rank} outside world of {world}")
    base, extra = divmod(int(n_envs), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_scene(sc, world: int, rank: int):
    """The scene restricted to this rank's environments (shares the mesh, slices every [E, ...] array).
    Returns None when the rank owns no environment."""
    lo, hi = env_block(sc.n_envs, world, rank)
    if hi == lo:
        return None
    s = copy.copy(sc)
    s.n_envs = hi - lo
    for k in _ENV_FIELDS:
        a = getattr(sc, k)
        if a.shape[0] == sc.n_envs:
            setattr(s, k, np.ascontiguousarray(a[lo:hi]))
    if getattr(sc, "truth", None):
        s.truth = {k: (v[lo:hi] if v.shape[0] == sc.n_envs else v) for k, v in sc.truth.items()}
    tgt = getattr(sc, "target", None)
    if tgt is not None:
        t = np.asarray(tgt)
        # final_centroid targets are [E, 3]; frame targets are [n_t, E, ...]
        s.target = t[lo:hi] if t.shape[0] == sc.n_envs and t.ndim == 2 else (t[:, lo:hi] if t.ndim >= 3 and t.shape[1] == sc.n_envs else t)
    return s


def gather_env_rows(local, n_envs: int, dist=None):
    """All ranks' per-environment rows ([E_local, k] torch tensor, env order) -> [n_envs, k] on every rank.
    One all_gather of padded blocks at the end of a job; `dist` defaults to torch.distributed."""
    import torch

    if dist is None:
        import torch.distributed as dist
    world, rank = dist.get_world_size(), dist.get_rank()
    k = local.shape[1:]
    cap = -(-n_envs // world)  # largest block
    pad = torch.zeros((cap,) + tuple(k), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    rows = []
    for r in range(world):
        lo, hi = env_block(n_envs, world, r)
        rows.append(parts[r][: hi - lo])
    out = torch.cat(rows, 0)
    assert out.shape[0] == n_envs and env_block(n_envs, world, rank)[1] - env_block(n_envs, world, rank)[0] == local.shape[0]
    return out
