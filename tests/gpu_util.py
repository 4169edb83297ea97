"""Drives the CUDA path (through the C ABI binding) over a whole scene, mirroring oracle.run_scene's
outputs so the parity tests can compare key by key.  Imports nothing from oracle/."""
import numpy as np
import torch

from paper_2104_02646_b200 import gradsim as gs

DEV = "cuda:0"


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(np.asarray(a, dtype=np.float32)), device=DEV)


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def rel_inf(a, b):
    """||a - b||_inf / ||b||_inf per array (reading A18)."""
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    den = np.abs(b).max() if b.size else 0.0
    if den == 0.0:
        return float(np.abs(a).max()) if a.size else 0.0
    return float(np.abs(a - b).max() / den)


def gpu_run_scene(sc, target, K=None, plan=gs.GS_PLAN_AUTO, model=None):
    """rollout + loss + backward on the GPU.  target: as oracle.truth_targets(sc) returns
    (final_centroid [E,3]; pos_mse_frames [n_t,E,N,3]; centroid_traj [n_t,E,3]), fp64 numpy."""
    m = gs.Model(sc, plan=plan) if model is None else model
    m.request_grads("gravity")  # off by default (gradsim.h, GS_GRAVITY)
    K = sc.checkpoint_every if K is None else K
    T, s = sc.n_substeps, sc.frame_stride
    tape = m.tape(T, K)
    act = getattr(sc, "act", None)  # optional activation schedule: dict(stride=, tet=[F,E,M] or None, hinge=[F,E,Mh] or None)
    if act:
        F = next(a.shape[0] for a in (act.get("tet"), act.get("hinge")) if a is not None)
        m.actuation(F, act["stride"])
        for kind in ("tet", "hinge"):
            if act.get(kind) is not None:
                m.set_actuation(kind, dev(act[kind]))
    m.zero_grads()
    xT, vT = tape.rollout(dev(sc.x0), dev(sc.v0))
    lt = sc.loss_times()
    E, N = m.E, m.N
    out = {}
    if sc.loss == "final_centroid":
        loss, adj = gs.loss_centroid(xT, dev(target))
        ax0, av0 = tape.backward(adj_x_T=adj)
        rec = [xT]
    else:
        n_t = len(lt)
        frames_t = [t for t in lt if t % s == 0 and t // s >= 1]
        assert frames_t == [(k + 1) * s for k in range(len(frames_t))]
        cot = torch.zeros((len(frames_t), E, N, 3), dtype=torch.float32, device=DEV)
        loss = torch.zeros(E, dtype=torch.float32, device=DEV)
        rec = []
        adj_T = None
        tgt = dev(target)
        for k, t in enumerate(lt):
            xt = xT if t == T else tape.read(t, want_v=False)[0]
            rec.append(xt)
            if sc.loss == "pos_mse_frames":
                _, a = gs.loss_pos(xt, tgt[k], scale=1.0 / (n_t * N), loss=loss, accumulate=True)
            else:
                _, a = gs.loss_centroid(xt, tgt[k], scale=1.0 / n_t, loss=loss, accumulate=True)
            if t in frames_t:
                cot[frames_t.index(t)] = a
            else:
                adj_T = a
        ax0, av0 = tape.backward(adj_x_T=adj_T, adj_x_frames=cot if len(frames_t) else None, frame_stride=s)
    bad = m.check_finite()
    out.update(xT=host(xT), vT=host(vT), loss=host(loss), adj_x0=host(ax0), adj_v0=host(av0), bad=bad,
               rec_x=np.stack([host(r) for r in rec]))
    for g in gs.GROUPS:
        if g == "wind" or (g == "hinge_theta0" and not m.act_frames):
            continue  # read from the hinge actuation gradients: needs a schedule (gradsim.h, GS_HINGE_THETA0)
        out["g_" + g] = host(m.param_grads(g))
    if act:
        out["g_act_tet"], out["g_act_hinge"] = host(m.actuation_grads("tet")), host(m.actuation_grads("hinge"))
    out["model"] = m
    return out
