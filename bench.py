#!/usr/bin/env python
"""bench.py -- element-substeps/s of the gradSim hot path (forward and forward+adjoint) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference] [--shard-envs]

One "step" = one pass of the whole hot path over one batch of synthetic input: gs_rollout (T forward substeps writing
the on-device tape), the config's own loss at its loss times (SURVEY.md 8(c) "Losses"), and gs_rollout_backward (T adjoint
substeps + parameter gradients).  Default workload: BASELINE.json configs[4] (the 1M-tet + 512x512-cloth HBM stress case,
the largest single-GPU configuration); its line carries configs[3] (the 1024-environment batch, the other config
north_star names) as the sub-record "config3", measured in the same run.  --config 0..3 runs one of the others alone.

Prints ONE JSON line (rank 0): value = whole-job element-substeps/s for forward+adjoint, plus
  forward      : the same for gs_rollout alone
  e2e          : through gs_rollout_loss_backward_host with pinned HOST buffers (H2D/D2H inside the timed region), same loss
  roofline     : the dominant kernel's algorithmic bytes (or flops) / its CUDA-event duration vs MEASURED_PEAKS.json
  cpu_baseline : the fp64 oracle, as it stands, on a bounded sample of the same workload: all host cores and one thread
  clocks       : nvidia-smi samples taken during the timed region
N > 1 (torchrun): every rank runs an independent replica of the workload (replicas only, no
data-path collective); time = max over ranks.  --shard-envs splits the environments of a batched config over the ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "element-substeps/s (forward+adjoint)"
UNIT = "element-substeps/s"
HBM_FALLBACK_GBS = 6650.0  # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent

# SURVEY.md 8(d) / DESIGN.md "Algorithmic bytes": fp32, every array touched once per substep
BYTES_FWD = dict(tet=68, tri=44, hinge=28, particle=52)
BYTES_ADJ = dict(tet=92, tri=68, hinge=28, particle=96)
KERNELS = ["k_elements_fwd", "k_particles_fwd", "k_particles_adj", "k_elements_adj", "other", "k_resident_fwd", "k_resident_adj"]
# SURVEY.md 8(d) "Algorithmic flops" (fp32, counted from the 8(c) formulas): per tet / triangle / hinge / particle
FLOPS_FWD = dict(tet=420, tri=250, hinge=240, particle=60)
FLOPS_ADJ = dict(tet=1020, tri=650, hinge=800, particle=120)
# plain fp32 ALU peak: 148 SMs x 128 lanes x 2 flop x clocks.max.sm (1965 MHz)
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def substep_bytes(sc, table):
    E = sc.n_envs
    return E * (sc.tets.shape[0] * table["tet"] + sc.tris.shape[0] * table["tri"] + sc.hinges.shape[0] * table["hinge"]
                + sc.n_particles * table["particle"])


def substep_flops(sc, table):
    return substep_bytes(sc, table)  # same weighted sum, other table


def element_stream_bytes(sc, table):
    E = sc.n_envs
    return E * (sc.tets.shape[0] * table["tet"] + sc.tris.shape[0] * table["tri"] + sc.hinges.shape[0] * table["hinge"])


def resident_stream_bytes(sc, adjoint):
    """SURVEY.md 8(d) streaming byte model of a mesh that stays on chip (config 3): per environment-substep the state goes
    in and out once and the connectivity is shared by all environments -- forward N x 52 B + 3 material parameters,
    adjoint N x 96 B (125 x 52 + 12 = 6.5 KB and 125 x 96 = 12 KB per env-substep for config 3: 18.5 KB)."""
    return sc.n_envs * (sc.n_particles * BYTES_ADJ["particle"] if adjoint else sc.n_particles * BYTES_FWD["particle"] + 12)


# DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, copied from the ncu --set full
# captures summarised under profiles/ -- NOT measured by this run: "source" names the capture and the commit whose kernels
# it profiled; a kernel change after that commit makes the figure stale until the capture is refreshed.  The resident
# kernels were captured at 64 substeps: bytes per substep of the launch, scaled by the rollout length.
NCU_TRAFFIC = {
    "config4-large-1000000tets-522242tris": {
        "source": "profiles/r2_ncu_config4_streaming.md (round-2 kernels; k_particles_adj still from profiles/r1d_ncu_config4_streaming.md)",
        "k_elements_fwd": ("per_launch", 161725952), "k_particles_fwd": ("per_launch", 24154368),
        "k_elements_adj": ("per_launch", 205242880), "k_particles_adj": ("per_launch", 40113664),
    },
    "config3-sysid-E1024": {"source": "profiles/r2_ncu_config3_resident.md (round-2 kernels, 64-substep capture gpurun_out/r2_ncu_res.ncu-rep)",
                            "k_resident_fwd": ("per_substep", 3495948), "k_resident_adj": ("per_substep", 4730524)},
}


def ncu_traffic(workload, kernel, T):
    """(DRAM bytes per launch of `kernel` from the committed ncu capture of this workload, its source) or (None, None)."""
    w = NCU_TRAFFIC.get(workload, {})
    kind, val = w.get(kernel, (None, None))
    if kind is None:
        return None, None
    return (val if kind == "per_launch" else val * T), w["source"]


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def __exit__(self, *a):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
            self.th.join(timeout=1)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for n, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def make_workload(config, small):
    from paper_2104_02646_b200 import scenes

    return scenes.make_scene(config, small=small)


def centroid_target(sc):
    """[E,3] seeded final-centroid target: the bench's loss is the final-centroid distance on every config."""
    from paper_2104_02646_b200 import scenes

    return scenes._final_centroid_target(sc.config, sc.x0)


def oracle_sample(sc, sample_substeps, threads=None):
    """The oracle as it stands on a bounded sample: the first `sample_substeps` substeps of the workload,
    forward + final-centroid loss + adjoint.  threads: OpenMP threads (None = all cores).
    Returns (element-substeps/s, seconds, threads used)."""
    from oracle import oracle as orc

    n_all = orc.num_threads()
    if threads is not None:
        orc.set_num_threads(threads)
    try:
        o = orc.Oracle(sc)
        T = sample_substeps
        x0, v0 = sc.x0.astype(np.float64), sc.v0.astype(np.float64)
        t0 = time.perf_counter()
        ro = o.rollout(x0, v0, T, K=1, rec_times=[T])
        tgt = centroid_target(sc)
        _, cot = orc.loss_and_cotangents("final_centroid", ro["rec_x"], tgt)
        o.zero_grads()
        o.rollout_backward(ro, [T], cot)
        dt = time.perf_counter() - t0
        used = orc.num_threads()
    finally:
        orc.set_num_threads(n_all)
    return sc.n_elements * sc.n_envs * T / dt, dt, used


def sample_size(sc, rate=4e7):
    """substeps of the workload the oracle can do in roughly 10-30 s (about 2e6 element-substeps/s/thread fwd+adj);
    `rate` = element-substeps of the sample."""
    per = sc.n_elements * sc.n_envs
    return int(max(1, min(sc.n_substeps, rate // max(per, 1))))


def cpu_baseline_record(sc):
    """SURVEY.md 8(d) timing protocol: the oracle on all host cores AND on a single thread (the canonical CPU baseline),
    each on a bounded sample of the workload."""
    T = sc.n_substeps
    Ts = sample_size(sc)
    val, dt_s, th = oracle_sample(sc, Ts)
    T1 = sample_size(sc, 1e7)
    v1, dt1, th1 = oracle_sample(sc, T1, threads=1)
    return {"value": val, "unit": UNIT, "cores": th, "kind": "oracle", "seconds": dt_s,
            "sample": f"first {Ts} of {T} substeps of {sc.name}, forward + final-centroid loss + adjoint, fp64",
            "single_thread": {"value": v1, "unit": UNIT, "cores": th1, "seconds": dt1,
                              "sample": f"first {T1} of {T} substeps of {sc.name}, forward + final-centroid loss + adjoint, fp64"}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sc = make_workload(args.config, args.small)
    T = sample_size(sc)
    vals = []
    for _ in range(args.warmup):
        oracle_sample(sc, max(1, T // 4))
    t_tot = 0.0
    for _ in range(args.steps):
        v, dt, th = oracle_sample(sc, T)
        vals.append(v); t_tot += dt
    val = sc.n_elements * sc.n_envs * T * args.steps / t_tot
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": sc.name, "config_index": args.config},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": th, "kind": "oracle",
                         "sample": f"first {T} of {sc.n_substeps} substeps of {sc.name}, forward + loss + adjoint, fp64"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


class Workload:
    """One config on the device: model, tape, inputs, the scene's own loss (SURVEY.md 8(c) "Losses") and the step."""

    def __init__(self, sc, plan, devs):
        import torch

        from paper_2104_02646_b200 import gradsim as gs

        self.gs, self.torch, self.sc, self.devs = gs, torch, sc, devs
        E, N, T, K = sc.n_envs, sc.n_particles, sc.n_substeps, sc.checkpoint_every
        self.m = gs.Model(sc, plan=plan, device=devs)
        self.tape = self.m.tape(T, K)
        self.x0 = torch.as_tensor(sc.x0, device=devs)
        self.v0 = torch.as_tensor(sc.v0, device=devs)
        s = sc.frame_stride
        self.lt = sc.loss_times()
        self.frames_t = [t for t in self.lt if sc.loss != "final_centroid" and t % s == 0]
        self.n_frames = len(self.frames_t)
        self.target_np = self._targets()
        self.tgt = torch.as_tensor(self.target_np, device=devs)
        self.cot = torch.zeros((max(self.n_frames, 1), E, N, 3), dtype=torch.float32, device=devs)
        self.cot_T = torch.zeros((E, N, 3), dtype=torch.float32, device=devs)
        self.loss = torch.zeros(E, dtype=torch.float32, device=devs)
        self.xt = torch.zeros((E, N, 3), dtype=torch.float32, device=devs)
        self.ax0, self.av0 = torch.zeros_like(self.xt), torch.zeros_like(self.xt)
        self.groups = ["mass"] + (["tet_mu", "tet_lambda"] if sc.tets.shape[0] else []) + (["tri_mu"] if sc.tris.shape[0] else [])

    def _targets(self):
        """fp32 targets of the scene's loss.  Seeded ones come with the scene; configs 2 and 3 compare against a rollout
        of the SAME simulator with the truth-stream parameters (guess -> unroll -> compare): produced here
        by the CUDA path itself (a second model), outside every timed region."""
        sc, gs, torch = self.sc, self.gs, self.torch
        if sc.target is not None:
            return np.ascontiguousarray(sc.target, dtype=np.float32)
        import copy

        tsc = copy.copy(sc)
        for k, val in sc.truth.items():
            setattr(tsc, k, val)
        mt = gs.Model(tsc, device=self.devs)
        tt = mt.tape(sc.n_substeps, sc.frame_stride)  # holds exactly the frame states
        xT, _ = tt.rollout(self.x0, self.v0)
        rec = [xT if t == sc.n_substeps else tt.read(t, want_v=False)[0] for t in self.lt]
        rec = torch.stack(rec)  # [n_t, E, N, 3]
        out = rec if sc.loss == "pos_mse_frames" else rec.mean(dim=2)
        return np.ascontiguousarray(out.cpu().numpy(), dtype=np.float32)

    def fwd_only(self):
        self.tape.rollout(self.x0, self.v0, want_final=False)

    def fwd_bwd(self):
        """gs_rollout, the scene's loss at its loss times (tape reads + loss kernels), gs_rollout_backward."""
        gs, sc, m, tape = self.gs, self.sc, self.m, self.tape
        L = gs.lib()
        st = gs._stream()
        m.zero_grads()
        gs._check(L.gs_rollout(m.h, tape.h, gs._dp(self.x0), gs._dp(self.v0), gs._dp(self.xt), None, st))
        E, N, T, n_t = m.E, m.N, sc.n_substeps, len(self.lt)
        adj_T = None
        if sc.loss == "final_centroid":
            gs._check(L.gs_loss_centroid(E, N, gs._dp(self.xt), gs._dp(self.tgt), 1.0, 0, gs._dp(self.loss), gs._dp(self.cot_T), st))
            adj_T = self.cot_T
        else:
            for k, t in enumerate(self.lt):
                if t != T:
                    gs._check(L.gs_tape_read(m.h, tape.h, t, gs._dp(self.xt), None, st))
                elif k > 0:
                    gs._check(L.gs_tape_read(m.h, tape.h, T, gs._dp(self.xt), None, st))
                if t in self.frames_t:
                    a = self.cot[self.frames_t.index(t)]
                else:
                    a = adj_T = self.cot_T
                if sc.loss == "pos_mse_frames":
                    gs._check(L.gs_loss_pos(E, N, gs._dp(self.xt), gs._dp(self.tgt[k]), 1.0 / (n_t * N), int(k > 0), gs._dp(self.loss), gs._dp(a), st))
                else:
                    gs._check(L.gs_loss_centroid(E, N, gs._dp(self.xt), gs._dp(self.tgt[k]), 1.0 / n_t, int(k > 0), gs._dp(self.loss), gs._dp(a), st))
        gs._check(L.gs_rollout_backward(m.h, tape.h, self.n_frames, sc.frame_stride if self.n_frames else 1,
                                        gs._dp(self.cot) if self.n_frames else None, gs._dp(adj_T), None, gs._dp(self.ax0), gs._dp(self.av0), st))


def measure(args, config, rank, world, local, dist, with_cpu):
    """All timed legs of one config; returns the JSON record (rank 0) or None."""
    import torch

    from paper_2104_02646_b200 import gradsim as gs

    devs = f"cuda:{local}"

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sc = make_workload(config, args.small)
    if args.substeps > 0:
        sc.n_substeps = args.substeps
        sc.frame_stride = min(sc.frame_stride, sc.n_substeps)
    E_total = sc.n_envs
    sharded = bool(args.shard_envs and world > 1 and sc.n_envs >= world)
    if sharded:
        # the environment axis is the one axis that shards without a per-substep exchange: every rank
        # owns a contiguous block of environments, no data-path collective, one gather of per-environment rows at the end
        from paper_2104_02646_b200 import sharding

        sc = sharding.shard_scene(sc, world, rank)
    E, N, T, K = sc.n_envs, sc.n_particles, sc.n_substeps, sc.checkpoint_every
    w = Workload(sc, args.plan, devs)
    m, tape = w.m, w.tape
    L = gs.lib()
    units_per_step = m.n_elements * E * T          # this rank's units
    job_units = m.n_elements * T * (E_total if sharded else E * world)  # whole job

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        barrier()
        n0 = L.gs_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if dist is not None:
            t = torch.tensor([ms], device=devs)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms, L.gs_launch_count() - n0

    with ClockSampler(local) as clk:
        ms_fb, launches = timed(w.fwd_bwd, args.steps, args.warmup)
        ms_f, _ = timed(w.fwd_only, args.steps, 1)
    bad = m.check_finite()
    loss_dev = w.loss.detach().cpu().numpy().astype(np.float64)

    # ---- e2e through the host-buffer entry point (pinned host memory, copies inside the timed region), same loss
    hx0, hv0, htg = torch.as_tensor(sc.x0).pin_memory(), torch.as_tensor(sc.v0).pin_memory(), torch.as_tensor(w.target_np).pin_memory()

    def e2e_step():
        return m.rollout_loss_backward_host(tape, hx0, hv0, htg, groups=w.groups, loss=sc.loss, frame_stride=sc.frame_stride)

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        res = e2e_step()  # synchronises: the result is on the host when it returns
    barrier()
    t_e2e = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([t_e2e], device=devs)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_e2e = float(t.item())
    loss_e2e = res["loss"].numpy().astype(np.float64)
    # the e2e call runs the same kernels as the device-buffer path: same loss up to the atomics' summation order
    assert np.abs(loss_e2e - loss_dev).max() <= 1e-3 * np.abs(loss_dev).max(), (loss_e2e[:4], loss_dev[:4])
    h2d = hx0.numel() * 4 + hv0.numel() * 4 + htg.numel() * 4
    d2h = 4 * (E + 2 * E * N * 3 + sum(E * m.group_count(g) for g in w.groups))
    e2e = {"value": job_units * args.steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "call": "gs_rollout_loss_backward_host", "loss_kind": sc.loss, "loss": float(loss_e2e[0]), "loss_device_path": float(loss_dev[0])}


    # ---- per-kernel CUDA-event durations over one more pass of the same step (events on the launching stream)
    roofline, kernels = None, {}
    peak, peak_src = hbm_peak()
    resident = m.plan == gs.GS_PLAN_RESIDENT and K == 1
    if rank == 0:
        L.gs_kernel_timing(m.h, 1)
        w.fwd_bwd()
        ms_k = (gs.C.c_double * len(KERNELS))()
        n_k = (gs.C.c_uint64 * len(KERNELS))()
        gs._check(L.gs_kernel_times(m.h, gs._stream(), len(KERNELS), ms_k, n_k))
        L.gs_kernel_timing(m.h, 0)
        tot = sum(ms_k)
        for name, a, b in zip(KERNELS, ms_k, n_k):
            kernels[name] = {"launches": int(b), "ms_total": a, "us_avg": (1e3 * a / b) if b else None, "share": a / tot if tot else None}
        # algorithmic bytes per launch: the streaming kernels move one substep's element / particle
        # streams; a resident launch covers all T substeps of the state-in / state-out model with shared connectivity
        alg = {"k_elements_fwd": element_stream_bytes(sc, BYTES_FWD), "k_elements_adj": element_stream_bytes(sc, BYTES_ADJ),
               "k_particles_fwd": E * N * BYTES_FWD["particle"], "k_particles_adj": E * N * BYTES_ADJ["particle"],
               "k_resident_fwd": resident_stream_bytes(sc, False) * T, "k_resident_adj": resident_stream_bytes(sc, True) * T}
        flops = {"k_resident_fwd": substep_flops(sc, FLOPS_FWD) * T, "k_resident_adj": substep_flops(sc, FLOPS_ADJ) * T,
                 "k_elements_fwd": element_stream_bytes(sc, FLOPS_FWD), "k_elements_adj": element_stream_bytes(sc, FLOPS_ADJ)}
        dom = max(alg, key=lambda k: kernels[k]["ms_total"])
        for k in alg:
            if kernels[k]["us_avg"]:
                sec = kernels[k]["us_avg"] * 1e-6
                kernels[k].update(alg_bytes=alg[k], alg_gbs=alg[k] / sec / 1e9, hbm_frac=alg[k] / sec / 1e9 / peak)
                if k in flops:
                    kernels[k].update(alg_flops=flops[k], alg_tflops=flops[k] / sec / 1e12, alu_frac=flops[k] / sec / 1e12 / ALU_PEAK_TFLOPS)
        if kernels[dom]["us_avg"]:
            traffic, tsrc = (None, None) if (args.substeps or args.small) else ncu_traffic(sc.name, dom, T)
            kd = kernels[dom]
            common = {"kernel": dom, "traffic": traffic, "traffic_source": tsrc, "us_per_launch": kd["us_avg"], "alg_bytes_per_launch": alg[dom],
                      "alg_flops_per_launch": flops.get(dom)}
            hbm = {"achieved": kd["alg_gbs"], "peak": peak, "unit": "GB/s", "frac": kd["hbm_frac"], "peak_source": peak_src}
            alu = {"achieved": kd.get("alg_tflops"), "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": kd.get("alu_frac"),
                   "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 x 1965 MHz (DESIGN.md section 6)"}
            if resident:
                # state stays on-chip: the binding roofline is the plain fp32 ALU; the HBM fraction under the
                # survey's streaming byte model is reported beside it
                roofline = {"bound": "alu", **alu, **common, "hbm_streaming_model": hbm}
            else:
                roofline = {"bound": "hbm", **hbm, **common, "alu": alu}

    if sharded:
        # the one exchange of the sharded job, after the timed region: per-environment rows (loss, total dL/dmu, dL/dlambda, dL/dm)
        from paper_2104_02646_b200 import sharding

        rows = torch.stack([w.loss] + [m.param_grads(g).sum(1) for g in ("tet_mu", "tet_lambda", "mass")], 1)
        rows = sharding.gather_env_rows(rows, E_total, dist)
        assert rows.shape == (E_total, 4) and bool(torch.isfinite(rows).all())
    if rank != 0:
        return None

    cpu = cpu_baseline_record(sc) if with_cpu else None
    step_s = ms_fb * 1e-3 / args.steps
    fwd_s = ms_f * 1e-3 / args.steps
    if resident:
        b_f, b_a = resident_stream_bytes(sc, False) * T, resident_stream_bytes(sc, True) * T
    else:
        b_f, b_a = substep_bytes(sc, BYTES_FWD) * T, substep_bytes(sc, BYTES_ADJ) * T
    bytes_fb = b_f + b_a + (b_f if K > 1 else 0)  # checkpointed tapes replay every segment once
    fl_fb = (substep_flops(sc, FLOPS_FWD) * (2 if K > 1 else 1) + substep_flops(sc, FLOPS_ADJ)) * T
    return {
        "metric": METRIC, "value": job_units / step_s, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * step_s, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": sc.name, "config_index": config, "particles": N, "tets": int(sc.tets.shape[0]), "tris": int(sc.tris.shape[0]),
                   "hinges": int(sc.hinges.shape[0]), "envs": E, "substeps": T, "substeps_overridden": bool(args.substeps), "checkpoint_every": K, "plan": m.plan,
                   "loss": sc.loss, "loss_times": len(w.lt), "frame_stride": sc.frame_stride,
                   "l2": "inputs larger than L2 (state tape + element streams stream from HBM every step)" if tape.nbytes > 3e8 else "working set may sit in L2",
                   "friction_reading": "BASELINE kf -> mu_c, k_f = 50 (DESIGN.md A9)", "parallelism": (f"environments sharded over {world} ranks, no data-path collective" if sharded else f"replicas x{world}")},
        "forward": {"value": job_units / fwd_s, "unit": UNIT, "ms_per_step": 1e3 * fwd_s,
                    "model_gbs": b_f / fwd_s / 1e9, "hbm_frac": b_f / fwd_s / 1e9 / peak},
        "step_model": {"bytes_per_step": bytes_fb, "model_gbs": bytes_fb / step_s / 1e9, "hbm_frac": bytes_fb / step_s / 1e9 / peak,
                       "byte_model": "SURVEY.md 8(d): " + ("state in/out per env-substep, shared connectivity (resident)" if resident else "element + particle streams per substep"),
                       "flops_per_step": fl_fb, "model_tflops": fl_fb / step_s / 1e12, "alu_frac": fl_fb / step_s / 1e12 / ALU_PEAK_TFLOPS},
        "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "kernels": kernels, "cpu_baseline": cpu, "clocks": clk.summary(),
        "first_bad_substep": bad, "tape_bytes": tape.nbytes,
    }


RASTER_FLOPS_FWD, RASTER_FLOPS_BWD = 95, 325  # per evaluated (pixel, triangle) pair: 3 point-segment distances, 3 edge functions,
# a sigmoid (forward); the adjoint walks the pairs twice and adds the closest-edge weights
RASTER_FLOPS_FWD_RGB, RASTER_FLOPS_BWD_RGB = 175, 530  # colour channel: + barycentrics, clamp, depth, colour, two exp, the running
# softmax (forward); the adjoint walks twice, adds the chain through the barycentrics and a transposing warp sum of the 18 vertex components


def raster_record(devs, steps):
    """the soft silhouette rasteriser + adjoint on E = 64 deformed copies of config 1's 32 x 32 cloth
    (1922 triangles), 256 x 256 pixels.  ALU-bound: flops = evaluated (pixel, triangle) pairs (those the tile culling
    keeps, counted here from the oracle's projection) x the per-pair counts above."""
    import torch

    from oracle import raster_oracle as ro
    from paper_2104_02646_b200 import gradsim as gs
    from paper_2104_02646_b200 import scenes

    sc = scenes.make_scene(1)
    E, W, H, sigma = 64, 256, 256, 1e-4
    r = scenes.rng_for(1, "misc", 123)
    x = (sc.x0[0][None] + 0.003 * r.normal(size=(E,) + sc.x0[0].shape)).astype(np.float32)
    th = 0.4
    R = np.array([[1, 0, 0], [0, np.cos(-1.0), -np.sin(-1.0)], [0, np.sin(-1.0), np.cos(-1.0)]]) @ np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]])
    cam_args = (R, np.array([-0.15, 0.1, 0.6]), 2.0, 2.0, W, H, sigma)
    cg, co = gs.make_camera(*cam_args), ro.Camera(*cam_args)
    xd = torch.as_tensor(x, device=devs)
    tris = torch.as_tensor(np.ascontiguousarray(sc.tris, dtype=np.int32), device=devs)
    target = gs.render_silhouette(torch.as_tensor(x + np.float32(0.004), device=devs), tris, cg)

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps

    ms_f = timed(lambda: gs.render_silhouette(xd, tris, cg))
    ms_b = timed(lambda: gs.loss_silhouette(xd, tris, cg, target))
    # colour channel (A22b): random vertex colours, depth softmax gamma = 0.05
    sg = gs.make_shading(0.05, 1e-3, 3.0, (0.1, 0.2, 0.3))
    cold = torch.as_tensor(r.uniform(0.0, 1.0, x.shape).astype(np.float32), device=devs)
    target_rgb = gs.render_rgb(torch.as_tensor(x + np.float32(0.004), device=devs), tris, cold, cg, sg)
    ms_fc = timed(lambda: gs.render_rgb(xd, tris, cold, cg, sg))
    ms_bc = timed(lambda: gs.loss_rgb(xd, tris, cold, cg, sg, target_rgb))
    # evaluated pairs: triangles whose grown bounding box meets a 16 x 16 tile, x 256 pixels (environment 0, scaled by E)
    ndc, z = ro.project(x[0].astype(np.float64), co)
    q = ndc[sc.tris]
    m = np.sqrt(40.0 * sigma)
    lo, hi = q.min(1) - m, q.max(1) + m
    tu0 = np.arange(0, W, 16) * 2.0 / W - 1.0
    tv0 = np.arange(0, H, 16) * 2.0 / H - 1.0
    nx = ((lo[:, None, 0] <= tu0[None] + 32.0 / W) & (hi[:, None, 0] >= tu0[None])).sum(1)
    ny = ((lo[:, None, 1] <= tv0[None] + 32.0 / H) & (hi[:, None, 1] >= tv0[None])).sum(1)
    pairs = float((nx * ny).sum()) * 256 * E
    t0 = time.perf_counter()
    ro.silhouette(x[0], sc.tris, co)
    t_cpu = time.perf_counter() - t0
    return {"workload": f"config1 cloth 32x32 ({sc.tris.shape[0]} triangles) x {E} environments, {W}x{H} pixels, sigma {sigma}",
            "ms_render": ms_f, "ms_loss_and_adjoint": ms_b, "evaluated_pairs": pairs,
            "rgb": {"ms_render": ms_fc, "ms_loss_and_adjoint": ms_bc, "gamma": 0.05,
                    "alu_frac_upper": pairs * RASTER_FLOPS_FWD_RGB / (ms_fc * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                    "adjoint_alu_frac_upper": pairs * RASTER_FLOPS_BWD_RGB / (ms_bc * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                    "note": "upper bounds: flops per pair as if every culled-in pair passed the per-pixel 40 sigma cut"},
            "roofline": {"bound": "alu", "kernel": "k_rs_forward", "achieved": pairs * RASTER_FLOPS_FWD / (ms_f * 1e-3) / 1e12, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": pairs * RASTER_FLOPS_FWD / (ms_f * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                         "adjoint_frac": pairs * RASTER_FLOPS_BWD / (ms_b * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                         "note": "ms_render includes projection + triangle packing; flops per pair counted from csrc/gs_raster.cu"},
            "cpu_baseline": {"kind": "oracle", "seconds_per_image": t_cpu, "sample": "one environment, forward only, fp64 numpy", "images_per_s_gpu": E / (ms_f * 1e-3)}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--small", action="store_true", help="reduced variant of the config (debugging only; not a bench number)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-config3", action="store_true", help="skip the config-3 sub-record of the default (config 4) line")
    ap.add_argument("--shard-envs", action="store_true", help="N > 1 with a batched config: shard the environments over the ranks (strong scaling) instead of replicas")
    ap.add_argument("--plan", type=int, default=0)
    ap.add_argument("--substeps", type=int, default=0, help="override the rollout length (profiling runs only; recorded in config)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the gradSim hot path has no CPU fallback")
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    with_cpu = not args.no_cpu_baseline and world == 1
    line = measure(args, args.config, rank, world, local, dist, with_cpu)
    # the north_star names two target configs: the default line (config 4, the headline) carries config 3 (the
    # 1024-environment batch, ALU-bound) as a sub-record measured in the same run
    sub = None
    if args.config == 4 and not args.small and not args.substeps and not args.no_config3:
        torch.cuda.empty_cache()
        sub = measure(args, 3, rank, world, local, dist, with_cpu)
    if rank == 0:
        line["config3"] = sub
        line["raster"] = raster_record(f"cuda:{local}", args.steps) if (with_cpu and args.config == 4 and not args.small and not args.substeps) else None
        line["paper_context"] = "Table 4-right: 3721 Hz fwd / 1429 Hz bwd at 10k tets (3.7e7 / 1.4e7 tet-steps/s), hardware unstated (PAPER.md:464-478)"
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
