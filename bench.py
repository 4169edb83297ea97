#!/usr/bin/env python
"""bench.py -- element-substeps/s of the gradSim hot path (forward and forward+adjoint) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: gs_rollout (T forward
substeps writing the on-device tape), the loss, and gs_rollout_backward (T adjoint substeps + parameter
gradients).  Default workload: BASELINE.json configs[4] (the 1M-tet + 512x512-cloth HBM stress case, the
largest single-GPU configuration); --config 3 runs the 1024-environment batch, 0..2 the small scenes.

Prints ONE JSON line (rank 0): value = whole-job element-substeps/s for forward+adjoint, plus
  forward      : the same for gs_rollout alone
  e2e          : through gs_rollout_loss_backward_host with pinned HOST buffers (H2D/D2H inside the timed region)
  roofline     : the dominant kernel's algorithmic bytes / its CUDA-event duration vs MEASURED_PEAKS.json
  cpu_baseline : the fp64 oracle, as it stands, on a bounded sample of the same workload on the host cores
  clocks       : nvidia-smi samples taken during the timed region
N > 1 (torchrun): every rank runs an independent replica of the workload (replicas only,
no data-path collective); time = max over ranks.
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


# DRAM traffic per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the hot kernels, from the ncu --set full
# captures summarised under profiles/ (r1d_ncu_config4_streaming.md, r1d_ncu_config3_resident.md).  The resident kernels
# were captured at 64 substeps: bytes per substep of the launch, scaled by the rollout length.
NCU_TRAFFIC = {
    "config4-large-1000000tets-522242tris": {
        "k_elements_fwd": ("per_launch", 161568256), "k_particles_fwd": ("per_launch", 22874368),
        "k_elements_adj": ("per_launch", 204752896), "k_particles_adj": ("per_launch", 40113664),
    },
    "config3-sysid-E1024": {"k_resident_fwd": ("per_substep", 3468752), "k_resident_adj": ("per_substep", 4660056)},
}


def ncu_traffic(workload, kernel, T):
    """DRAM bytes per launch of `kernel` from the committed ncu capture of this workload, or None."""
    kind, val = NCU_TRAFFIC.get(workload, {}).get(kernel, (None, None))
    if kind is None:
        return None
    return val if kind == "per_launch" else val * T


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


def oracle_sample(sc, sample_substeps):
    """The oracle as it stands on a bounded sample: the first `sample_substeps` substeps of the workload,
    forward + final-centroid loss + adjoint.  Returns (element-substeps/s, seconds, threads)."""
    from oracle import oracle as orc

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
    return sc.n_elements * sc.n_envs * T / dt, dt, orc.num_threads()


def sample_size(sc):
    """substeps of the workload the oracle can do in roughly 10-30 s (about 2e6 element-substeps/s/thread fwd+adj)."""
    per = sc.n_elements * sc.n_envs
    return int(max(1, min(sc.n_substeps, 4e7 // max(per, 1))))


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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--small", action="store_true", help="reduced variant of the config (debugging only; not a bench number)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--plan", type=int, default=0)
    ap.add_argument("--substeps", type=int, default=0, help="override the rollout length (profiling runs only; recorded in config)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch

    from paper_2104_02646_b200 import gradsim as gs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the gradSim hot path has no CPU fallback")
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    devs = f"cuda:{local}"

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sc = make_workload(args.config, args.small)
    if args.substeps > 0:
        sc.n_substeps = args.substeps
    E, N, T, K = sc.n_envs, sc.n_particles, sc.n_substeps, sc.checkpoint_every
    m = gs.Model(sc, plan=args.plan, device=devs)
    tape = m.tape(T, K)
    L = gs.lib()
    x0 = torch.as_tensor(sc.x0, device=devs)
    v0 = torch.as_tensor(sc.v0, device=devs)
    tgt_np = centroid_target(sc)
    tgt = torch.as_tensor(tgt_np, device=devs)
    units_per_step = m.n_elements * E * T

    def fwd_only():
        tape.rollout(x0, v0, want_final=False)

    def fwd_bwd():
        m.zero_grads()
        xT, _ = tape.rollout(x0, v0)
        _, adj = gs.loss_centroid(xT, tgt)
        tape.backward(adj_x_T=adj, want_out=True)

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
        ms_fb, launches = timed(fwd_bwd, args.steps, args.warmup)
        ms_f, _ = timed(fwd_only, args.steps, 1)
    bad = m.check_finite()

    # ---- e2e through the host-buffer entry point (pinned host memory, copies inside the timed region)
    hx0, hv0, htg = torch.as_tensor(sc.x0).pin_memory(), torch.as_tensor(sc.v0).pin_memory(), torch.as_tensor(tgt_np).pin_memory()
    groups = ["mass"] + (["tet_mu", "tet_lambda"] if sc.tets.shape[0] else []) + (["tri_mu"] if sc.tris.shape[0] else [])
    if K == 1 or True:
        def e2e_step():
            return m.rollout_loss_backward_host(tape, hx0, hv0, htg, groups=groups)

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
        h2d = hx0.numel() * 4 + hv0.numel() * 4 + htg.numel() * 4
        d2h = 4 * (E + 2 * E * N * 3 + sum(E * m.group_count(g) for g in groups))
        e2e = {"value": units_per_step * world * args.steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "call": "gs_rollout_loss_backward_host", "loss": float(res["loss"][0])}

    # ---- per-kernel CUDA-event durations over one more pass of the same step (events on the launching stream)
    roofline, kernels = None, {}
    peak, peak_src = hbm_peak()
    if rank == 0:
        L.gs_kernel_timing(m.h, 1)
        fwd_bwd()
        ms_k = (gs.C.c_double * len(KERNELS))()
        n_k = (gs.C.c_uint64 * len(KERNELS))()
        gs._check(L.gs_kernel_times(m.h, gs._stream(), len(KERNELS), ms_k, n_k))
        L.gs_kernel_timing(m.h, 0)
        tot = sum(ms_k)
        # the streaming plan launches one element kernel per non-empty element type: "us_avg" of the element rows is
        # per SUBSTEP (all types together), so that it pairs with the whole element stream's algorithmic bytes
        n_types = 1  # all element types of a substep share one persistent launch
        for name, a, b in zip(KERNELS, ms_k, n_k):
            per = n_types if name in ("k_elements_fwd", "k_elements_adj") else 1
            kernels[name] = {"launches": int(b), "ms_total": a, "us_avg": (1e3 * a * per / b) if b else None, "share": a / tot if tot else None}
            if per > 1:
                kernels[name]["launches_per_substep"] = per
        alg = {"k_elements_fwd": element_stream_bytes(sc, BYTES_FWD), "k_elements_adj": element_stream_bytes(sc, BYTES_ADJ),
               "k_particles_fwd": E * N * BYTES_FWD["particle"], "k_particles_adj": E * N * BYTES_ADJ["particle"]}
        # resident plan: one launch covers all T substeps; streaming byte model (state in and out every substep) and flops
        alg["k_resident_fwd"] = substep_bytes(sc, BYTES_FWD) * T
        alg["k_resident_adj"] = substep_bytes(sc, BYTES_ADJ) * T
        flops = {"k_resident_fwd": substep_flops(sc, FLOPS_FWD) * T, "k_resident_adj": substep_flops(sc, FLOPS_ADJ) * T}
        elem_flops = {"k_elements_fwd": element_stream_bytes(sc, FLOPS_FWD), "k_elements_adj": element_stream_bytes(sc, FLOPS_ADJ)}
        dom = max(alg, key=lambda k: kernels[k]["ms_total"])
        for k in alg:
            if kernels[k]["us_avg"]:
                kernels[k]["alg_bytes"] = alg[k]
                kernels[k]["alg_gbs"] = alg[k] / (kernels[k]["us_avg"] * 1e-6) / 1e9
                if k in flops:
                    kernels[k]["alg_flops"] = flops[k]
                    kernels[k]["alg_tflops"] = flops[k] / (kernels[k]["us_avg"] * 1e-6) / 1e12
        if dom in flops and kernels[dom]["us_avg"]:
            # state stays on-chip: the binding roofline is the plain fp32 ALU;
            # the streaming-model HBM fraction is reported beside it
            ach = kernels[dom]["alg_tflops"]
            roofline = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach / ALU_PEAK_TFLOPS,
                        "traffic": None if args.substeps or args.small else ncu_traffic(sc.name, dom, T), "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 x 1965 MHz (DESIGN.md section 6)",
                        "alg_flops_per_launch": flops[dom], "us_per_launch": kernels[dom]["us_avg"],
                        "hbm_streaming_model": {"achieved": kernels[dom]["alg_gbs"], "peak": peak, "unit": "GB/s", "frac": kernels[dom]["alg_gbs"] / peak,
                                                "alg_bytes_per_launch": alg[dom]}}
        elif kernels[dom]["us_avg"]:
            ach = kernels[dom]["alg_gbs"]
            roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                        "traffic": None if args.small else ncu_traffic(sc.name, dom, T),
                        # the element kernels execute more instructions than their bytes need time: fp32 ALU view
                        "alu": ({"achieved": elem_flops[dom] / (kernels[dom]["us_avg"] * 1e-6) / 1e12, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                                 "frac": elem_flops[dom] / (kernels[dom]["us_avg"] * 1e-6) / 1e12 / ALU_PEAK_TFLOPS} if dom in elem_flops else None),
                        "peak_source": peak_src, "alg_bytes_per_launch": alg[dom], "us_per_launch": kernels[dom]["us_avg"]}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- the oracle on the host cores, bounded sample
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        Ts = sample_size(sc)
        val, dt_s, th = oracle_sample(sc, Ts)
        cpu = {"value": val, "unit": UNIT, "cores": th, "kind": "oracle", "seconds": dt_s,
               "sample": f"first {Ts} of {T} substeps of {sc.name}, forward + loss + adjoint, fp64"}

    step_s = ms_fb * 1e-3 / args.steps
    fwd_s = ms_f * 1e-3 / args.steps
    bytes_fb = (substep_bytes(sc, BYTES_FWD) + substep_bytes(sc, BYTES_ADJ)) * T
    if K > 1:
        bytes_fb += substep_bytes(sc, BYTES_FWD) * T  # segment replay
    line = {
        "metric": METRIC, "value": units_per_step * world / step_s, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * step_s, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": sc.name, "config_index": args.config, "particles": N, "tets": int(sc.tets.shape[0]), "tris": int(sc.tris.shape[0]),
                   "hinges": int(sc.hinges.shape[0]), "envs": E, "substeps": T, "substeps_overridden": bool(args.substeps), "checkpoint_every": K, "plan": m.plan,
                   "l2": "inputs larger than L2 (state tape + element streams stream from HBM every step)" if tape.nbytes > 3e8 else "working set may sit in L2",
                   "friction_reading": "BASELINE kf -> mu_c, k_f = 50 (DESIGN.md A9)", "parallelism": f"replicas x{world}"},
        "forward": {"value": units_per_step * world / fwd_s, "unit": UNIT, "ms_per_step": 1e3 * fwd_s,
                    "model_gbs": substep_bytes(sc, BYTES_FWD) * T / fwd_s / 1e9, "hbm_frac": substep_bytes(sc, BYTES_FWD) * T / fwd_s / 1e9 / peak},
        "step_model": {"bytes_per_step": bytes_fb, "model_gbs": bytes_fb / step_s / 1e9, "hbm_frac": bytes_fb / step_s / 1e9 / peak},
        "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "kernels": kernels, "cpu_baseline": cpu, "clocks": clk.summary(),
        "first_bad_substep": bad, "tape_bytes": tape.nbytes,
        "paper_context": "Table 4-right: 3721 Hz fwd / 1429 Hz bwd at 10k tets (3.7e7 / 1.4e7 tet-steps/s), hardware unstated (PAPER.md:464-478)",
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
