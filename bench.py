#!/usr/bin/env python
"""bench.py -- throughput of the SSP-RK3 step of the spectral hyperviscosity solver on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5|c4|c3|c2|c1] [--dtype f64|f32]
  python bench.py --impl reference ...      # the CPU oracle on the host cores (a deliberately slow baseline)

A "step" is one full SSP-RK3 step (eq. 2.6) = 3 x (passes a1..a7 of SURVEY.md 8(a)) + the device-side CFL
reduction, on one batch of seeded synthetic input (recipes in paper_2401_09843_b200/inputs.py).
Default workload: BASELINE.json configs[4] (N = 512^3 fp64, 1 sample), the largest single-GPU configuration
and the one the north_star's target is quoted on; c4 = configs[3] (32 x 128^3 ensemble) is the other target.
Metric: grid-point-stages/s = batch * N^3 * 3 * steps/s (steps/s is reported beside it).

Prints ONE JSON line (rank 0).  Multi-GPU (torchrun, one rank per GPU): the path does not shard a sample;
ranks run independent replicas of the workload (more Monte-Carlo samples, Algorithm 1), "scaling": "weak",
no data-path collective; value = total units / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2401_09843_b200 import inputs, roofline  # noqa: E402

WORKLOADS = {
    # name: (BASELINE.json configs index, N, batch, params, cfl, description, cpu sample N)
    "c1": dict(cfg=0, N=32, batch=1, params=dict(nu=0.01), dt=1e-3, desc="configs[0]: 32^3 Taylor-Green + 1e-3 noise, nu=0.01, dt=1e-3", cpuN=32),
    "c2": dict(cfg=1, N=128, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[1]: 128^3 Gaussian k^4 exp, hyperviscosity eps=0.05 s=1, CFL 0.2", cpuN=64),
    "c3": dict(cfg=2, N=256, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[2]: 256^3 perturbed shear layer, hyperviscosity, CFL 0.2", cpuN=64),
    "c4": dict(cfg=3, N=128, batch=32, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[3]: 32 x 128^3 shear-layer ensemble in one launch, CFL 0.2", cpuN=64),
    # the paper's own experiments, hyperviscosity order s = 1.5
    "tg3d": dict(cfg=None, N=256, batch=1, params=dict(eps=0.05, s=1.5), cfl=0.2, desc="paper eq. 6.1-6.3: 256^3 perturbed 3-D Taylor-Green, hyperviscosity eps=0.05 s=1.5, CFL 0.2", cpuN=64),
    "cyl": dict(cfg=None, N=256, batch=1, params=dict(eps=0.05, s=1.5), cfl=0.2, desc="paper eq. 6.4-6.6: 256^3 cylindrical shear flow rho=0.05, hyperviscosity eps=0.05 s=1.5, CFL 0.2", cpuN=64),
    "c5": dict(cfg=4, N=512, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[4]: 512^3 Gaussian k^-5/3, hyperviscosity eps=0.05 s=1, CFL 0.2", cpuN=64),
}


def make_input(name: str, N: int, batch: int) -> np.ndarray:
    """Physical-space samples [batch][3][N][N][N] of the workload recipe at grid size N."""
    if name == "c1":
        return inputs.taylor_green_perturbed(N, seed=1)[None]
    if name == "c2":
        return inputs.gaussian_k4(N, seed=2)[None]
    if name == "c3":
        return inputs.shear_layer(N, seed=3)[None]
    if name == "c4":
        return inputs.shear_layer_ensemble(N, batch, seed0=1000)
    if name == "c5":
        return inputs.gaussian_k53(N, seed=5)[None]
    if name == "tg3d":
        return inputs.taylor_green_3d_perturbed(N, seed=6)[None]
    if name == "cyl":
        return inputs.cylindrical_shear(N, seed=7, rho=0.05)[None]
    raise KeyError(name)


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def aggregate(local_ms_total: float, local_units: float, world: int, dist=None):
    """Max-over-ranks time and summed units (host logic; covered by a gloo world_size-2 CPU test)."""
    if world == 1 or dist is None:
        return local_ms_total, local_units
    import torch
    t = torch.tensor([local_ms_total], dtype=torch.float64)
    u = torch.tensor([local_units], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled every 100 ms during the timed region."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_run(name: str, steps: int, warmup: int = 0):
    """Time the oracle, as it stands, on a bounded sample of the workload: RK3 steps at a reduced grid."""
    from oracle import ns_oracle
    w = WORKLOADS[name]
    Ns = w["cpuN"]
    u = make_input(name, Ns, 1)[0]
    uh = ns_oracle.set_initial(Ns, u)
    p = ns_oracle.Params(**w["params"])
    dt = w.get("dt") or 0.2 * (2 * np.pi / Ns) / max(ns_oracle.max_velocity(Ns, uh), 1e-30)
    for _ in range(warmup):
        uh = ns_oracle.step(Ns, p, uh, dt)
    t0 = time.perf_counter()
    for _ in range(steps):
        uh = ns_oracle.step(Ns, p, uh, dt)
    el = time.perf_counter() - t0
    value = roofline.grid_point_stages(Ns, 1, steps) / el
    sample = f"{steps} RK3 step(s) of the {name} recipe on a {Ns}^3 grid (1 sample), fp64, naive radix-2/3 FFT, OpenMP"
    return dict(value=value, unit="grid-point-stages/s", cores=ns_oracle.num_threads(), kind="oracle", sample=sample,
                seconds=el, steps_per_s=steps / el), el / steps * 1e3


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    w = WORKLOADS[args.workload]
    cb, ms = cpu_oracle_run(args.workload, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": "grid_point_stages_per_s", "value": cb["value"], "unit": "grid-point-stages/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["desc"], "note": "CPU oracle on host cores; each step is a bounded sample: " + cb["sample"]},
        "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": cb["value"], "unit": "grid-point-stages/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c5", choices=sorted(WORKLOADS))
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3  # timing rule: at least 3 warm-up steps

    import torch
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist  # plumbing only: barrier + max/sum of two scalars
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    from paper_2401_09843_b200 import binding

    w = WORKLOADS[args.workload]
    N, batch = w["N"], w["batch"]
    cbytes = 16 if args.dtype == "f64" else 8
    t_gen = time.perf_counter()
    u0 = make_input(args.workload, N, batch)
    t_gen = time.perf_counter() - t_gen
    s = binding.Solver(N, batch=batch, dtype=args.dtype, **w["params"])
    s.set_initial(u0)
    chk = inputs.checksum(u0[0, 0, :2])
    del u0

    def one_step():
        if "dt" in w:
            s.step(w["dt"])
        else:
            s.step_cfl(w["cfl"], 1e30, return_dt=False)

    state_bytes = batch * 3 * N * N * (N // 2) * cbytes
    flush = state_bytes * 7 < 512 * 2 ** 20  # working set of a pass (~7x the state) not >> the 126 MB L2
    flush_buf = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device="cuda") if flush else None

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step()
    barrier()
    s.profile(True)
    launches0 = s.kernel_launches()
    sampler = ClockSampler(local)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps if flush else 1)]
    barrier()
    if flush:
        for a, b in evs:
            flush_buf.fill_(1)
            a.record()
            one_step()
            b.record()
    else:
        evs[0][0].record()
        for _ in range(args.steps):
            one_step()
        evs[0][1].record()
    barrier()
    total_ms = sum(a.elapsed_time(b) for a, b in evs)
    clocks = sampler.stop()
    launches = s.kernel_launches() - launches0
    prof = s.profile_read()
    s.profile(False)
    finite = bool(np.isfinite(s.max_velocity()).all())

    total_ms, units = aggregate(total_ms, roofline.grid_point_stages(N, batch, args.steps), world, dist)
    ms_per_step = total_ms / args.steps
    value = units / (total_ms * 1e-3)

    # ---- roofline of the dominant kernel and of the whole step (fixed model)
    peak, peak_src = measured_peaks()
    per_step = roofline.pass_bytes_per_step(N, batch, cbytes)        # fixed model
    built = roofline.built_pass_bytes_per_step(N, batch, cbytes)     # what the built kernels must move
    prof_label = {"a1_col_inv_x": "a1_col_inv_x", "a2_col_inv_y": "a2_col_inv_y", "a3_z_inv_prod": "a3a4_z_fused",
                  "a5_col_fwd_y": "a5_col_fwd_y", "a6_col_fwd_x": "a6_col_fwd_x", "a7_spectral": "a7_spectral"}
    kernels = {}
    for name, label in prof_label.items():
        ms, cnt = prof[name]
        if not cnt:
            continue
        nbytes, extra = built[label], {}
        if label == "a3a4_z_fused":
            # the fixed model charges a3 + a4 separately (six M^3 products written and read back)
            model = per_step["a3_z_inv_prod"] + per_step["a4_z_fwd"]
        else:
            model = per_step[name]
        if model != nbytes:
            extra = {"model_bytes_per_launch": model * args.steps / cnt,
                     "model_gbs_equivalent": model * args.steps / (ms * 1e-3) / 1e9}
        gbs = nbytes * args.steps / (ms * 1e-3) / 1e9
        kernels[label] = {"ms_per_launch": ms / cnt, "launches": cnt, "alg_bytes_per_launch": nbytes * args.steps / cnt,
                          "gbs": gbs, "frac": gbs / peak, "share_of_step": ms / (ms_per_step * args.steps), **extra}
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_launch"] * kernels[k]["launches"])
    # dram bytes per launch from the committed ncu --set full captures (profiles/traffic.csv), attached to every kernel
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            f = ln.split(",", 3)
            if len(f) >= 3 and f[0] == f"{args.workload}_{args.dtype}" and f[1] in kernels:
                kernels[f[1]]["traffic"] = float(f[2])
    traffic = kernels[dom].get("traffic")
    model_bytes = roofline.step_bytes(N, batch, cbytes)
    roof = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
            "frac": kernels[dom]["frac"], "traffic": traffic, "peak_source": peak_src,
            "alg_bytes_per_launch": kernels[dom]["alg_bytes_per_launch"], "ms_per_launch": kernels[dom]["ms_per_launch"]}
    if dom == "a3a4_z_fused":
        roof["note"] = ("fused a3+a4: by bytes HBM is the roofline (DRAM traffic = algorithmic 8*A2), but ncu shows a latency / "
                        "fp64-issue limited kernel (c5: fp64 pipe 44 %, l1tex 63 %, DRAM 23 % busy; profiles/r01b_tmem.md); the "
                        "unfused a3 + a4 of the fixed model would need model_bytes_per_launch / peak = "
                        f"{kernels[dom]['model_bytes_per_launch'] / (peak * 1e9) * 1e3:.2f} ms at the measured peak")
    step_roof = {"model_bytes_per_step": model_bytes, "achieved_gbs": model_bytes / (ms_per_step * 1e-3) / 1e9,
                 "frac_of_measured_peak": model_bytes / (ms_per_step * 1e-3) / 1e9 / peak,
                 "frac_of_nominal_8TBs": model_bytes / (ms_per_step * 1e-3) / 1e9 / 8000.0,
                 "t_model_ms_at_measured_peak": model_bytes / (peak * 1e9) * 1e3}
    actual = roofline.actual_step_bytes(N, batch, cbytes)
    step_roof["actual_bytes_per_step"] = actual
    step_roof["actual_frac_of_measured_peak"] = actual / (ms_per_step * 1e-3) / 1e9 / peak
    step_roof["note"] = ("a3+a4 are one kernel (products never reach HBM) and 5 trace-free flux components are transformed "
                         "instead of 6: frac_* use the FIXED model bytes of SURVEY.md 8(d); actual_* use the bytes the "
                         "built pass structure must move")

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D state, step, D2H state, every step
    e2e = None
    if not args.no_e2e:
        shape = s.spectral_shape
        ct = torch.complex128 if args.dtype == "f64" else torch.complex64
        h_in = torch.empty(shape, dtype=ct).pin_memory()
        h_out = torch.empty(shape, dtype=ct).pin_memory()
        a_in, a_out = h_in.numpy(), h_out.numpy()
        s.get_spectral(a_in)
        for _ in range(1):
            s.set_spectral(a_in); one_step(); s.get_spectral(a_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            s.set_spectral(a_in)
            one_step()
            s.get_spectral(a_out)
            a_in, a_out = a_out, a_in
        torch.cuda.synchronize()
        el = (time.perf_counter() - t0) * 1e3
        el, eunits = aggregate(el, roofline.grid_point_stages(N, batch, args.e2e_steps), world, dist)
        nbytes = int(np.prod(shape)) * cbytes
        e2e = {"value": eunits / (el * 1e-3), "unit": "grid-point-stages/s", "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes, "ms_per_step": el / args.e2e_steps, "steps": args.e2e_steps,
               "api": "ns_set_spectral(NS_HOST) + ns_step_cfl + ns_get_spectral(NS_HOST), pinned host buffers"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        nst = 20 if args.workload == "c1" else 12   # about 10 s on the GPU box's 16 cores, 30 s on 8
        cpu, _ = cpu_oracle_run(args.workload, nst)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "seconds")}

    if rank == 0:
        line = {
            "metric": "grid_point_stages_per_s", "value": value, "unit": "grid-point-stages/s",
            "steps_per_s": 1e3 / ms_per_step * world, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": w["desc"], "N": N, "batch_per_gpu": batch, "padded": 3 * N // 2,
                       "l2": "L2 flushed (256 MiB write) between timed steps" if flush else "inputs exceed L2 (126 MB): no flush needed",
                       "parallelism": "replicas only (independent samples per GPU)" if world > 1 else "single GPU",
                       "input_checksum": chk, "input_gen_s": round(t_gen, 1), "state_finite": finite},
            "roofline": roof, "step_roofline": step_roof, "kernels": kernels, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks, "device_bytes": s.device_bytes(),
        }
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
