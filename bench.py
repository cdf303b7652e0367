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
    "c2": dict(cfg=1, N=128, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[1]: 128^3 Gaussian k^4 exp, hyperviscosity eps=0.05 s=1, CFL 0.2", cpuN=128),
    "c3": dict(cfg=2, N=256, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[2]: 256^3 perturbed shear layer, hyperviscosity, CFL 0.2", cpuN=128),
    "c4": dict(cfg=3, N=128, batch=32, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[3]: 32 x 128^3 shear-layer ensemble in one launch, CFL 0.2", cpuN=128),
    # the paper's own experiments, hyperviscosity order s = 1.5
    "tg3d": dict(cfg=None, N=256, batch=1, params=dict(eps=0.05, s=1.5), cfl=0.2, desc="paper eq. 6.1-6.3: 256^3 perturbed 3-D Taylor-Green, hyperviscosity eps=0.05 s=1.5, CFL 0.2", cpuN=128),
    "cyl": dict(cfg=None, N=256, batch=1, params=dict(eps=0.05, s=1.5), cfl=0.2, desc="paper eq. 6.4-6.6: 256^3 cylindrical shear flow rho=0.05, hyperviscosity eps=0.05 s=1.5, CFL 0.2", cpuN=128),
    # a size N = 3 * 2^a, the c5 recipe at 384^3 (padded 576^3)
    "n384": dict(cfg=None, N=384, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="NEXT-3: 384^3 = (3 * 2^7)^3 Gaussian k^-5/3 (the configs[4] recipe), hyperviscosity eps=0.05 s=1, CFL 0.2", cpuN=96),
    "c5": dict(cfg=4, N=512, batch=1, params=dict(eps=0.05, s=1.0), cfl=0.2, desc="configs[4]: 512^3 Gaussian k^-5/3, hyperviscosity eps=0.05 s=1, CFL 0.2", cpuN=128),
}


def make_input(name: str, N: int, batch: int, rank: int = 0) -> np.ndarray:
    """Physical-space samples [batch][3][N][N][N] of the workload recipe at grid size N.  Under torchrun every rank draws
    its own Monte-Carlo samples (Algorithm 1): the seeds are offset by 10007 * rank."""
    o = 10007 * rank
    if name == "c1":
        return inputs.taylor_green_perturbed(N, seed=1 + o)[None]
    if name == "c2":
        return inputs.gaussian_k4(N, seed=2 + o)[None]
    if name == "c3":
        return inputs.shear_layer(N, seed=3 + o)[None]
    if name == "c4":
        return inputs.shear_layer_ensemble(N, batch, seed0=1000 + o)
    if name in ("c5", "n384"):
        return inputs.gaussian_k53(N, seed=5 + o)[None]
    if name == "tg3d":
        return inputs.taylor_green_3d_perturbed(N, seed=6 + o)[None]
    if name == "cyl":
        return inputs.cylindrical_shear(N, seed=7 + o, rho=0.05)[None]
    raise KeyError(name)


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def init_dist(world: int):
    """Process group for the N > 1 plumbing (barrier + max / sum of two host scalars; no data-path collective).  With GPUs:
    NCCL for CUDA tensors and gloo for the host scalars in ONE group; without (the CPU test): gloo only.  The same
    function is used by bench.py under torchrun and by tests/test_bench_host.py."""
    if world == 1:
        return None
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    backend = "cpu:gloo,cuda:nccl" if torch.cuda.is_available() else "gloo"
    if not dist.is_initialized():
        dist.init_process_group(backend)
    return dist


def host_barrier(dist):
    """Barrier over the host (gloo) side of the group: an all-reduce of a CPU scalar."""
    if dist is not None:
        import torch
        dist.all_reduce(torch.zeros(1, dtype=torch.float64))


def aggregate(local_ms_total: float, local_units: float, world: int, dist=None):
    """Max-over-ranks time and summed units; CPU tensors, i.e. the gloo side of the group."""
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
    """Time the oracle, as it stands, on a bounded sample of the workload: RK3 steps of ONE sample of the same recipe on
    a grid of at most 128^3 (a 512^3 oracle step needs ~28 GB and a quarter of an hour; its cost per grid point grows only
    with log N).  A reported baseline for context -- a deliberately naive program -- never a speed-up denominator."""
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
    sample = (f"{steps} RK3 step(s) of one sample of the {name} recipe on a {Ns}^3 grid (workload grid {w['N']}^3 x {w['batch']}), "
              "fp64, full-complex padded transforms with a naive recursive radix-2/3 FFT, OpenMP over lines")
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


def cufft_compare(torch, N: int, batch: int, dtype: str, reps: int = 3):
    """Comparison line only (north_star: "cuFFT may be timed only as a comparison line"; SURVEY.md 8(d) last paragraph): the
    transform structure of the paper's own design ("cuFFT on the device", Algorithm 2) on the same box --
    library c2r / r2c on FULLY padded arrays with separate pad, product and truncate passes -- through torch.fft (cuFFT).  One
    "RHS" = 3 padded inverse transforms, 6 pointwise products, 6 forward transforms, 6 truncations; the spectral / RK kernel is
    left out (it favours the library line).  Random data; nothing here is linked into libns.so or used by the product."""
    M, H, Hp = 3 * N // 2, N // 2 + 1, 3 * N // 4 + 1
    rt = torch.float64 if dtype == "f64" else torch.float32
    ct = torch.complex128 if dtype == "f64" else torch.complex64
    g = torch.Generator(device="cuda").manual_seed(7)
    uh = torch.view_as_complex(torch.randn(3, N, N, H, 2, dtype=rt, device="cuda", generator=g))
    pad = torch.zeros(M, M, Hp, dtype=ct, device="cuda")
    h = N // 2
    pairs = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]

    def one_rhs():
        u = []
        for c in range(3):      # Algorithm 2 steps 1-2: pad, inverse transform
            pad[:h, :h, :H] = uh[c, :h, :h]
            pad[:h, M - h:, :H] = uh[c, :h, h:]
            pad[M - h:, :h, :H] = uh[c, h:, :h]
            pad[M - h:, M - h:, :H] = uh[c, h:, h:]
            u.append(torch.fft.irfftn(pad, s=(M, M, M), norm="forward"))
        out = []
        for i, j in pairs:      # steps 3-5: product, forward transform, truncate
            bh = torch.fft.rfftn(u[i] * u[j], norm="forward")
            out.append(torch.cat([torch.cat([bh[:h, :h, :H], bh[:h, M - h:, :H]], 1), torch.cat([bh[M - h:, :h, :H], bh[M - h:, M - h:, :H]], 1)], 0))
            del bh
        return out

    try:
        one_rhs()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            one_rhs()
        b.record()
        torch.cuda.synchronize()
        ms_rhs = a.elapsed_time(b) / reps * batch      # samples one after the other
    except Exception as e:      # a comparison line must never fail the bench
        return {"unavailable": f"{type(e).__name__}: {e}"[:200]}
    finally:
        del pad, uh
        torch.cuda.empty_cache()
    return {"ms_per_rhs": ms_rhs, "ms_per_step_3_rhs": 3 * ms_rhs, "library": "cuFFT via torch.fft.irfftn / rfftn",
            "what": f"{batch} x (3 padded {M}^3 c2r + 6 products + 6 r2c + truncation), {dtype}; pad / product / truncate as separate "
                    "passes, no spectral kernel: the paper's Algorithm 2 with the library FFT, timed for context only"}


PROF_LABEL = {"a1_col_inv_x": "a1_col_inv_x", "a2_col_inv_y": "a2_col_inv_y", "a3_z_inv_prod": "a3a4_z_fused",
              "a5_col_fwd_y": "a5_col_fwd_y", "a6_col_fwd_x": "a6_col_fwd_x", "a7_spectral": "a7_spectral"}


def run_workload(binding, torch, name, dtype, steps, warmup, dist, world, rank, local, state=None, split_steps=None):
    """Time `steps` RK3 steps of one workload with the state resident in HBM (CUDA events on the solver's stream, per-pass
    profiler OFF), then a second short run with the per-pass event profiler ON for the split.  Returns (record, solver,
    extras); the caller owns the solver."""
    w = WORKLOADS[name]
    N, batch = w["N"], w["batch"]
    cbytes = 16 if dtype == "f64" else 8
    t_gen = time.perf_counter()
    s = binding.Solver(N, batch=batch, dtype=dtype, **w["params"])
    if state is None:
        u0 = make_input(name, N, batch, rank)
        chk = inputs.checksum(u0[0, 0, :2])
        s.set_initial(u0)
        del u0
    else:
        s.set_spectral(state.astype(s.cplx))
        chk = "state of the f64 run of the same workload"
    t_gen = time.perf_counter() - t_gen

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
        host_barrier(dist)
        torch.cuda.synchronize()

    for _ in range(warmup):
        one_step()
    barrier()
    launches0 = s.kernel_launches()
    sampler = ClockSampler(local)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps if flush else 1)]
    barrier()
    if flush:
        for a, b in evs:
            flush_buf.fill_(1)
            a.record()
            one_step()
            b.record()
    else:
        evs[0][0].record()
        for _ in range(steps):
            one_step()
        evs[0][1].record()
    barrier()
    total_ms = sum(a.elapsed_time(b) for a, b in evs)
    clocks = sampler.stop()
    launches = s.kernel_launches() - launches0
    # per-pass split: a second, short run with one event record between the kernels (not part of the timed value)
    nsplit = split_steps or min(steps, 5)
    s.profile(True)
    for _ in range(nsplit):
        if flush:
            flush_buf.fill_(1)
        one_step()
    prof = s.profile_read()
    s.profile(False)
    E = s.energy_spectrum(min(N, 4096))
    finite = bool(np.isfinite(E).all() and (E.sum(axis=1) > 0).all())   # finiteness of the STATE itself

    total_ms, units = aggregate(total_ms, roofline.grid_point_stages(N, batch, steps), world, dist)
    ms_per_step = total_ms / steps
    value = units / (total_ms * 1e-3)

    peak, peak_src = measured_peaks()
    per_step = roofline.pass_bytes_per_step(N, batch, cbytes)        # fixed model
    built = roofline.built_pass_bytes_per_step(N, batch, cbytes)     # what the built kernels must move
    split_ms = sum(prof[k][0] for k in PROF_LABEL) / nsplit
    kernels = {}
    for pname, label in PROF_LABEL.items():
        ms, cnt = prof[pname]
        if not cnt:
            continue
        nbytes, extra = built[label], {}
        model = per_step["a3_z_inv_prod"] + per_step["a4_z_fwd"] if label == "a3a4_z_fused" else per_step[pname]
        if model != nbytes:
            extra = {"fixed_model_bytes_per_launch": model * nsplit / cnt}
        gbs = nbytes * nsplit / (ms * 1e-3) / 1e9
        kernels[label] = {"ms_per_launch": ms / cnt, "launches": cnt, "alg_bytes_per_launch": nbytes * nsplit / cnt,
                          "gbs": gbs, "frac": gbs / peak, "share_of_step": ms / nsplit / split_ms, **extra}
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_launch"] * kernels[k]["launches"])
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            f = ln.split(",", 3)
            if len(f) >= 3 and f[0] == f"{name}_{dtype}" and f[1] in kernels:
                kernels[f[1]]["traffic"] = float(f[2])
    roof = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
            "frac": kernels[dom]["frac"], "traffic": kernels[dom].get("traffic"), "peak_source": peak_src,
            "alg_bytes_per_launch": kernels[dom]["alg_bytes_per_launch"], "ms_per_launch": kernels[dom]["ms_per_launch"]}
    if dom == "a3a4_z_fused":
        roof["note"] = ("fused a3+a4: by bytes HBM is the roofline (DRAM traffic = algorithmic 8*A2), but the kernel is bound by "
                        "fp64 issue / latency, not by HBM (profiles/); frac is bytes the kernel must move / time / measured peak")
    actual = roofline.actual_step_bytes(N, batch, cbytes)
    model_bytes = roofline.step_bytes(N, batch, cbytes)
    step_roof = {
        "bound": "hbm", "bytes_per_step": actual, "achieved_gbs": actual / (ms_per_step * 1e-3) / 1e9, "peak": peak,
        "frac": actual / (ms_per_step * 1e-3) / 1e9 / peak,
        "frac_of_nominal_8TBs": actual / (ms_per_step * 1e-3) / 1e9 / 8000.0,
        "note": "frac = bytes the BUILT pass structure must move per RK3 step (a3+a4 fused: products never reach HBM; 5 trace-free "
                "flux components) / measured time / measured HBM peak -- the HBM utilisation of the step",
        "fixed_model": {
            "bytes_per_step": model_bytes, "t_model_ms_at_measured_peak": model_bytes / (peak * 1e9) * 1e3,
            "speed_ratio_vs_model_at_measured_peak": model_bytes / (peak * 1e9) * 1e3 / ms_per_step,
            "speed_ratio_vs_model_at_nominal_8TBs": model_bytes / 8e12 * 1e3 / ms_per_step,
            "note": "SURVEY.md 8(d) fixed reference model (unfused a3 / a4, six products): T_model / T_measured, a SPEED ratio against "
                    "a pass structure that moves more bytes than this one -- it can exceed 1 and is not an HBM utilisation"},
    }
    rec = {"workload": name, "dtype": dtype, "ms_per_step": ms_per_step, "value": value, "unit": "grid-point-stages/s",
           "steps": steps, "steps_per_s": 1e3 / ms_per_step * world, "step_roofline": step_roof, "roofline": roof,
           "kernels": kernels, "clocks": clocks, "gpu_launches": launches, "state_finite": finite,
           "l2": "L2 flushed (256 MiB write) between timed steps" if flush else "inputs exceed L2 (126 MB): no flush needed",
           "input_checksum": chk, "setup_s": round(t_gen, 1), "device_bytes": s.device_bytes(),
           "profiler": f"timed region: per-pass profiler off; split from {nsplit} further step(s) with one event record per kernel"}
    return rec, s, one_step


WORKLOADS_2D = {
    # the two-dimensional solver on a large ensemble in one launch
    "e2d": dict(N=512, batch=1024, params=dict(eps=0.05, s=1.0), cfl=0.2,
                desc="NEXT-4: 1024 x 512^2 two-dimensional perturbed shear-layer ensemble in one launch, hyperviscosity eps=0.05 s=1, CFL 0.2"),
}


def run_workload_2d(binding, torch, name, dtype, steps, warmup, local, rank=0):
    """The 2-D solver on a large batch: same timing rules as run_workload (CUDA events on the solver's stream, profiler off in
    the timed region, split from a second short run)."""
    w = WORKLOADS_2D[name]
    N, batch = w["N"], w["batch"]
    cbytes = 16 if dtype == "f64" else 8
    t0 = time.perf_counter()
    u0 = np.stack([inputs.shear_layer_2d(N, 2000 + 10007 * rank + i) for i in range(batch)])
    s = binding.Solver2D(N, batch=batch, dtype=dtype, **w["params"])
    s.set_initial(u0)
    chk = inputs.checksum(u0[0])
    del u0
    setup = time.perf_counter() - t0
    for _ in range(warmup):
        s.step_cfl(w["cfl"], 1e30, return_dt=False)
    torch.cuda.synchronize()
    launches0 = s.kernel_launches()
    sampler = ClockSampler(local)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(steps):
        s.step_cfl(w["cfl"], 1e30, return_dt=False)
    b.record()
    torch.cuda.synchronize()
    total_ms = a.elapsed_time(b)
    clocks = sampler.stop()
    launches = s.kernel_launches() - launches0
    nsplit = min(steps, 5)
    s.profile(True)
    for _ in range(nsplit):
        s.step_cfl(w["cfl"], 1e30, return_dt=False)
    prof = s.profile_read()
    s.profile(False)
    E = s.energy_spectrum(N)
    finite = bool(np.isfinite(E).all() and (E.sum(axis=1) > 0).all())
    ms_per_step = total_ms / steps
    peak, peak_src = measured_peaks()
    built = roofline.built_pass_bytes_per_step_2d(N, batch, cbytes)
    split_ms = sum(prof[k][0] for k in built) / nsplit
    kernels = {}
    for k, nbytes in built.items():
        ms, cnt = prof[k]
        if cnt:
            gbs = nbytes * nsplit / (ms * 1e-3) / 1e9
            kernels[k] = {"ms_per_launch": ms / cnt, "launches": cnt, "alg_bytes_per_launch": nbytes * nsplit / cnt, "gbs": gbs,
                          "frac": gbs / peak, "share_of_step": ms / nsplit / split_ms}
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_launch"] * kernels[k]["launches"])
    actual = sum(built.values())
    model = roofline.fixed_step_bytes_2d(N, batch, cbytes)
    return {"workload": name, "desc": w["desc"], "dtype": dtype, "ms_per_step": ms_per_step, "steps": steps,
            "value": roofline.grid_point_stages_2d(N, batch, steps) / (total_ms * 1e-3), "unit": "grid-point-stages/s (2-D: batch * N^2 * 3 per step)",
            "step_roofline": {"bound": "hbm", "bytes_per_step": actual, "achieved_gbs": actual / (ms_per_step * 1e-3) / 1e9, "peak": peak,
                              "frac": actual / (ms_per_step * 1e-3) / 1e9 / peak,
                              "fixed_model": {"bytes_per_step": model, "speed_ratio_vs_model_at_measured_peak": model / (peak * 1e9) * 1e3 / ms_per_step}},
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s", "frac": kernels[dom]["frac"],
                         "traffic": None, "peak_source": peak_src},
            "kernels": kernels, "clocks": clocks, "gpu_launches": launches, "state_finite": finite, "input_checksum": chk,
            "setup_s": round(setup, 1), "device_bytes": s.device_bytes(), "l2": "inputs exceed L2 (126 MB): no flush needed"}


def run_slab(args):
    """One sample over several GPUs of this node (include/ns_mg.h): "scaling": "strong".  Needs DISTINCT
    devices -- ranks that share a GPU are how the decomposition is TESTED, never a measurement."""
    import torch
    from paper_2401_09843_b200 import binding
    devs = [int(x) for x in args.slab_devices.split(",")]
    if len(set(devs)) != len(devs) or max(devs) >= torch.cuda.device_count():
        raise SystemExit(f"--slab-devices needs distinct ordinals below {torch.cuda.device_count()} (got {devs})")
    w = WORKLOADS[args.workload]
    if w["batch"] != 1:
        raise SystemExit("the slab decomposition distributes ONE sample: use a single-sample workload (c2, c3, c5, tg3d, cyl, n384)")
    N = w["N"]
    one = binding.Solver(N, dtype=args.dtype, **w["params"])        # state from the seeded input on device 0
    one.set_initial(make_input(args.workload, N, 1))
    uh = one.get_spectral()[0]
    del one
    s = binding.SolverMG(N, devs, dtype=args.dtype, **w["params"])
    s.set_spectral(uh)
    for _ in range(args.warmup):
        s.step_cfl(w.get("cfl", 0.2), 1e30, return_dt=False)
    s.step_cfl(w.get("cfl", 0.2), 1e30)                              # synchronises every rank
    sampler = ClockSampler(devs[0])
    launches0 = s.kernel_launches()
    t0 = time.perf_counter()
    for _ in range(args.steps - 1):
        s.step_cfl(w.get("cfl", 0.2), 1e30, return_dt=False)
    s.step_cfl(w.get("cfl", 0.2), 1e30)                              # ... so the wall clock spans complete steps on all devices
    ms = (time.perf_counter() - t0) * 1e3 / args.steps
    print(json.dumps({"metric": "grid_point_stages_per_s", "value": roofline.grid_point_stages(N, 1, 1) / (ms * 1e-3),
                      "unit": "grid-point-stages/s", "n_gpus": len(devs), "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                      "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
                      "config": {"workload": w["desc"], "N": N, "parallelism": f"slab decomposition over devices {devs}, one process "
                                 "(ns_mg.h): exchanges fused into a1 / a5 as peer stores", "timer": "host wall clock around synchronised steps"},
                      "exchange_bytes_per_rhs": s.exchange_bytes(), "gpu_launches": s.kernel_launches() - launches0, "clocks": sampler.stop()}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c5", choices=sorted(WORKLOADS) + sorted(WORKLOADS_2D))
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT (torch.fft) comparison line")
    ap.add_argument("--no-also", action="store_true", help="skip the sub-records of the other north-star targets")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--slab-devices", default=None,
                    help="comma-separated DISTINCT CUDA ordinals: time ONE sample of the workload slab-decomposed over these GPUs "
                         "(include/ns_mg.h, single process; strong scaling) instead of the replica run")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.slab_devices is not None:
        return run_slab(args)

    import torch
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = init_dist(world)   # plumbing only: barrier + max/sum of two scalars
    if dist is not None:      # one NCCL collective so that a broken NVLink / NCCL setup fails here, not silently
        x = torch.ones(1, device="cuda")
        dist.all_reduce(x)
        assert int(x.item()) == world
    from paper_2401_09843_b200 import binding

    if args.workload in WORKLOADS_2D:      # the 2-D solver as the headline of this invocation (single GPU)
        r = run_workload_2d(binding, torch, args.workload, args.dtype, args.steps, args.warmup, local, rank)
        if rank == 0:
            print(json.dumps({"metric": "grid_point_stages_per_s", "value": r["value"], "unit": r["unit"], "n_gpus": 1, "steps": args.steps,
                              "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                              "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
                              "config": {"workload": r["desc"], "N": WORKLOADS_2D[args.workload]["N"], "batch_per_gpu": WORKLOADS_2D[args.workload]["batch"],
                                         "l2": r["l2"], "state_finite": r["state_finite"], "input_checksum": r["input_checksum"]},
                              "roofline": r["roofline"], "step_roofline": r["step_roofline"], "kernels": r["kernels"], "cpu_baseline": None,
                              "e2e": None, "also": {}, "gpu_launches": r["gpu_launches"], "clocks": r["clocks"], "device_bytes": r["device_bytes"]}))
        return 0

    w = WORKLOADS[args.workload]
    N, batch = w["N"], w["batch"]
    cbytes = 16 if args.dtype == "f64" else 8
    rec, s, one_step = run_workload(binding, torch, args.workload, args.dtype, args.steps, args.warmup, dist, world, rank, local)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D state, step, D2H state, every step
    e2e = None
    state64 = None
    if not args.no_e2e:
        shape = s.spectral_shape
        ct = torch.complex128 if args.dtype == "f64" else torch.complex64
        h_in = torch.empty(shape, dtype=ct).pin_memory()
        h_out = torch.empty(shape, dtype=ct).pin_memory()
        a_in, a_out = h_in.numpy(), h_out.numpy()
        s.get_spectral(a_in)
        for _ in range(1):
            s.set_spectral(a_in); one_step(); s.get_spectral(a_out)
        torch.cuda.synchronize()
        host_barrier(dist)
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
        del h_in, h_out, a_in, a_out

    # ---- the other north-star targets in the same invocation (BASELINE.json: "the 512^3 single-sample and the 32 x 128^3
    #      ensemble"; configs[4]: "plus the same run in fp32"), 10 steps each, as sub-records
    also = {}
    if args.workload == "c5" and args.dtype == "f64" and not args.no_also:
        state64 = s.get_spectral()
        del s
        r32, s32, _ = run_workload(binding, torch, "c5", "f32", 10, 3, dist, world, rank, local, state=state64)
        del s32, state64
        also["c5_f32"] = r32
        r4, s4, _ = run_workload(binding, torch, "c4", "f64", 10, 3, dist, world, rank, local)
        del s4
        also["c4_f64"] = r4
        if world == 1:
            also["e2d_f64"] = run_workload_2d(binding, torch, "e2d", "f64", 10, 3, local, rank)
    else:
        del s

    cufft = None
    if rank == 0 and world == 1 and not args.no_cufft:
        cufft = cufft_compare(torch, N, batch, args.dtype)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        nst = 20 if args.workload == "c1" else 3   # 128^3: about 6 s per step on the GPU box's 16 cores
        cpu, _ = cpu_oracle_run(args.workload, nst)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "seconds")}

    if rank == 0:
        line = {
            "metric": "grid_point_stages_per_s", "value": rec["value"], "unit": "grid-point-stages/s",
            "steps_per_s": rec["steps_per_s"], "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": rec["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": w["desc"], "N": N, "batch_per_gpu": batch, "padded": 3 * N // 2, "l2": rec["l2"],
                       "parallelism": "replicas only (independent Monte-Carlo samples per GPU, seeds offset by rank)" if world > 1 else "single GPU",
                       "input_checksum": rec["input_checksum"], "setup_s": rec["setup_s"], "state_finite": rec["state_finite"],
                       "profiler": rec["profiler"]},
            "roofline": rec["roofline"], "step_roofline": rec["step_roofline"], "kernels": rec["kernels"], "cpu_baseline": cpu,
            "e2e": e2e, "cufft_compare": cufft, "also": also, "gpu_launches": rec["gpu_launches"], "clocks": rec["clocks"], "device_bytes": rec["device_bytes"],
        }
        print(json.dumps(line))
    if dist is not None:
        host_barrier(dist)
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
