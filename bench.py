#!/usr/bin/env python
"""bench.py -- whole ABM steps of the TDSLDA/BdG path on B200 (see DESIGN.md section 7 for every definition).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4|cfg5|cfg3|cfg2|cfg1] [--n-wf n]
    python bench.py --impl reference ...       # the CPU oracle on the host cores (rank 0 only)

One "step" = one complete wslda_abm_step (Alg. 2: predictor, H P, corrector, H phi, with the densities and
potentials rebuilt at both stages when the functional is self-consistent) over the whole resident spinor
batch.  metric = quasiparticle-wavefunction time steps per second = n_wf * K / time.  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "qp_wavefunction_time_steps_per_s"
UNIT = "spinor-steps/s"


def make_workload(name, n_wf=None, kin_form=None):
    if name == "cfg1":
        return wl.cfg1(n_wf), "configs[0]: 3D BdG 8^3, fixed potentials, AB4AM4"
    if name == "cfg2":
        w = wl.cfg2()
        return w, "configs[1]: quasi-1D SLDA Nx=128, 32x32 modes x 256 spinors, self-consistent, AB4AM5"
    if name == "cfg3":
        w = wl.cfg3()
        return w, "configs[2]: quasi-2D SLDA vortex 64^2 x 16 kz, self-consistent, AB4AM5"
    if name == "cfg4":
        if kin_form in (0, 2):           # the other discretisations of the kinetic term on the same workload (comparison lines)
            form = {0: "Eq.14 Laplacian operator (alpha treated as 1 in the kinetic term)", 2: "DIVGRAD operator (3 gradient + 3 divergence transforms; general path)"}[kin_form]
            return wl.cfg4(n_wf=n_wf, kin_form=kin_form), f"configs[3] variant: 3D SLDA 32^3 trap, {form}, self-consistent, AB4AM5"
        return wl.cfg4(n_wf=n_wf), "configs[3]: 3D SLDA 32^3 trap, general-alpha Eq.40 operator, self-consistent, AB4AM5"
    if name == "cfg5":
        return wl.cfg5(n_wf=n_wf or 2048), "configs[4]: 3D ASLDA-like 64^3, h_a != h_b, fixed smooth potentials, AB4AM5"
    raise SystemExit(f"unknown config {name}")


def restrict(w, n_wf):
    """The same workload on its first n_wf spinors (mode table clipped)."""
    import copy
    v = copy.copy(w)
    v.n_wf = n_wf
    for k in ("kidx", "branch", "mode_of", "w_a", "w_b", "E"):
        a = getattr(w, k)
        if a is not None:
            setattr(v, k, a[:n_wf])
    if w.first is not None:
        v.first = np.minimum(np.asarray(w.first), n_wf)
    return v


def alg_bytes_per_spinor_step(w):
    """full-buffer accesses Alg. 2 itself needs, x 32 M bytes."""
    m = w.history
    if w.func_id == 0:
        acc = (1 + m) + 2                       # read phi, f_1..f_m; write phi_new, f_new
    else:
        acc = (1 + m) + 2 + 3 + 2               # + write P, C_part | read P, C_part, write phi | read phi, write f
    return acc * 32 * w.M


def ffts_per_spinor_step(w):
    """Transforms Alg. 2 needs per spinor-step: per component and H-apply 2 (Eq. 14), 4 (Eq. 40: w and alpha w,
    forward and inverse) or 1 + 3 nd (successive first derivatives); x 2 components x 2 H-applies."""
    per_comp = {0: 2, 1: 4, 2: 1 + 3 * w.mode}[w.kin_form]
    return 2 * 2 * per_comp


def alg_flops_per_spinor_step(w):
    return ffts_per_spinor_step(w) * 5.0 * w.M * math.log2(w.M) + 300.0 * w.M


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled in the background during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.strip().lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def make_gpu(w):
    """A CUDA context configured from the workload (product only: neither the oracle nor the test harness is imported)."""
    import paper_2602_08982_b200 as ws
    return wl.configure(ws.Context(w.mode, w.dims, w.dx, w.n_wf, **wl.context_kwargs(w)), w)


def make_oracle(w):
    import oracle as orc
    return wl.configure(orc.Oracle(w.mode, w.dims, w.dx, w.n_wf, **wl.context_kwargs(w)), w)


def time_oracle(w, budget_s=20.0, steps=2):
    """The oracle as it stands on the host cores: abm steps on the first n_sub spinors of the workload."""
    import oracle as orc                     # the only legs that touch oracle/: cpu_baseline and --impl reference
    threads = orc.num_threads()
    n_sub = min(w.n_wf, max(threads, 1) * 2)
    best = None
    while True:
        ws_ = restrict(w, n_sub)
        o = make_oracle(ws_)
        phi = ws_.spinors()
        hist = [np.zeros_like(phi) for _ in range(o.m)]
        hist = o.abm_init(phi, hist, ws_.dt, 0)
        t0 = time.perf_counter()
        for _ in range(steps):
            hist = o.abm_step(phi, hist, ws_.dt)
        dt = time.perf_counter() - t0
        best = (n_sub, dt)
        if dt >= budget_s / 4 or n_sub >= w.n_wf or n_sub * 32 * w.M * (o.m + 2) > 8e9:
            break
        n_sub = min(w.n_wf, int(n_sub * min(8.0, max(2.0, budget_s / 2 / max(dt, 1e-3)))))
    n_sub, dt = best
    return {"value": n_sub * steps / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{steps} abm steps on the first {n_sub} of {w.n_wf} spinors (zero-history start), {dt:.2f} s; "
                      f"cost is linear in n_wf (PAPER.md:1053)"}, dt / steps * 1e3


def run_reference(args):
    """--impl reference: W + K abm steps of the oracle on a bounded sample of the workload (host cores)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, desc = make_workload(args.config, args.n_wf, args.kin_form)
    if getattr(args, "friction", False):
        w.friction = dict(qf_alpha=6.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.03, qf_nreq=float(np.sum(np.asarray(w.w_a) + np.asarray(w.w_b))))
        desc += " + quantum friction (Eqs. 66-70)"
    if getattr(args, "polarised", False):
        w.spin_symmetric = 0
        w.w_a = 0.6 * np.asarray(w.w_b)
        desc += " (polarised: w_a = 0.6 w_b, tau rebuilt every stage)"
    if getattr(args, "force_a1", False):
        w.force_a1 = 1
        desc += " (alpha = 1: force_a1)"
    if getattr(args, "velocity", 0.0):
        Mv, ndv = int(np.prod(w.shape)), len(w.shape)
        vv = args.velocity * wl.normal(977, 0, 6 * Mv).reshape(2, 3, *w.shape)
        w.current_terms = 1
        w.vel = (vv[0, :ndv], vv[1, :ndv])
        desc += f" + external velocity fields (amplitude {args.velocity}) through the coupling of Eq. 4c"
    import oracle as orc
    orc.build()
    cal, _ = time_oracle(w, budget_s=4.0, steps=1)                 # calibration: spinor-steps/s
    total = args.steps + args.warmup
    n_sub = int(min(w.n_wf, max(orc.num_threads(), cal["value"] * 90.0 / total)))
    n_sub = int(min(n_sub, 8e9 / (32 * w.M * (w.history + 2))))
    ws_ = restrict(w, n_sub)
    o = make_oracle(ws_)
    phi = ws_.spinors()
    hist = [np.zeros_like(phi) for _ in range(o.m)]
    hist = o.abm_init(phi, hist, ws_.dt, 0)
    for _ in range(args.warmup):
        hist = o.abm_step(phi, hist, ws_.dt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        hist = o.abm_step(phi, hist, ws_.dt)
    dt = time.perf_counter() - t0
    v = n_sub * args.steps / dt
    sample = f"{args.steps} abm steps on the first {n_sub} of {w.n_wf} spinors (zero-history start), {dt:.2f} s"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128",
                      "data": "synthetic", "config": {"workload": desc, "n_wf": w.n_wf, "M": w.M},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                                       "sample": sample},
                      "gpu_launches": 0,
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def max_over_ranks(ms, world, device):
    """Multi-GPU timing rule: the step time of the job is the MAX over ranks of the device-timed region."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(n_wf_per_rank, steps, world, ms):
    """Whole-job throughput of `world` independent replicas (weak scaling, no data-path collective)."""
    return world * n_wf_per_rank * steps / (ms * 1e-3)


def run_gpu(args):
    import torch
    import torch.distributed as dist
    import paper_2602_08982_b200 as ws

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if os.environ.get("NCCL_DEBUG", "VERSION").upper() == "VERSION":
        os.environ["NCCL_DEBUG"] = "WARN"              # keep NCCL's version banner off stdout: rank 0 prints ONE JSON line
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    elif args.shard:                                   # a 1-rank group, so that the collective path can be run on one GPU
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29655", rank=0, world_size=1,
                                device_id=torch.device("cuda", local))
    ws.build()
    w, desc = make_workload(args.config, args.n_wf, args.kin_form)
    if getattr(args, "friction", False):
        w.friction = dict(qf_alpha=6.0, qf_beta=5.0, qf_gamma=0.1, qf_rho0=0.03, qf_nreq=float(np.sum(np.asarray(w.w_a) + np.asarray(w.w_b))))
        desc += " + quantum friction (Eqs. 66-70)"
    if getattr(args, "polarised", False):
        w.spin_symmetric = 0
        w.w_a = 0.6 * np.asarray(w.w_b)
        desc += " (polarised: w_a = 0.6 w_b, tau rebuilt every stage)"
    if getattr(args, "force_a1", False):
        w.force_a1 = 1
        desc += " (alpha = 1: force_a1)"
    if getattr(args, "velocity", 0.0):
        Mv, ndv = int(np.prod(w.shape)), len(w.shape)
        vv = args.velocity * wl.normal(977, 0, 6 * Mv).reshape(2, 3, *w.shape)
        w.current_terms = 1
        w.vel = (vv[0, :ndv], vv[1, :ndv])
        desc += f" + external velocity fields (amplitude {args.velocity}) through the coupling of Eq. 4c"
    w_full, n_lo = w, 0
    if args.shard:                                     # shard the spinor index, all-reduce the densities
        n_lo, n_hi = wl.shard_range(w_full.n_wf, rank, world)
        w = wl.shard(w_full, n_lo, n_hi)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md 6.65 TB/s)"
    fp64_peak, n_sm = ws.fp64_probe()          # measured now, on this device: dependent-chain DFMA kernel (wslda_fp64_probe)
    fp64_src = (f"measured in this run: DFMA-chain probe {fp64_peak / 1e12:.2f} TFLOP/s on {n_sm} SMs "
                f"(nominal {n_sm} x 64 lanes x 2 x 1.965 GHz = {n_sm * 64 * 2 * 1.965e9 / 1e12:.1f})")

    # ---- resident state: every rank holds its own replica of the workload ("replicas only")
    g = make_gpu(w)
    if args.shard:
        g.set_density_allreduce()
    shape = (w.n_wf, 2) + w.shape
    phi = torch.empty(shape, dtype=torch.complex128, device="cuda")
    wl.spinors_device(w_full, n_lo, n_lo + w.n_wf, phi)
    hist = [torch.zeros(shape, dtype=torch.complex128, device="cuda") for _ in range(g.m)]
    torch.cuda.synchronize()
    hist = g.abm_init(phi, hist, w.dt, 0)            # zero-history start: the timed steps are plain Alg. 2 steps
    sampler = ClockSampler(local) if rank == 0 else None      # samples through the warm-up and the timed steps (same load)
    for _ in range(args.warmup):
        hist = g.abm_step(phi, hist, w.dt)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        hist = g.abm_step(phi, hist, w.dt)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = max_over_ranks(ms, world, "cuda")
    finite = bool(torch.isfinite(torch.view_as_real(phi[:: max(1, w.n_wf // 64)])).all())
    value = w_full.n_wf * args.steps / (ms * 1e-3) if args.shard else job_value(w.n_wf, args.steps, world, ms)

    # ---- per-kernel device times (separate pass, event pairs around every launch) -> dominant kernel
    prof_steps = min(args.steps, 2)
    g.profile(True)
    for _ in range(prof_steps):
        hist = g.abm_step(phi, hist, w.dt)
    rep = g.profile_report()
    g.profile(False)
    # launches on the three stage-1 streams overlap: rank and share by the attributed time (it adds up to the busy
    # time), keep the raw event-pair duration for the kernel's own achieved rate
    tot_ms = sum(v[4] for v in rep.values()) or 1.0
    kern = sorted(rep.items(), key=lambda kv: -kv[1][4])
    top, (top_cnt, top_ms, top_bytes, top_flops, top_share) = kern[0]
    t_b, t_f = top_bytes / (hbm_peak * 1e9), top_flops / fp64_peak
    if t_b >= t_f:
        ach = top_bytes / (top_ms * 1e-3) / 1e9
        roof = {"kernel": top, "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                "traffic": None, "peak_source": peak_src}
    else:
        ach = top_flops / (top_ms * 1e-3) / 1e12
        roof = {"kernel": top, "bound": "alu", "achieved": ach, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                "frac": ach / (fp64_peak / 1e12), "traffic": None, "peak_source": fp64_src}
    # `traffic` (DRAM bytes per launch) is an ncu figure and is not measured by this run: see profiles/ for the captures
    roof["traffic_note"] = "not measured in a bench run; ncu --set full captures of this kernel are summarised under profiles/"
    roof.update({"share_of_step": top_share / tot_ms, "launches_per_step": top_cnt / prof_steps,
                 "avg_launch_ms": top_ms / top_cnt, "alg_bytes_per_launch": top_bytes / top_cnt,
                 "alg_flops_per_launch": top_flops / top_cnt})
    B, F = alg_bytes_per_spinor_step(w), alg_flops_per_spinor_step(w)
    t_roof = max(B / (hbm_peak * 1e9), F / fp64_peak)
    step_roof = {"bound": "hbm" if B / (hbm_peak * 1e9) >= F / fp64_peak else "alu",
                 "t_roof_us_per_spinor_step": t_roof * 1e6, "t_measured_us_per_spinor_step": 1e6 * world / value,
                 "frac": t_roof * value / world, "bytes_per_spinor_step": B, "flops_per_spinor_step": F,
                 "hbm_gbs_achieved": B * value / world / 1e9, "hbm_peak_gbs": hbm_peak, "fp64_peak_tflops": fp64_peak / 1e12,
                 "fp64_peak_source": fp64_src}
    kernels = {k: {"launches_per_step": v[0] / prof_steps, "ms_per_step": round(v[1] / prof_steps, 4),
                   "attributed_ms_per_step": round(v[4] / prof_steps, 4), "share": round(v[4] / tot_ms, 4)} for k, v in kern}
    del hist, phi
    torch.cuda.empty_cache()
    cmp_cufft = None
    if rank == 0 and not args.no_cufft and not args.shard:
        try:
            cmp_cufft = cufft_compare(w, g)
        except RuntimeError as e:                          # out of memory for the library's temporaries: report, do not fail
            cmp_cufft = {"error": str(e)[:200]}

    # ---- end to end: the same step through wslda_abm_step_host (pinned HOST buffers, copies inside the timed region)
    e2e = None
    if not args.no_e2e and not args.shard:
        n_e = min(w.n_wf, max(1, int(2 ** 31 // (32 * w.M))))          # <= 2 GiB per buffer on the host
        we = restrict(w, n_e)
        del g
        torch.cuda.empty_cache()
        ge = make_gpu(we)
        shp = (n_e, 2) + w.shape
        dphi = torch.empty(shp, dtype=torch.complex128, device="cuda")
        wl.spinors_device(we, 0, n_e, dphi)
        dh = [torch.zeros(shp, dtype=torch.complex128, device="cuda") for _ in range(ge.m)]
        dh = ge.abm_init(dphi, dh, w.dt, 0)
        hphi = torch.empty(shp, dtype=torch.complex128).pin_memory()
        hphi.copy_(dphi)
        hh = [torch.zeros(shp, dtype=torch.complex128).pin_memory() for _ in range(ge.m)]
        hh, dh = ge.abm_step_host(hphi, hh, dphi, dh, w.dt)               # warm-up
        barrier()
        t0 = time.perf_counter()
        e0.record()
        n_e2e_steps = max(1, min(args.steps, 3))
        for _ in range(n_e2e_steps):
            hh, dh = ge.abm_step_host(hphi, hh, dphi, dh, w.dt)
        e1.record()
        barrier()
        ms_e = e0.elapsed_time(e1)
        ms_e = max_over_ranks(ms_e, world, "cuda")
        buf = n_e * 32 * w.M
        e2e = {"value": world * n_e * n_e2e_steps / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": buf * (1 + ge.m),
               "d2h_bytes_per_step": 2 * buf, "n_wf": n_e, "steps": n_e2e_steps,
               "note": "wslda_abm_step_host: phi + m history buffers copied host->device, phi_new and f_new device->host, every step"}
        del ge, dphi, dh, hphi, hh
        torch.cuda.empty_cache()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle as orc
        orc.build()
        cpu, _ = time_oracle(w, budget_s=20.0, steps=2)

    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
               "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None,
               "dtype": "c128", "data": "synthetic",
               "config": {"workload": desc, "name": w.name, "n_wf_per_gpu": w.n_wf, "M": w.M, "mode": w.mode,
                          "tuning": args.tuning or "defaults", "kin_form": w.kin_form, "func_id": w.func_id, "ab_am": [w.ab_order, w.am_order], "dt": w.dt,
                          "resident_bytes": (1 + w.history) * w.n_wf * 32 * w.M, "parallelism": (f"spinor index sharded x{world}, one NCCL all-reduce of the density block per density build"
                                          if args.shard else f"replicas x{world}"),
                          "l2": "inputs larger than L2 (no flush)" if (1 + w.history) * w.n_wf * 32 * w.M > 4e8
                                else "working set near L2 size: numbers are L2-assisted"},
               "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "step_roofline": step_roof,
               "kernels": kernels, "cpu_baseline": cpu, "cufft_compare": cmp_cufft, "finite": finite}
        print(json.dumps(out))
    if world > 1 or args.shard:
        dist.destroy_process_group()


def cufft_compare(w, g, n_cmp=256, reps=3):
    """H psi by library transforms as an outside yardstick ("cuFFT-based H psi is timed as a second
    comparison only"): torch.fft (cuFFT) forward / inverse 3-D transforms of w and alpha w plus the pointwise BdG mix in
    torch ops, against wslda_apply_h on the same spinors.  Same operator (Eq. 40 / Eq. 14 per w.kin_form); fields
    read back from the context.  Not part of the product path."""
    import torch
    if w.mode != 3 or w.kin_form == 2:
        return None
    n = min(w.n_wf, n_cmp)
    shape = (w.n_wf, 2) + w.shape
    psi = torch.empty(shape, dtype=torch.complex128, device="cuda")
    wl.spinors_device(w, 0, w.n_wf, psi)
    F = {k: g.get_field(k) for k in ("alpha_a", "alpha_b", "U_a", "U_b", "delta", "lap_alpha_a", "lap_alpha_b")}
    ks = [torch.as_tensor(wl.kgrid(w.dims[d], w.dx[d]), device="cuda") for d in range(3)]
    k2 = ks[0][:, None, None] ** 2 + ks[1][None, :, None] ** 2 + ks[2][None, None, :] ** 2
    mu = w.mu

    def lap(x):
        return torch.fft.ifftn(-k2 * torch.fft.fftn(x, dim=(-3, -2, -1)), dim=(-3, -2, -1))

    def hpsi(p):
        u, v = p[:, 0], p[:, 1]
        if w.kin_form == 1:
            ku = -0.25 * (lap(F["alpha_a"] * u) + F["alpha_a"] * lap(u) - F["lap_alpha_a"] * u)
            kv = -0.25 * (lap(F["alpha_b"] * v) + F["alpha_b"] * lap(v) - F["lap_alpha_b"] * v)
        else:
            ku, kv = -0.5 * lap(u), -0.5 * lap(v)
        hu = ku + (F["U_a"] - mu[0]) * u + F["delta"] * v
        hv = torch.conj(F["delta"]) * u - (kv + (F["U_b"] - mu[1]) * v)
        return torch.stack([hu, hv], 1)

    ev = lambda: torch.cuda.Event(enable_timing=True)
    sub = psi[:n]
    ref = hpsi(sub)                                         # warm-up (cuFFT plans) + cross-check
    out = torch.empty_like(psi)
    eps = torch.zeros(w.n_wf, dtype=torch.float64, device="cuda")
    g.apply_h(psi, out, eps, 0, n)
    err = float((out[:n] - ref).abs().max() / ref.abs().max())
    t = {}
    for name, fn in (("cufft", lambda: hpsi(sub)), ("wslda", lambda: g.apply_h(psi, out, eps, 0, n))):
        e0, e1 = ev(), ev()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record(); e1.synchronize()
        t[name] = e0.elapsed_time(e1) / reps
    del psi, out, ref
    torch.cuda.empty_cache()
    return {"what": "H psi on %d spinors: torch.fft (cuFFT) transforms + torch pointwise ops vs wslda_apply_h" % n,
            "cufft_spinors_per_s": n / (t["cufft"] * 1e-3), "wslda_spinors_per_s": n / (t["wslda"] * 1e-3),
            "speedup": t["cufft"] / t["wslda"], "max_rel_difference": err}


def run_sweep(args):
    """configs[4] as BASELINE.json words it: resident batches of 512 / 1024 / 2048 spinors streamed over 32768
    wavefunctions on the 64^3 lattice (R23: device-resident batches, re-used; no host traffic in the timed path), with
    H psi, the accumulation of ALL density fields (rho, nu, tau, j; accumulate = 1 across the batches) and the ABM step
    timed separately with CUDA events.  One JSON line per batch size."""
    import torch
    import paper_2602_08982_b200 as ws
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep needs a CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    ws.build()
    total = args.sweep_total
    fp64_peak, n_sm = ws.fp64_probe()
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    for batch in [int(b) for b in args.sweep_batches.split(",")]:
        w, desc = make_workload("cfg5", batch)
        g = make_gpu(w)
        shape = (batch, 2) + w.shape
        phi = torch.empty(shape, dtype=torch.complex128, device="cuda")
        wl.spinors_device(w, 0, batch, phi)
        hpsi = torch.empty_like(phi)
        eps = torch.zeros(batch, dtype=torch.float64, device="cuda")
        hist = [torch.zeros(shape, dtype=torch.complex128, device="cuda") for _ in range(g.m)]
        hist = g.abm_init(phi, hist, w.dt, 0)
        nb = max(1, total // batch)
        ev = lambda: torch.cuda.Event(enable_timing=True)
        for _ in range(2):                                     # warm-up of every piece
            g.apply_h(phi, hpsi, eps); g.densities(phi); hist = g.abm_step(phi, hist, w.dt)
        torch.cuda.synchronize()
        t = {"h_psi": 0.0, "densities_all": 0.0, "abm_step": 0.0}
        l0 = g.launch_count()
        sampler = ClockSampler(torch.cuda.current_device())
        for b in range(nb):
            for key, fn in (("h_psi", lambda: g.apply_h(phi, hpsi, eps)),
                            ("densities_all", lambda: g.densities(phi, accumulate=1 if b else 0)),
                            ("abm_step", lambda: g.abm_step(phi, hist, w.dt))):
                e0, e1 = ev(), ev()
                e0.record()
                r = fn()
                e1.record()
                e1.synchronize()
                t[key] += e0.elapsed_time(e1)
                if key == "abm_step":
                    hist = r
        clocks = sampler.stop()
        launches = g.launch_count() - l0
        n_done = nb * batch
        M = w.M
        per = {k: v * 1e3 / n_done for k, v in t.items()}      # us per spinor
        lg = math.log2(M)
        # algorithmic work per spinor: H psi reads + writes a spinor, 8 transforms (Eq. 40, w and alpha w,
        # two components, forward + inverse); densities read a spinor, 2 forward + 6 inverse transforms for the gradients
        alg = {"h_psi": (64.0 * M, 8 * 5.0 * M * lg), "densities_all": (32.0 * M, 8 * 5.0 * M * lg),
               "abm_step": (alg_bytes_per_spinor_step(w), alg_flops_per_spinor_step(w))}
        roof = {k: max(by / (hbm_peak * 1e9), fl / fp64_peak) * 1e6 for k, (by, fl) in alg.items()}
        out = {"metric": METRIC, "value": n_done / (t["abm_step"] * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": nb, "warmup": 2,
               "ms_per_step": t["abm_step"] / nb, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
               "dtype": "c128", "data": "synthetic",
               "config": {"workload": desc + f"; sweep: resident batch {batch}, {nb} batches = {n_done} wavefunctions",
                          "resident_batch": batch, "wavefunctions": n_done, "M": M, "kin_form": w.kin_form,
                          "l2": "inputs larger than L2 (no flush)"},
               "pieces_us_per_spinor": per,
               "pieces_spinors_per_s": {k: 1e6 / v for k, v in per.items()},
               "pieces_roofline_frac": {k: roof[k] / per[k] for k in per},
               "pieces_alg_bytes_flops_per_spinor": {k: list(v) for k, v in alg.items()},
               "peaks": {"hbm_gbs": hbm_peak, "fp64_tflops": fp64_peak / 1e12},
               "clocks": clocks, "gpu_launches": launches}
        print(json.dumps(out), flush=True)
        del g, phi, hpsi, hist
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="wslda", choices=["wslda", "reference"])
    ap.add_argument("--config", default="cfg4")
    ap.add_argument("--n-wf", type=int, default=None)
    ap.add_argument("--kin-form", type=int, default=None, choices=[0, 1, 2],
                    help="cfg4 only: time another discretisation of the kinetic term (0 Eq. 14, 2 DIVGRAD) instead of Eq. 40")
    ap.add_argument("--velocity", type=float, default=0.0,
                    help="add seeded external velocity fields of this amplitude (NEXT-1 current / velocity coupling, Eq. 4c) to the workload")
    ap.add_argument("--force-a1", action="store_true", help="SLDA with alpha = 1 (the functional's force_a1 switch) on the chosen workload")
    ap.add_argument("--polarised", action="store_true",
                    help="both spin densities populated (w_a = 0.6 w_b, no spin folding): alpha_sigma depends on p and tau enters V_sigma")
    ap.add_argument("--friction", action="store_true",
                    help="quantum friction (NEXT-3, Eqs. 66-70): j and B' rebuilt at both stages, dissipative terms in V and Delta")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: shard the spinor index over the ranks (strong scaling, density all-reduce) instead of replicas")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT-based H psi comparison leg")
    ap.add_argument("--tuning", default="", help="wslda_set_tuning fields, e.g. enable_tma_stage=1,tma_group=8 (kernel selection only)")
    ap.add_argument("--sweep", action="store_true",
                    help="configs[4]: resident batches streamed over --sweep-total wavefunctions, pieces timed separately")
    ap.add_argument("--sweep-batches", default="512,1024,2048")
    ap.add_argument("--sweep-total", type=int, default=32768)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.tuning:
        import paper_2602_08982_b200 as ws
        ws.build()
        ws.set_tuning(**{k: (float(v) if "." in v else int(v)) for k, v in (kv.split("=") for kv in args.tuning.split(","))})
    if args.sweep:
        return run_sweep(args)
    run_gpu(args)


if __name__ == "__main__":
    main()
