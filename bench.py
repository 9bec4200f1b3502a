#!/usr/bin/env python
"""bench.py -- time steps/s of the nsCouette predictor-corrector step (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5]

One "step" = one ``nsc_step``: 2 nonlinear evaluations (N1-N6) + 2 implicit sub-steps (L1-L5),
i.e. every row of SURVEY.md 8(a), on the synthetic fields of DESIGN.md "Input recipe".
Default workload: BASELINE.json configs[3] (N_r = 256, M_theta = K_z = 256), the configuration
the metric and the north-star target are quoted on.

--gpus N > 1 (under torchrun): the path is single-GPU by BASELINE.json ("Everything runs on one
GPU"); ranks run independent replicas (replicas only, no collective on
the data path), timed as the max over ranks after a barrier; value = N * steps / time.

--impl reference: times the oracle (oracle/nsc_oracle.py, as it stands) on the host cores on a
bounded sample of the same workload (see ``oracle_sample``); rank 0 only.

Prints ONE JSON line.  Never reads /root/reference.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "time steps/s at N_r x M_theta x K_z (fp64)"
NOMINAL_HBM_GBS = 8000.0            # BASELINE.json: "achieved HBM GB/s vs 8 TB/s peak"
FALLBACK_HBM_GBS = 6650.0           # /opt/skills/guides/B200_PROFILING.md fallback


# ------------------------------------------------------------------------------------------
# byte / flop models
# ------------------------------------------------------------------------------------------
def sizes(cfg):
    N_r, M, K = cfg["N_r"], cfg["M"], cfg["K"]
    nf = 4 if cfg["Ra"] != 0.0 else 3
    Nt, Nz = 3 * M, 3 * K
    F = N_r * (M + 1) * (2 * K + 1) * 16            # bytes of one spectral field
    I = N_r * (M + 1) * Nz * 16                     # bytes of one half-transformed field
    return dict(N_r=N_r, M=M, K=K, nf=nf, Nt=Nt, Nz=Nz, F=F, I=I)


def algorithmic_bytes(cfg):
    """Per-kernel algorithmic bytes PER STEP (two nonlinear evaluations + predictor + corrector)
    and the step total B_step = 2 (2 nf F + 6 nf I) + (7 nf + 3) F."""
    s = sizes(cfg)
    nf, F, I = s["nf"], s["F"], s["I"]
    per = {
        # nonlinear, two-pass 2-D transform: z pass <-> theta pass through one round trip
        "k_zinv": 2 * (nf * F + 2 * nf * I),            # read f once, write f and dz f half-transformed
        "k_theta": 2 * (2 * nf * I + nf * I),           # read 2 nf, write nf half-transformed products
        "k_zfwd": 2 * (nf * I + nf * F),
        # linear stage: predictor (3 nf + 1) F, corrector (4 nf + 2) F, shared out over its kernels
        "linear": (7 * nf + 3) * F,
    }
    per["step"] = per["k_zinv"] + per["k_theta"] + per["k_zfwd"] + per["linear"]
    return per


def flops_per_nonlinear(cfg):
    """5 N log2 N per complex line, half for real lines, + 22/30 flop per physical point."""
    s = sizes(cfg)
    N_r, M, nf, Nt, Nz = s["N_r"], s["M"], s["nf"], s["Nt"], s["Nz"]
    import math
    zl = 5 * Nz * math.log2(Nz)
    tl = 2.5 * Nt * math.log2(Nt)
    inv = N_r * ((M + 1) * 2 * nf * zl + Nz * 4 * nf * tl)
    fwd = N_r * (Nz * nf * tl + (M + 1) * nf * zl)
    return inv + fwd + N_r * Nt * Nz * (22 if nf == 3 else 30)


LINEAR_KERNELS = ("k_rhs_fwd", "k_bwd_div", "k_poisson_fwd", "k_poisson_bwd_correct")

# nominal fp64 peak of the plain DFMA pipe (context; the roofline uses the peaks measured by nsc_fp64_peak):
# 148 SM x 64 lanes x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12

def ncu_traffic(kernel, config):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of ``kernel`` at BASELINE config ``config`` from the
    committed `ncu --set full` capture (profiles/r02_ncu_traffic.csv: kernel, config, bytes per launch, capture), or
    (None, None) if that kernel was not captured."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_traffic.csv")
    try:
        with open(path) as fh:
            for line in fh:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) >= 4 and parts[0] == kernel and parts[1] == str(config):
                    return float(parts[2]), parts[3]
    except OSError:
        pass
    return None, None


def flops_theta_per_nonlinear(cfg):
    """The theta kernel's share of flops_per_nonlinear: 4 nf inverse + nf forward real lines of length
    N_theta per (j, z) point-line (2.5 N log2 N each) + the physical-space products."""
    import math
    s = sizes(cfg)
    tl = 2.5 * s["Nt"] * math.log2(s["Nt"])
    return s["N_r"] * s["Nz"] * (5 * s["nf"] * tl + s["Nt"] * (22 if s["nf"] == 3 else 30))


# ------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        with open(self.path) as fh:
            for line in fh:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    sm.append(float(parts[0]))
                    mx.append(float(parts[1]))
                except ValueError:
                    continue
                for nm, v in zip(names, parts[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        os.unlink(self.path)
        if not sm:
            return None
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_sample(cfg, n_nodes=8, n_modes=512):
    """Times the oracle, as it stands, on a bounded sample of ``cfg`` and extrapolates one step:
      - nonlinear term (naive-DFT backend) at ``n_nodes`` radial nodes spread over the gap, with
        the full (M+1) x (2K+1) mode set -> seconds per node;
      - one implicit sub-step (dense equilibrated LU per mode) on ``n_modes`` Fourier modes of an
        N_r-node problem (m <= 4, |k| <= K; the cost per mode does not depend on m) -> s per mode;
      step = 2 * N_r * t_node + 2 * N_modes * t_mode.
    Returns (seconds per step, description, threads)."""
    from oracle.nsc_oracle import Oracle, Params, radial_grid
    from paper_1908_00587_b200 import synth
    nf = 4 if cfg["Ra"] != 0.0 else 3
    N_r, M, K = cfg["N_r"], cfg["M"], cfg["K"]
    r = radial_grid(N_r, cfg["eta"], cfg["grid"])
    st = synth.make_state(cfg, r)
    o = Oracle(Params(**{k: cfg[k] for k in synth.PHYS_KEYS}))
    n_nodes = min(n_nodes, N_r)
    nodes = np.unique(np.linspace(0, N_r - 1, n_nodes).round().astype(int))
    t0 = time.perf_counter()
    o.nonlinear(*st[:nf], nodes=nodes)
    t_node = (time.perf_counter() - t0) / len(nodes)
    # linear stage on a slab of modes
    Ms = min(M, 4)
    cfg_s = dict(cfg)
    cfg_s["M"] = Ms
    st_s = [None if a is None else np.ascontiguousarray(a[:, :Ms + 1, :]) for a in st]
    o_s = Oracle(Params(**{k: cfg_s[k] for k in synth.PHYS_KEYS}))
    E = [0.1 * a for a in st_s[:nf]]
    total = (Ms + 1) * (2 * K + 1)
    nm = min(n_modes, total)
    IM, IK = np.divmod(np.arange(nm), 2 * K + 1)
    t0 = time.perf_counter()
    o_s.substep(st_s, E, cfg["dt"], modes=(IM, IK))
    t_mode = (time.perf_counter() - t0) / nm
    n_modes_all = (M + 1) * (2 * K + 1)
    t_step = 2 * N_r * t_node + 2 * n_modes_all * t_mode
    threads = os.cpu_count() or 1
    try:
        from threadpoolctl import threadpool_info
        ths = [d.get("num_threads", 1) for d in threadpool_info()]
        if ths:
            threads = max(ths)
    except Exception:
        pass
    desc = (f"oracle nonlinear (naive DFT) at {len(nodes)} of {N_r} radial nodes + oracle sub-step "
            f"(dense LU) on {nm} of {n_modes_all} modes; step = 2*N_r*t_node + 2*N_modes*t_mode "
            f"(t_node {t_node:.3g} s, t_mode {t_mode:.3g} s)")
    return t_step, desc, threads


# ------------------------------------------------------------------------------------------
def run_reference(args, cfg, rank):
    if rank != 0:
        return
    w = max(0, min(args.warmup, 1))
    k = max(1, min(args.steps, 2))
    for _ in range(w):
        oracle_sample(cfg, n_nodes=2, n_modes=64)
    ts = []
    for _ in range(k):
        t_step, desc, threads = oracle_sample(cfg)
        ts.append(t_step)
    t = sum(ts) / len(ts)
    s = sizes(cfg)
    val = 1.0 / t
    out = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "steps/s", "n_gpus": args.gpus,
        "steps": k, "warmup": w, "ms_per_step": 1e3 * t, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "N_r": s["N_r"], "M_theta": s["M"], "K_z": s["K"],
                   "physical_grid": [s["Nt"], s["Nz"]], "dt": cfg["dt"]},
        "cpu_baseline": {"value": val, "unit": "steps/s", "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def workload_name(cfg):
    s = sizes(cfg)
    return (f"BASELINE.json configs[{cfg['index']}]: N_r={s['N_r']}, M_theta={s['M']}, K_z={s['K']}, "
            f"eta={cfg['eta']}, k_theta0={cfg['k_theta0']}, Re_i={cfg['Re_i']:g}, Re_o={cfg['Re_o']:g}, "
            f"Ra={cfg['Ra']:g}, temperature {'on' if s['nf'] == 4 else 'off'}")


def time_extra_config(ci, args, stream):
    """Device-resident steps/s of another BASELINE.json configuration in the same run (parity-test cases, not the
    headline: 3 warm-up steps, then args.steps timed steps), with the per-kernel CUDA-event times."""
    import torch
    from paper_1908_00587_b200 import nsc, synth
    cfg = synth.config(ci - 1)
    cfg["index"] = ci - 1
    model = algorithmic_bytes(cfg)
    with nsc.Context.from_config(cfg) as ctx:
        ctx.set_stream(stream)
        st = synth.make_state(cfg, ctx.grid())
        ctx.set_state(*st)
        del st
        nsteps = args.steps if ci < 5 else min(args.steps, 3)
        for _ in range(3):
            ctx.step(cfg["dt"])
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(nsteps):
            ctx.step(cfg["dt"])
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / nsteps
        ctx.set_profiling(True)
        ctx.profile_read()
        for _ in range(nsteps):
            ctx.step(cfg["dt"])
        prof = ctx.profile_read()
        ctx.set_profiling(False)
        dev_bytes = ctx.device_bytes()
    peak, _ = measured_peaks()
    return {"workload": workload_name(cfg), "ms_per_step": ms, "steps_per_s": 1e3 / ms,
            "step_algorithmic_GB": model["step"] / 1e9, "step_frac_of_measured_hbm": model["step"] / 1e6 / ms / peak,
            "device_bytes": dev_bytes,
            "steps": nsteps,
            "kernels_ms_per_step": {n: k / nsteps for n, (k, c) in prof.items() if c and n != "k_factor"}}


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    from paper_1908_00587_b200 import build, nsc, synth, replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if rank == 0:
        build.build()
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    nsc.load_library()
    s = sizes(cfg)
    nf, F = s["nf"], s["F"]
    dt = cfg["dt"]
    stream = torch.cuda.Stream()            # a non-default stream: nsc_step replays its CUDA graph on it
    torch.cuda.set_stream(stream)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    with nsc.Context.from_config(cfg, radial_chunk=args.radial_chunk, linear_slices=args.linear_slices) as ctx:
        ctx.set_stream(stream)
        st = synth.make_state(replicas.rank_config(cfg, rank), ctx.grid())
        # pinned host copies of the state (inputs of a step) and of the result
        names = [0, 1, 2] + ([3] if nf == 4 else []) + [4]
        pin_in, pin_out = {}, {}
        for i in names:
            t = torch.empty(st[i].shape, dtype=torch.complex128, pin_memory=True)
            t.numpy()[...] = st[i]
            pin_in[i] = t
            pin_out[i] = torch.empty(st[i].shape, dtype=torch.complex128, pin_memory=True)
        del st
        host_in = [pin_in[i].numpy() if i in pin_in else None for i in range(5)]
        host_out = [pin_out[i].numpy() if i in pin_out else None for i in range(5)]
        ctx.set_state(*host_in)

        # ---- device-resident timing: W warm-up steps, then exactly K steps between events
        for _ in range(args.warmup):
            ctx.step(dt)
        barrier()
        clocks = ClockSampler(local_rank)
        if rank == 0:
            clocks.start()
        l0 = ctx.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(args.steps):
            ctx.step(dt)
        ev1.record(stream)
        barrier()
        ms = ev0.elapsed_time(ev1)
        launches = ctx.launch_count() - l0
        clk = clocks.stop() if rank == 0 else None
        ms = replicas.max_over_ranks(ms, dist, "cuda")
        ms_per_step = ms / args.steps

        # ---- per-kernel CUDA-event timing of the same K steps (events bracket every launch)
        ctx.set_profiling(True)
        ctx.profile_read()
        evp0, evp1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        evp0.record(stream)
        for _ in range(args.steps):
            ctx.step(dt)
        evp1.record(stream)
        prof = ctx.profile_read()
        ms_prof_per_step = evp0.elapsed_time(evp1) / args.steps
        ctx.set_profiling(False)

        # ---- NEXT-1: the step with three corrector passes (nsc_step_iterated, tol = 0), device-resident
        # (its first call allocates 2 n_f + 2 more fields: skipped when the device has no room for them, cfg 5)
        it_k = it_err = ms_iter = controller = None
        if torch.cuda.mem_get_info()[0] > (2 * nf + 3) * F:
            evi0, evi1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.step_iterated(dt, 0.0, 3)
            torch.cuda.synchronize()
            evi0.record(stream)
            for _ in range(2):
                it_k, it_err = ctx.step_iterated(dt, 0.0, 3)
            evi1.record(stream)
            torch.cuda.synchronize()
            ms_iter = evi0.elapsed_time(evi1) / 2

            # ---- NEXT-1: the step-size controller (nsc_advance, R17) for a few attempts from the same state
            torch.cuda.synchronize()
            tc0 = time.perf_counter()
            adv_info, adv_log = ctx.advance(1e3 * dt, 4, dt, 1e-6, 0.5, 3)
            torch.cuda.synchronize()
            adv_ms = 1e3 * (time.perf_counter() - tc0)
            controller = {"what": "nsc_advance(t_end=1000 dt, max_steps=4, dt0=dt, tol=1e-6, cfl=0.5, max_corr=3)",
                          "attempts": [{"dt": a[0], "passes": a[1], "err": a[2], "accepted": a[3]} for a in adv_log],
                          "cfl_rate": adv_info["cfl_rate_last"], "ms_total": adv_ms}

        # ---- end to end through the C ABI with HOST buffers: H2D state, step, D2H state
        ke = max(1, min(args.steps, args.e2e_steps))
        ctx.set_state(*host_in)
        ctx.step(dt)
        ctx.get_state(*host_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            ctx.set_state(*host_in)           # nsc_set_state_host: pinned host -> device, synchronises
            ctx.step(dt)
            ctx.get_state(*host_out)          # nsc_get_state_host: device -> pinned host, synchronises
        torch.cuda.synchronize()
        e2e_sync_s = (time.perf_counter() - t0) / ke
        e2e_sync_s = replicas.max_over_ranks(e2e_sync_s, dist, "cuda")
        ref_out = host_out[1].copy()
        # the same loop with the double-buffered transfers: the host-to-device copy of step k + 1 and the device-to-host copy
        # of step k - 1 overlap the compute of step k (every step still carries both copies; the last ones are waited for)
        for a in host_out:
            if a is not None:
                a[...] = 0
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            ctx.set_state_host_async(*host_in)
            ctx.step(dt)
            ctx.get_state_host_async(*host_out)
        ctx.host_copies_wait()
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / ke
        e2e_s = replicas.max_over_ranks(e2e_s, dist, "cuda")
        if not np.array_equal(host_out[1], ref_out):
            raise SystemExit("bench.py: the double-buffered read-out returned another state than the synchronous one")
        finite = bool(np.isfinite(host_out[1]).all())
        dev_bytes = ctx.device_bytes()

    # ---- measured fp64 peaks of this device (register-only kernels, nsc_fp64_peak) and the other configurations
    fp64_fma = nsc.fp64_peak(0)
    fp64_addmul = nsc.fp64_peak(1)
    extra = []
    if rank == 0 and world == 1:
        for ci in args.extra_configs:
            try:
                extra.append(time_extra_config(ci, args, stream))
            except Exception as exc:                  # e.g. no room for cfg 5 on a smaller device: reported, not fatal
                extra.append({"workload": f"BASELINE.json configs[{ci - 1}]", "error": str(exc)[:200]})

    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    if not finite:
        raise SystemExit("bench.py: the state went non-finite during the run")

    # ---- roofline figures
    peak, peak_src = measured_peaks()
    model = algorithmic_bytes(cfg)
    kern = []
    lin_ms = 0.0
    for name, (kms, cnt) in prof.items():
        if cnt == 0 or name == "k_factor":
            continue
        per_step_ms = kms / args.steps
        if name in LINEAR_KERNELS:
            lin_ms += per_step_ms
        kern.append({"kernel": name, "launches_per_step": cnt / args.steps, "ms_per_step": per_step_ms,
                     "avg_launch_us": 1e3 * kms / cnt})
    tot_ms = sum(k["ms_per_step"] for k in kern) or 1.0
    for k in kern:
        k["share"] = k["ms_per_step"] / tot_ms
        if k["kernel"] in model:
            k["algorithmic_GB_per_step"] = model[k["kernel"]] / 1e9
            k["achieved_GBs"] = model[k["kernel"]] / 1e6 / k["ms_per_step"]
    kern.sort(key=lambda k: -k["ms_per_step"])
    dom = next((k for k in kern if "achieved_GBs" in k), None)
    # the linear stage as one unit
    lin = {"kernel": "linear stage (L1-L5, all kernels)", "ms_per_step": lin_ms,
           "algorithmic_GB_per_step": model["linear"] / 1e9,
           "achieved_GBs": model["linear"] / 1e6 / lin_ms if lin_ms else None, "share": lin_ms / tot_ms}
    if dom is None or (lin_ms > dom["ms_per_step"]):
        dom = lin
    launches_dom = dom.get("launches_per_step", None)
    traffic, traffic_src = ncu_traffic(dom["kernel"], args.config)
    for k in kern:
        k["bound"] = "alu" if k["kernel"] == "k_theta" else "hbm"
    th = next((k for k in kern if k["kernel"] == "k_theta"), None)
    hbm_view = {"achieved": dom["achieved_GBs"], "peak": peak, "unit": "GB/s", "frac": dom["achieved_GBs"] / peak,
                "peak_source": peak_src}
    if dom["kernel"] == "k_theta":
        # the dominant kernel (the fused theta transforms) is bound by the plain fp64 pipe, not by HBM: its model flops
        # (5 N log2 N per complex transform + the products) over its time against the fp64 peak MEASURED in this run
        flops = 2 * flops_theta_per_nonlinear(cfg)
        tf = flops / 1e9 / th["ms_per_step"]
        head = {"bound": "alu", "kernel": "k_theta", "achieved": tf, "peak": fp64_fma, "unit": "TFLOP/s",
                "frac": tf / fp64_fma,
                "peak_source": "measured: nsc_fp64_peak(kind 0): register-only DFMA kernel on every SM, 2 flop per instruction",
                "note": ("fp64 butterflies are mostly additions and multiplications that cannot fuse; against the measured "
                         "DADD+DMUL rate (1 flop per instruction) the same flops are frac_of_addmul_peak"),
                "addmul_peak": fp64_addmul, "frac_of_addmul_peak": tf / fp64_addmul,
                "nominal_dfma_peak": FP64_NOMINAL_TFLOPS,
                "hbm_view": hbm_view}
    else:
        head = dict(hbm_view, bound="hbm", kernel=dom["kernel"])
    roofline = dict(head)
    roofline.update({
        "traffic": traffic, "traffic_source": traffic_src,
        "share_of_step": dom["share"],
        "algorithmic_bytes_per_launch": (model.get(dom["kernel"], model["linear"]) / launches_dom
                                         if launches_dom else None),
        "avg_launch_us": dom.get("avg_launch_us"),
        "step": {"algorithmic_GB": model["step"] / 1e9, "achieved_GBs": model["step"] / 1e6 / ms_per_step,
                 "frac_of_measured": model["step"] / 1e6 / ms_per_step / peak,
                 "frac_of_nominal_8TBs": model["step"] / 1e6 / ms_per_step / NOMINAL_HBM_GBS},
        "fp64": {"GF_per_nonlinear": flops_per_nonlinear(cfg) / 1e9, "dfma_peak_TFLOPs": fp64_fma, "addmul_peak_TFLOPs": fp64_addmul},
        "kernels": kern + [lin],
        "ms_per_step_with_event_brackets": ms_prof_per_step,
    })
    value = replicas.aggregate_rate(world, args.steps, ms / 1e3)
    mode_points = s["N_r"] * (s["M"] + 1) * (2 * s["K"] + 1)
    nbytes_state = len(names) * F
    out = {
        "metric": METRIC, "value": value, "unit": "steps/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "N_r": s["N_r"], "M_theta": s["M"], "K_z": s["K"],
                   "physical_grid": [s["Nt"], s["Nz"]], "dt": dt, "parallelism": f"replicas x{world}",
                   "l2": f"no flush: the step streams {model['step'] / 1e9:.1f} GB of fields "
                         f"(one spectral field {F / 1e6:.0f} MB) against 126 MB of L2",
                   "device_bytes": dev_bytes},
        "mode_points_per_s": value * mode_points,
        "iterated_corrector": ({"what": "nsc_step_iterated(dt, tol=0, max_corr=3): SURVEY 8(f) NEXT-1, DESIGN.md R16",
                                "passes": it_k, "last_norm": it_err, "ms_per_step": ms_iter,
                                "ms_per_extra_pass": (ms_iter - ms_per_step) / 2} if ms_iter is not None else None),
        "step_size_controller": controller,
        "gpu_launches": launches,
        "clocks": clk,
        "e2e": {"value": replicas.aggregate_rate(world, 1, e2e_s), "unit": "steps/s", "h2d_bytes_per_step": nbytes_state,
                "d2h_bytes_per_step": nbytes_state, "steps": ke,
                "what": ("per step: nsc_set_state_host_async (pinned host -> staging set on a private stream -> state) + "
                         "nsc_step + nsc_get_state_host_async (snapshot -> pinned host on a second private stream): the "
                         "copies of neighbouring steps overlap the compute; nsc_host_copies_wait at the end, inside "
                         "the timed region; the result is checked against the synchronous loop"),
                "synchronous": {"value": replicas.aggregate_rate(world, 1, e2e_sync_s), "unit": "steps/s",
                                "what": "nsc_set_state_host + nsc_step + nsc_get_state_host per step, no overlap"}},
        "roofline": roofline,
        "other_configs": extra,
    }
    if not args.no_cpu_baseline and world == 1:
        t_step, desc, threads = oracle_sample(cfg)
        out["cpu_baseline"] = {"value": 1.0 / t_step, "unit": "steps/s", "cores": threads, "kind": "oracle",
                               "sample": desc}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config 1..5 (default 4: N_r=256, M=K=256)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--radial-chunk", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--linear-slices", type=int, default=0, help="nsc_params.linear_slices (0: the library's default, 2)")
    ap.add_argument("--extra-configs", type=lambda v: [int(x) for x in v.split(",") if x], default=[3, 5],
                    help="other BASELINE.json configs timed in the same run and reported under other_configs (default 3,5; "
                         "cfg 5 holds 148 GB on the device and adds about 90 s)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"bench.py: note: warmup {args.warmup} < 3 breaks the timing rules", file=sys.stderr)
    from paper_1908_00587_b200 import synth
    cfg = synth.config(args.config - 1)
    cfg["index"] = args.config - 1
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
