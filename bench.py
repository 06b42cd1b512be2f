#!/usr/bin/env python
"""bench.py -- throughput of the hot path of arXiv 1004.1932 on B200, beside the CPU oracle.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-sweep] [--quick]

One bench "step" = one Heun time step of BASELINE.json config 4: a 3d random
suspension of S = 2048 dumbbells (N = 4096 spheres), FP32 pair arithmetic, RPY tensor (the tensor
the paper simulates with): force (Eq. 4) -> mobility apply (Eq. 3a,3b) -> predictor ->
force -> mobility apply -> corrector, all on the device through ds_step (include/ds.h): one persistent
kernel launch runs the K steps of a ds_step(K) call.  Timing: at least 50 ms of warm-up steps, then R back-to-back
ds_step(K) launches (R such that the timed region exceeds 30 ms), each bracketed by CUDA events; ms_per_step is the
median launch / K (min and max are in `timed_region`).
Metric: ordered pair interactions per second, 2 N (N-1) per Heun step; timesteps/s is reported
beside it for this and every other config.  The path does not shard: --gpus N runs N independent
replicas, value = all replicas' pairs / the slowest replica's time.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the host
cores instead; it is the only other place, with `cpu_baseline`, where this file runs oracle code.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pair_interactions_per_s"
UNIT = "pairs/s"
# Algorithmic FLOP per ordered pair (FMA = 2, rsqrt not counted): SURVEY.md 8(d)'s per-unit figure, the contract's count
# (27 Oseen, 34 RPY).  The kernel's own pair body has 21 packed instructions for RPY, 12 of them FMA = 33 FLOP; the
# fraction with that smaller count is reported beside it (roofline.frac_kernel_count).  DESIGN.md "FLOP count".
FLOP_PER_PAIR = {"oseen": 27, "rpy": 34}
FLOP_PER_PAIR_KERNEL = {"oseen": 27, "rpy": 33}
# DRAM bytes (read + write) of one whole ds_step launch of the headline workload, from the ncu --set full capture of
# the same command (profiles/r2_pipe_kernel_ncu_full.md): the path is ALU-bound and L2-resident
NCU_DRAM_BYTES_PER_LAUNCH = {"f32": 301568, "f64": None}
# ALU peaks derived in DESIGN.md "Roofline": SMs x lanes x 2 x f_SM(max).  FP32: 128 lanes/SM.  FP64: the
# DFMA rate of B200 is what ds_peak_probe measures; the nominal figure used is 64 lanes/SM.
N_SM, F32_LANES, F64_LANES = 148, 128, 64


def pairs_per_apply(N, B=1):
    return B * N * (N - 1)


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock, power and throttle reasons of one GPU through NVML while a timed region runs."""

    def __init__(self, index, period=0.002):
        self.index, self.period = index, period
        self.sm, self.power, self.reasons = [], [], 0
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:  # CUDA ordinal -> NVML handle through the UUID (CUDA_VISIBLE_DEVICES may renumber)
                import torch
                self.h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(index).uuid))
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # no NVML: report that, never invent numbers
            self.nv, self.err = None, repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.sm.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                self.reasons |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        reasons = [n for bit, n in names.items() if self.reasons & bit and n != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(self.sm),
                "power_w_max": max(self.power) if self.power else None}


# ----------------------------------------------------------------------------------------- GPU legs
def _events(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


WARM_S = 0.06      # at least this much device time of warm-up steps, whatever --warmup says (a lease may start at a low clock)
TIMED_S = 0.03     # the timed region: back-to-back ds_step(K) launches until their device time exceeds this


def time_steps(torch, ds, w, precision, tensor, n_steps, warmup, ranks=None, sampler=None, pipeline=None):
    """Device time of n_steps Heun steps of workload w through ds_step/ds_batch_step, state resident in HBM.
    Warm-up: `warmup` steps, repeated until WARM_S of device time has passed.  Timed: R back-to-back launches of
    n_steps steps each (every launch bracketed by its own pair of CUDA events on the launching stream), R such that the
    region exceeds TIMED_S; the reported time is the MEDIAN launch.  Returns (seconds per launch, launches per call,
    info)."""
    npdt = np.float32 if precision == ds.F32 else np.float64
    stream = torch.cuda.current_stream()
    sc = w.scalars
    with ds.System(w.S, n_batch=w.B, precision=precision, tensor=tensor, integrator=ds.HEUN, a=sc["a"], eta=sc["eta"],
                   ell=sc["ell"], lam=sc["lam"], omega=sc["omega"], k0=sc["k0"], dt=sc["dt"],
                   device=torch.cuda.current_device(), stream=stream.cuda_stream) as s:
        if pipeline is not None:
            s.set_pipeline(pipeline)
        pos = torch.as_tensor(np.ascontiguousarray(w.pos, dtype=npdt), device="cuda")
        phase = torch.as_tensor(w.phase, device="cuda")
        s.set_state(pos, phase, 0.0)
        step = s.batch_step if w.B > 1 else s.step
        if sampler is not None:
            sampler.__enter__()
        # ---- warm-up ----
        wsteps = max(int(warmup), 3)
        e0, e1 = _events(torch)
        warm, wl = 0.0, 0
        while warm < WARM_S and wl < 10000:
            e0.record(stream)
            step(wsteps)
            e1.record(stream)
            torch.cuda.synchronize()
            warm += e0.elapsed_time(e1) * 1e-3
            wl += 1
        est = warm / wl * (n_steps / wsteps)
        reps = int(min(200, max(3, np.ceil(TIMED_S / max(est, 1e-9)))))
        if ranks is not None:
            reps = int(ranks.max(reps))
            ranks.barrier()
        torch.cuda.synchronize()
        l0 = s.launch_count()
        ev = [_events(torch) for _ in range(reps)]
        for a, b in ev:
            a.record(stream)
            step(int(n_steps))
            b.record(stream)
        torch.cuda.synchronize()
        launches = (s.launch_count() - l0) // reps      # kernels launched per timed ds_step call
        if sampler is not None:
            sampler.__exit__()
        if ranks is not None:
            ranks.barrier()
        out = torch.empty_like(pos)
        s.get_state(out)
        torch.cuda.synchronize()
        if not bool(torch.isfinite(out).all()):
            raise RuntimeError("non-finite state after the timed steps")
        t = np.array([a.elapsed_time(b) * 1e-3 for a, b in ev])
        info = {"repeats": reps, "warmup_launches": wl, "warmup_device_ms": warm * 1e3,
                "ms_per_step_min": 1e3 * t.min() / n_steps, "ms_per_step_max": 1e3 * t.max() / n_steps,
                "timed_region_ms": 1e3 * t.sum(), "pipelined_kernel": s.pipeline_active() == 1,
                "step_kernel": {0: "small" if w.S <= 16 else "one-pass", 1: "pipelined", 2: "cluster", 3: "cluster-latency"}[s.pipeline_active()]}
        return float(np.median(t)), int(launches), info


def time_steps_cold_l2(torch, ds, w, precision, tensor, n_steps):
    """Same step, one at a time, with L2 flushed (a 512 MiB write) before each: per-step device time."""
    npdt = np.float32 if precision == ds.F32 else np.float64
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    with ds.System(w.S, n_batch=w.B, precision=precision, tensor=tensor, device=torch.cuda.current_device(),
                   stream=stream.cuda_stream) as s:
        pos = torch.as_tensor(np.ascontiguousarray(w.pos, dtype=npdt), device="cuda")
        s.set_state(pos, torch.as_tensor(w.phase, device="cuda"), 0.0)
        s.batch_step(3)
        tot = 0.0
        for _ in range(n_steps):
            flush.fill_(1)
            e0, e1 = _events(torch)
            e0.record(stream)
            s.batch_step(1)
            e1.record(stream)
            torch.cuda.synchronize()
            tot += e0.elapsed_time(e1) * 1e-3
        return tot / n_steps


def time_e2e(torch, ds, w, precision, tensor, n_steps, warmup, ranks=None):
    """The same step through the C ABI with HOST buffers: every step copies the positions and phases
    from pinned host memory to the device (ds_set_state), advances one Heun step (ds_step) and reads
    the positions back to pinned host memory (ds_get_state).  Wall clock, synchronised on both sides."""
    tdt = torch.float32 if precision == ds.F32 else torch.float64
    npdt = np.float32 if precision == ds.F32 else np.float64
    stream = torch.cuda.current_stream()
    pos = torch.as_tensor(np.ascontiguousarray(w.pos, dtype=npdt)).pin_memory()
    phase = torch.as_tensor(w.phase).pin_memory()
    assert pos.dtype == tdt and not pos.is_cuda
    h2d = pos.numel() * pos.element_size() + phase.numel() * phase.element_size()
    d2h = pos.numel() * pos.element_size()
    with ds.System(w.S, n_batch=w.B, precision=precision, tensor=tensor, device=torch.cuda.current_device(),
                   stream=stream.cuda_stream) as s:
        def one(k):
            s.set_state(pos, phase, k * w.scalars["dt"])
            s.batch_step(1)
            s.get_state(pos)          # host pointer: synchronises the stream before returning
        for k in range(max(int(warmup), 3)):
            one(k)
        torch.cuda.synchronize()
        if ranks is not None:
            ranks.barrier()
        l0 = s.launch_count()
        t0 = time.perf_counter()
        for k in range(n_steps):
            one(k)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if ranks is not None:
            ranks.barrier()
        if not bool(torch.isfinite(pos).all()):
            raise RuntimeError("non-finite state in the e2e loop")
        return dt, h2d, d2h, s.launch_count() - l0


def time_apply(torch, ds, N, precision, tensor, X, F, reps):
    """Standalone ds_mobility_apply (a2 + a3 with arbitrary F), device buffers, `reps` back-to-back
    launches replayed from a CUDA graph so that host launch cost does not enter.  Seconds per apply."""
    npdt = np.float32 if precision == ds.F32 else np.float64
    side = torch.cuda.Stream()
    Xd = torch.as_tensor(np.ascontiguousarray(X, dtype=npdt), device="cuda")
    Fd = torch.as_tensor(np.ascontiguousarray(F, dtype=npdt), device="cuda")
    ud = torch.empty_like(Xd)
    with ds.System(1, precision=precision, tensor=tensor, device=torch.cuda.current_device(),
                   stream=side.cuda_stream) as s:
        s.mobility_apply(Xd, Fd, ud, N)     # allocates the scratch outside the capture
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            s.set_stream(torch.cuda.current_stream().cuda_stream)
            for _ in range(reps):
                s.mobility_apply(Xd, Fd, ud, N)
        s.set_stream(side.cuda_stream)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        best = float("inf")
        for _ in range(5):
            e0, e1 = _events(torch)
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) * 1e-3 / reps)
        if not bool(torch.isfinite(ud).all()):
            raise RuntimeError("non-finite apply output")
        del g
        return best


def peak_probe(ds, torch):
    """Measured FMA-chain peaks (TFLOP/s) of this GPU: FP32 (packed FFMA2), FP64 (DFMA)."""
    out = {}
    try:
        for name, prec in (("f32", ds.F32), ("f64", ds.F64)):
            out[name + "_tflops"] = ds.peak_probe(prec, torch.cuda.current_device()) * 1e-12
    except AttributeError:
        return None
    return out


# ----------------------------------------------------------------------------------------- CPU legs
def oracle_steps(w, tensor_name, n_steps, threads):
    """Times the oracle, as it stands, on n_steps Heun steps of w (first system).  Returns seconds."""
    import oracle
    oracle.set_threads(threads)
    sc = w.scalars
    p = oracle.Params(a=sc["a"], eta=sc["eta"], ell=sc["ell"], lam=sc["lam"], omega=sc["omega"], k0=sc["k0"],
                      dt=sc["dt"], tensor=oracle.RPY if tensor_name == "rpy" else oracle.OSEEN, integrator=oracle.HEUN)
    X0 = np.asarray(w.pos[0], dtype=np.float32).astype(np.float64)
    t0 = time.perf_counter()
    X = oracle.step(X0, w.phase[0], 0.0, 0, n_steps, p)
    dt = time.perf_counter() - t0
    assert np.isfinite(X).all()
    return dt


def run_reference(args, ranks):
    """--impl reference: the oracle on the host cores, same config/metric/unit; rank 0 only."""
    if ranks.rank != 0:
        return
    import oracle
    from paper_1004_1932_b200 import inputs
    w = inputs.config4()
    cores = oracle.max_threads()
    N = w.N
    for _ in range(min(args.warmup, 1)):
        oracle_steps(w, args.tensor, 1, cores)
    per = []
    for _ in range(args.steps):
        per.append(oracle_steps(w, args.tensor, 1, cores))
    tot = sum(per)
    value = args.steps * 2 * pairs_per_apply(N) / tot
    sample = f"{args.steps} x 1 Heun step of C4 (N={N}), fp64 oracle, OpenMP over alpha on {cores} threads"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, args, "f64"),
            "timesteps_per_s": args.steps / tot,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(w, args, dtype):
    return {"workload": f"BASELINE.json configs[3]: 3d random suspension S={w.S} dumbbells (N={w.N} spheres), "
                        f"density 1/(4 ell)^3, hard core 2.5a, seed {w.seed}; one step = one Heun time step "
                        f"(2 mobility applies + forces + predictor/corrector)",
            "N": w.N, "S": w.S, "B": w.B, "tensor": args.tensor, "precision": dtype, "integrator": "heun",
            "dt": w.scalars["dt"], "k0": w.scalars["k0"],
            "pairs_per_step": 2 * pairs_per_apply(w.N, w.B), "flop_per_pair": FLOP_PER_PAIR[args.tensor],
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU",
            "l2": "warm by construction: the 256 KB state is produced on the device by the previous step and "
                  "never leaves it (the method has no host round trip per step); the cold-L2 per-step figure "
                  "(512 MiB flush before every step) is in extra.cold_l2"}


AVG_FLOP_PER_PAIR = 93


def avg_model_extra(torch, ds, sizes=(729, 2048, 8192)):
    """The stroke-averaged far-field model (Eq. 9): one right-hand side (S^2 dumbbell pairs) and one
    Heun step at the paper's largest S = 729 and two larger sizes."""
    avg = {}
    for S_ in sizes:
        rng = np.random.default_rng(S_)
        Rr = torch.as_tensor(rng.uniform(-200, 200, (S_, 3)).astype(np.float32), device="cuda")
        Nr = rng.standard_normal((S_, 3)); Nr /= np.linalg.norm(Nr, axis=1, keepdims=True)
        Nr = torch.as_tensor(Nr.astype(np.float32), device="cuda")
        ph = torch.as_tensor(rng.uniform(0, 6.28, S_), device="cuda")
        dRr, dNr = torch.empty_like(Rr), torch.empty_like(Nr)
        with ds.System(1, precision=ds.F32, device=torch.cuda.current_device(),
                       stream=torch.cuda.current_stream().cuda_stream) as sa:
            for _ in range(3):
                sa.avg_rhs(Rr, Nr, ph, dRr, dNr, S_)
            torch.cuda.synchronize()
            e0, e1 = _events(torch)
            e0.record()
            for _ in range(50):
                sa.avg_rhs(Rr, Nr, ph, dRr, dNr, S_)
            e1.record()
            torch.cuda.synchronize()
            t = e0.elapsed_time(e1) * 1e-3 / 50
            nst = 400
            sa.avg_step(Rr, Nr, ph, S_, 0.5, 8)
            torch.cuda.synchronize()
            e0.record()
            sa.avg_step(Rr, Nr, ph, S_, 0.5, nst)
            e1.record()
            torch.cuda.synchronize()
            ts = e0.elapsed_time(e1) * 1e-3 / nst
        avg[f"S{S_}"] = {"us_per_rhs": t * 1e6, "dumbbell_pairs_per_s": S_ * (S_ - 1) / t,
                         "us_per_heun_step": ts * 1e6, "dumbbell_pairs_per_s_stepping": 2 * S_ * (S_ - 1) / ts,
                         # 93 FLOP per ordered dumbbell pair of Eq. (9c,d) as the kernel evaluates it (FMA = 2)
                         "flop_per_pair": AVG_FLOP_PER_PAIR,
                         "frac_of_alu_peak_stepping": 2 * S_ * (S_ - 1) * AVG_FLOP_PER_PAIR / ts / (N_SM * F32_LANES * 2 * 1.965e9),
                         "note": "ds_avg_rhs on device buffers (sin/cos table kernel + pair kernel per call: 32 dumbbells x 8 "
                                 "slices per CTA, clusters of <= 8 CTAs per block of dumbbells) and ds_avg_step (S <= 4096: one "
                                 "device-resident cooperative launch for all steps, tagged hand-over between stages; larger S: 2 "
                                 "launches per Heun step); FP64 state, FP32 pair arithmetic"}
    return avg


def cpu_apply_sweep(inputs):
    """the oracle's mobility apply (RPY, FP64) timed single-threaded and on all host cores at every sweep
    size up to N = 16384, and once at N = 65536 on all cores.  Pair-interactions/s, pairs = N (N - 1)."""
    import oracle
    cores = oracle.max_threads()
    out = {"cores": cores, "kind": "oracle", "tensor": "rpy", "unit": UNIT}
    for lg in range(8, 15):
        Xs, Fs = inputs.sweep_case(lg)
        n = 1 << lg
        row = {}
        for name, th in (("single_thread", 1), ("all_cores", cores)):
            oracle.set_threads(th)
            reps = max(1, min(20, int(2e8 * th / (n * n))))
            t0 = time.perf_counter()
            for _ in range(reps):
                oracle.mobility_apply(Xs, Fs, 1.0, 1.0, oracle.RPY)
            row[name] = pairs_per_apply(n) * reps / (time.perf_counter() - t0)
        out[f"N{n}"] = row
    Xs, Fs = inputs.sweep_case(16)
    oracle.set_threads(cores)
    t0 = time.perf_counter()
    oracle.mobility_apply(Xs, Fs, 1.0, 1.0, oracle.RPY)
    out["N65536"] = {"all_cores": pairs_per_apply(65536) / (time.perf_counter() - t0)}
    return out


def extras(torch, ds, inputs, w, args, precision, tensor):
    """Beside the headline: the standalone apply at N = 4096 (4 variants), timesteps/s of every config,
    the cold-L2 per-step figure, the N = 256 .. 65536 apply sweep (BASELINE.json configs[4]) and the oracle's apply
    timings at the sweep sizes; --no-sweep leaves the last two out."""
    extra = {}
    # apply at N = 4096, all four variants (the standalone sweep of config 4)
    Xa, Fa = inputs.apply_case(4096, 1004, 2004)
    ap = {}
    for pname, pr in (("f32", ds.F32), ("f64", ds.F64)):
        for tname, tn in (("oseen", ds.OSEEN), ("rpy", ds.RPY)):
            t = time_apply(torch, ds, 4096, pr, tn, Xa, Fa, reps=200)
            ln = F32_LANES if pname == "f32" else F64_LANES
            ap[f"{pname}_{tname}"] = {"us": t * 1e6, "pairs_per_s": pairs_per_apply(4096) / t,
                                      "frac_of_alu_peak": pairs_per_apply(4096) * FLOP_PER_PAIR[tname] / t /
                                      (N_SM * ln * 2 * 1.965e9)}
    extra["apply_N4096"] = ap
    # timesteps/s for every config
    cfgs = {}
    for name, mk, pr, nst in (("C1_N16_f64", inputs.config1, ds.F64, 10_000),
                              ("C2_N128_f32", inputs.config2, ds.F32, 10_000),
                              ("C2_N128_f64", inputs.config2, ds.F64, 10_000),
                              ("C3_N1024_f32", inputs.config3, ds.F32, 100_000),
                              ("C4_N4096_f32", inputs.config4, ds.F32, 1000),
                              ("C4_N4096_f64", inputs.config4, ds.F64, 1000),
                              ("C5_B64_N512_f32", inputs.config5, ds.F32, 10_000)):
        wc = w if mk is inputs.config4 else mk()
        t, _, info = time_steps(torch, ds, wc, pr, ds.RPY, nst, 64)
        lanes_c = F64_LANES if pr == ds.F64 else F32_LANES
        cfgs[name] = {"timesteps_per_s": nst / t, "pairs_per_s": nst * 2 * pairs_per_apply(wc.N, wc.B) / t,
                      "us_per_stage": 1e6 * t / (2 * nst), "steps_per_launch": nst, "repeats": info["repeats"],
                      "step_kernel": info["step_kernel"],
                      "frac_of_alu_peak": nst * 2 * pairs_per_apply(wc.N, wc.B) * FLOP_PER_PAIR["rpy"] / t / (N_SM * lanes_c * 2 * 1.965e9)}
    extra["configs_rpy_heun"] = cfgs
    extra["avg_model_eq9"] = avg_model_extra(torch, ds)
    extra["cold_l2"] = {"ms_per_step": 1e3 * time_steps_cold_l2(torch, ds, w, precision, tensor, 30),
                        "steps": 30, "flush": "512 MiB fill before every step"}
    if not args.no_sweep:
        # BASELINE.json configs[4]: scaling sweep of one mobility apply, N = 256 .. 65536, FP32, both tensors
        sw = {}
        for lg in range(8, 17):
            Xs, Fs = inputs.sweep_case(lg)
            n = 1 << lg
            for tname, tn in (("oseen", ds.OSEEN), ("rpy", ds.RPY)):
                reps = max(2, min(200, int(2e10 / (n * n))))
                t = time_apply(torch, ds, n, ds.F32, tn, Xs, Fs, reps=reps)
                sw[f"N{n}_{tname}"] = {"us": t * 1e6, "pairs_per_s": pairs_per_apply(n) / t,
                                       "frac_of_alu_peak": pairs_per_apply(n) * FLOP_PER_PAIR[tname] / t /
                                       (N_SM * F32_LANES * 2 * 1.965e9)}
        extra["sweep_f32"] = sw
        extra["cpu_apply"] = cpu_apply_sweep(inputs)
    return extra


# ----------------------------------------------------------------------------------------- main
def run_ours(args, ranks):
    import torch
    from paper_1004_1932_b200 import ds, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback "
                         "(use --impl reference for the CPU oracle)")
    torch.cuda.set_device(ranks.local_rank)
    ds.lib()  # fails loudly if libds.so cannot be built / loaded
    precision = ds.F32 if args.precision == "f32" else ds.F64
    tensor = ds.RPY if args.tensor == "rpy" else ds.OSEEN
    w = inputs.config4()
    N = w.N
    flop_pair = FLOP_PER_PAIR[args.tensor]

    # ---- the timed region: K Heun steps per launch, state resident in HBM; R launches, median (time_steps) ----
    sampler = ClockSampler(torch.cuda.current_device())
    sec, launches, tinfo = time_steps(torch, ds, w, precision, tensor, args.steps, max(args.warmup, 3), ranks, sampler)
    clocks = sampler.summary()
    sec_max = ranks.max(sec)
    pairs_step = 2 * pairs_per_apply(N)
    value = ranks.sum(args.steps * pairs_step) / sec_max

    # ---- e2e through host buffers ----
    e_sec, h2d, d2h, e_launches = time_e2e(torch, ds, w, precision, tensor, args.steps, args.warmup, ranks)
    e_value = ranks.sum(args.steps * pairs_step) / ranks.max(e_sec)

    def roofline_of(prec_name, sec_launch, info):
        """roofline object of one ds_step(K) launch: 2 K mobility stages of N (N - 1) ordered pairs each."""
        kernel_s = sec_launch / (2 * args.steps)
        lanes = F32_LANES if prec_name == "f32" else F64_LANES
        peak_nominal = N_SM * lanes * 2 * 1.965e9 * 1e-12
        achieved = pairs_per_apply(N) * flop_pair / kernel_s * 1e-12
        roof = {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                "frac": achieved / peak_nominal,
                "frac_kernel_count": achieved / peak_nominal * FLOP_PER_PAIR_KERNEL[args.tensor] / flop_pair,
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(prec_name),
                "traffic_note": "DRAM bytes (read + write) of one 50-step launch by ncu --set full "
                                "(profiles/r2_pipe_kernel_ncu_full.md); the algorithmic traffic of the ALU-bound path is the "
                                "L2-resident stream (24 B per sphere and stage in FP32) read by each CTA once per stage",
                "kernel": ("ds::pipe_kernel" if info["pipelined_kernel"] else "ds::run_kernel") +
                          "<float|double, tensor, Heun> (persistent: per stage pair sums + reduction + Eq. (3a) + Heun update + "
                          "Eq. (4) + stage hand-over; ONE launch for all K steps of a ds_step call)",
                "stage_us": kernel_s * 1e6, "stages_per_step": 2, "launch_us": sec_launch * 1e6,
                "flop_per_launch": args.steps * 2 * pairs_per_apply(N) * flop_pair,
                "peak_kind": f"derived: {N_SM} SMs x {lanes} {prec_name} FMA lanes x 2 x 1.965 GHz "
                             f"(MEASURED_PEAKS.json sm_max_mhz); MEASURED_PEAKS.json has no ALU entry",
                "flop_per_pair": flop_pair, "flop_per_pair_kernel": FLOP_PER_PAIR_KERNEL[args.tensor],
                "pairs_per_stage": pairs_per_apply(N), "timing": info}
        return roof

    line = None
    if ranks.rank == 0:
        roof = roofline_of(args.precision, sec, tinfo)
        if clocks.get("sm_mhz"):
            lanes = F32_LANES if args.precision == "f32" else F64_LANES
            roof["frac_at_sampled_clock"] = roof["achieved"] / (N_SM * lanes * 2 * clocks["sm_mhz"] * 1e6 * 1e-12)
        probe = peak_probe(ds, torch)
        if probe:
            roof["measured_fma_chain"] = probe
            roof["frac_of_measured_chain"] = roof["achieved"] / probe[args.precision + "_tflops"]
        # the paper's own arithmetic is FP64: the same workload and launch in the other precision
        other = "f64" if args.precision == "f32" else "f32"
        o_sec, _, o_info = time_steps(torch, ds, w, ds.F64 if other == "f64" else ds.F32, tensor, args.steps,
                                      max(args.warmup, 3))
        roof_other = roofline_of(other, o_sec, o_info)
        roof_other["timesteps_per_s"] = args.steps / o_sec
        if probe:
            roof_other["frac_of_measured_chain"] = roof_other["achieved"] / probe[other + "_tflops"]

        extra = None if args.quick else extras(torch, ds, inputs, w, args, precision, tensor)

        # ---- the oracle beside it (bounded sample) ----
        import oracle
        cores = oracle.max_threads()
        n_or = 1 if args.quick else args.cpu_steps
        oracle_steps(w, args.tensor, 1, cores)
        t_or = oracle_steps(w, args.tensor, n_or, cores)
        t_or1 = oracle_steps(w, args.tensor, 1, 1)
        cpu = {"value": n_or * pairs_step / t_or, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{n_or} Heun steps of the same C4 workload (N={N}), fp64, OpenMP over alpha",
               "timesteps_per_s": n_or / t_or,
               "single_thread": {"value": pairs_step / t_or1, "unit": UNIT, "cores": 1, "sample": "1 Heun step"}}

        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * sec_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
                "config": workload_config(w, args, args.precision),
                "timesteps_per_s": args.steps / sec_max,
                "clocks": clocks,
                "e2e": {"value": e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": 1e3 * e_sec / args.steps,
                        "path": "ds_set_state(host pos, host phase) + ds_step(1) + ds_get_state(host pos), pinned"},
                "gpu_launches": int(launches * tinfo["repeats"]),
                "timed_region": {"launches": tinfo["repeats"], "steps_per_launch": args.steps, "statistic": "median launch",
                                 "ms_per_step_min": tinfo["ms_per_step_min"], "ms_per_step_max": tinfo["ms_per_step_max"],
                                 "warmup_device_ms": tinfo["warmup_device_ms"]},
                "roofline": roof, "roofline_" + other: roof_other, "cpu_baseline": cpu, "extra": extra}
    ranks.barrier()
    if line is not None:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--precision", choices=["f32", "f64"], default="f32")
    ap.add_argument("--tensor", choices=["oseen", "rpy"], default="rpy")
    ap.add_argument("--cpu-steps", type=int, default=20, help="oracle Heun steps timed for cpu_baseline")
    ap.add_argument("--no-sweep", action="store_true", help="leave the N = 256 .. 65536 apply sweep and the oracle's apply timings out of extra")
    ap.add_argument("--quick", action="store_true", help="headline + e2e only (used under ncu)")
    ap.add_argument("--avg-model", action="store_true",
                    help="only the averaged-model timing of extra.avg_model_eq9 at S = 729 (used under ncu)")
    args = ap.parse_args()
    ref = args.impl == "reference"
    if args.steps is None:
        args.steps = 10 if ref else 4000
    if args.warmup is None:
        args.warmup = 1 if ref else 200
    from paper_1004_1932_b200.replicas import Ranks
    if ref:
        # rank 0 alone runs the oracle; the other ranks exit 0 without work (no process group needed)
        class _R:
            rank = int(os.environ.get("RANK", "0"))
        run_reference(args, _R())
        return
    if args.avg_model:
        import torch
        from paper_1004_1932_b200 import ds
        print(json.dumps({"avg_model_eq9": avg_model_extra(torch, ds, sizes=(729,))}), flush=True)
        return
    ranks = Ranks()
    if ranks.world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={ranks.world}: launch with torch.distributed.run "
                         f"--nproc-per-node {args.gpus}")
    try:
        run_ours(args, ranks)
    finally:
        ranks.close()


if __name__ == "__main__":
    main()
