#!/usr/bin/env python
"""bench.py — train samples/s (fwd+bwd+Adam) of nsm_train_step on B200, all five BASELINE.json configs in one run.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config C]

BASELINE.json's metric names no configuration and its north_star asks for "all five configs", so the default run
measures them all and prints ONE JSON line whose top level (`value`, `ms_per_step`, `e2e`, `roofline`, `cpu_baseline`,
`kernels`) is the LARGEST training configuration -- configs[3], the large-table stress, "config 4": 2^12 rays x 512
candidates, L=16 F=4 T=2^22 (719 MB of tables), bf16 MLPs -- timed over exactly K steps after W warm-up steps; the other
four configurations follow under `configs` with their own fixed step counts (config 3: 100 steps including the six
occupancy refreshes; config 5: forward-only render, rays/s).  `--config C` measures one configuration
alone as the headline.  A "step" is one pass of the whole hot path (S1-S13) over a fresh pre-generated synthetic ray batch
(DESIGN.md "Input recipe").

N > 1 runs N independent replicas (one field per GPU, no data-path collective), timed as the max
over ranks; value = all ranks' samples / that time.  --impl reference times the float64 CPU oracle (oracle/) on the
host cores instead, on the headline configuration.
"""
import argparse
import ctypes
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "train samples/sec (fwd+bwd+Adam) on 1 B200; % of HBM/L2 and tensor-pipe peak"
UNIT = "samples/s"
HEADLINE = 4
# (steps, warm-up) of the configurations that are not the headline; config 3's 100 steps are SURVEY.md 8(d)'s protocol
SUB_STEPS = {1: (300, 20), 2: (300, 20), 3: (100, 16), 4: (40, 5), 5: (4, 1)}   # config 5: its four views, one per step
N_BATCHES = {1: 1, 2: 16, 3: 100, 4: 8}
FP32_ALU_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12        # 148 SMs x 128 FMA lanes x 2 flop x max SM clock


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_tflops_sustained=d.get("bf16_tflops_sustained"),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """SM clock and throttle reasons sampled through NVML from a thread of this process while the timed region runs
    (a 25 ms region is over before `nvidia-smi -lms` prints its first line)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        self.sm, self.reasons, self.max_mhz, self.h, self.err = [], set(), None, None, None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:            # no NVML: the line says so instead of inventing clocks
            self.err = repr(e)
        self._stop = threading.Event()
        self.t = threading.Thread(target=self._run, daemon=True)

    def _sample(self):
        self.sm.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
        r = self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for bit, name in self.REASONS.items():
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception as e:
                self.err = repr(e)
                return
            time.sleep(0.0005)

    def start(self):
        if self.h is not None:
            self.t.start()
        return self

    def stop(self):
        if self.h is not None:
            self._stop.set()
            self.t.join(timeout=2)
        out = dict(sm_mhz=float(np.median(self.sm)) if self.sm else None, sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons),
                   samples=len(self.sm), how="NVML polled in-process during the timed region")
        if self.err:
            out["error"] = self.err
        return out


WORKLOADS = {
    1: "BASELINE.json configs[0] (config 1): tiny fp32 case, 256 rays x 32 samples, full occupancy, L=4 F=2 T=2^10, 16-wide MLPs",
    2: "BASELINE.json configs[1] (config 2): Instant-NGP-default field, 4096 rays x 128 candidates, 128^3 sphere-union occupancy, "
       "L=16 F=2 T=2^19, MLPs 32->64->16 / 31->64->64->3, fp16",
    3: "BASELINE.json configs[2] (config 3): keyframe-window mapping, 10 synthetic 1200x680 keyframes of the 8x6x3 m room, 2^14 rays x "
       "128 candidates per step, 100 steps, occupancy FULL then FROM_FIELD every 16 steps, field as config 2",
    4: "BASELINE.json configs[3] (config 4, the largest training configuration): large-table stress, 2^12 rays x 512 candidates, "
       "L=16 F=4 T=2^22 N_max=8192 (719 MB of tables), 256^3 occupancy at ~10 %, bf16 MLPs, 25-keyframe room",
    5: "BASELINE.json configs[4] (config 5): full-frame render of 4 held-out 1200x680 views, 256 candidates/ray, cut 1e-4, field trained "
       "500 steps on config 3's data",
}
L2_NOTE = {
    1: "flushed: a 256 MB buffer is rewritten between steps, each step timed by its own event pair (the whole working set is < 1 MB)",
    2: "not flushed: tables + Adam moments (16 B per parameter, 195 MB) exceed the 126 MB L2 and every step gets a fresh ray batch",
    3: "not flushed: tables + Adam moments (195 MB) plus ~0.3-1 M samples of workspace per step exceed the 126 MB L2",
    4: "not flushed: tables + Adam moments are 2.9 GB, far beyond the 126 MB L2; every step gets a fresh ray batch",
    5: "not flushed: 816 000 rays x 256 candidates of workspace per view exceed the 126 MB L2",
}


def make_workload(cfg):
    from workloads import configs
    if cfg == 1:
        return configs.config1()
    if cfg == 2:
        return configs.config2(n_batches=N_BATCHES[2])
    if cfg == 3:
        return configs.config3(n_batches=N_BATCHES[3])
    if cfg == 4:
        return configs.config4(n_batches=N_BATCHES[4])
    raise ValueError(cfg)


# ----------------------------------------------------------------------------- CPU oracle legs

def time_oracle(w, steps, warmup, budget_s, n_rays=None):
    """The oracle as it stands (-fopenmp build) on the host cores, whole steps of the workload (n_rays = None) or its first
    n_rays rays.  Stops early once budget_s has passed; reports the steps actually done."""
    from oracle import oracle as orc
    from workloads import configs
    fc = w.field
    nt, _ = orc.param_count(fc)
    O = orc.Oracle(fc, configs.init_params(fc.seed, nt, orc.mlp_shapes(fc)), omp=True)
    O.set_occupancy(w.bits)
    bs = w.batches
    if n_rays is not None:
        bs = [configs.RayBatch(b.origins[:n_rays], b.dirs[:n_rays], b.rgb[:n_rays], b.depth[:n_rays], b.depth_var[:n_rays],
                               b.t_min, b.t_max, b.n_candidates) for b in w.batches]
    for i in range(warmup):
        O.train_step(bs[i % len(bs)], w.lambda_d)
    t0 = time.perf_counter()
    total, done = 0, 0
    for i in range(steps):
        st, _ = O.train_step(bs[(warmup + i) % len(bs)], w.lambda_d)
        total += st["n_samples"]
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return dict(value=total / dt, seconds=dt, steps=done, samples=total, cores=O.num_threads(), rays=bs[0].n_rays)


def oracle_baseline(cfg, w, steps, budget_s):
    """cpu_baseline of one training configuration: whole steps for configs 1, 2, 4; config 3 one whole
    step of 2^14 rays at FULL occupancy (~1 M live samples: the first, most expensive step of its 100)."""
    r = time_oracle(w, steps, 0 if cfg in (3, 4) else 1, budget_s)
    return dict(value=r["value"], unit=UNIT, cores=r["cores"], kind="oracle",
                sample=f"{r['steps']} whole oracle step(s) of config {cfg} ({r['rays']} rays each, {r['samples']} live samples in "
                       f"{r['seconds']:.1f} s; float64, -fopenmp)")


def oracle_render_baseline(fc, theta, bits, view, stride=8):
    """Config 5: the oracle renders a 1/64 pixel-strided subset of one view; rays/s as measured."""
    from oracle import oracle as orc
    from workloads import configs
    O = orc.Oracle(fc, theta, omp=True)
    O.set_occupancy(bits)
    H, W = 680, 1200
    sel = (np.arange(H)[::stride, None] * W + np.arange(W)[None, ::stride]).reshape(-1)
    sub = configs.RayBatch(view.origins[sel], view.dirs[sel], None, None, None, view.t_min, view.t_max, view.n_candidates)
    t0 = time.perf_counter()
    _, _, _, n = O.render(sub, 1e-4)
    dt = time.perf_counter() - t0
    return dict(value=sub.n_rays / dt, unit="rays/s", cores=O.num_threads(), kind="oracle",
                sample=f"one view, every {stride}th pixel in x and y ({sub.n_rays} of 816000 rays, {n} samples evaluated in {dt:.1f} s; "
                       "rays/s as measured on the subset, not scaled)")


def run_reference(args):
    """The reference arm of this tier: the oracle on the headline configuration, whole steps, host cores."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    cfg = args.config or HEADLINE
    if cfg == 5:
        cfg = HEADLINE
    w = make_workload(cfg)
    r = time_oracle(w, args.steps, args.warmup, budget_s=150.0)
    sample = (f"{r['steps']} whole oracle steps of config {cfg} ({r['rays']} rays each, {r['samples']} live samples in {r['seconds']:.1f} s; "
              f"{args.steps} asked, stops past 150 s)")
    line = dict(impl="reference", metric=METRIC, value=r["value"], unit=UNIT, n_gpus=args.gpus, steps=r["steps"], warmup=args.warmup,
                ms_per_step=1e3 * r["seconds"] / max(r["steps"], 1), higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=workload_config(cfg, w, None),
                cpu_baseline=dict(value=r["value"], unit=UNIT, cores=r["cores"], kind="oracle", sample=sample),
                e2e=dict(value=r["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- the CUDA arm

def workload_config(cfg, w, f, extra=None):
    fc = w.field
    b0 = w.batches[0]
    c = dict(workload=WORKLOADS[cfg], config=cfg, rays_per_step=b0.n_rays, candidates_per_ray=b0.n_candidates,
             occupancy_fraction=round(w.extra["occupancy_fraction"], 4) if "occupancy_fraction" in w.extra else None,
             lambda_d=w.lambda_d, mlp_precision=["fp32", "fp16", "bf16"][fc.mlp_precision], l2=L2_NOTE[cfg],
             batches=f"{len(w.batches)} distinct pre-generated batches, cycled")
    if f is not None:
        c.update(table_params=f.n_table, mlp_params=f.n_mlp, mlp_path=f.nsm_mlp_path())
    if extra:
        c.update(extra)
    return c


def kernel_model(name, S, R, K, L, F, U, mac):
    """Algorithmic bytes / flops of ONE launch of a kernel class: SURVEY.md 8(d)'s per-unit figures x the units a launch
    processes: gather 8 L F 4 B per sample; scatter its read-modify-write, x 2; Adam 28 B per
    updated parameter = 28 F U; MLPs 2 MAC (forward) / 4 MAC (backward) flops per sample."""
    gather = 8 * L * F * 4 * S
    LF = L * F
    if name == "encode":
        return dict(bound="hbm", bytes=gather + 12 * S + 4 * LF * S)
    if name == "scatter":
        return dict(bound="hbm", bytes=2 * gather + 4 * LF * S + 12 * S)
    if name == "adam_table":
        return dict(bound="hbm", bytes=28 * F * U)
    if name == "mlp_fwd":
        return dict(bound="alu", flops=2 * mac * S)
    if name == "mlp_bwd":
        return dict(bound="alu", flops=4 * mac * S)
    if name == "composite":
        return dict(bound="hbm", bytes=S * (4 + 4 + 4 + 12) * 2 + S * (4 + 4 + 12) + R * 40)
    if name == "march":
        return dict(bound="alu", flops=40 * R * K)
    return dict(bound="hbm", bytes=0)


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, RECORDED from the committed
# `ncu --set full` capture of this command (bench.py cannot run ncu on itself; refreshed with every committed profile)
NCU_TRAFFIC = {(4, "adam_table"): 2.539e9}
NCU_TRAFFIC_SOURCE = ("recorded, not measured by this run: dram__bytes_read.sum + dram__bytes_write.sum of one adam_table_kernel<4> launch in the "
                      "`ncu --set full` capture of `python bench.py --config 4 --only-headline --steps 10 --warmup 3` (profiles/r2k_table_alignment_and_encoder.md)")


def probe_l2(dev_index):
    """Random 8-byte gathers/s and red.v2.f32/s over a 48 MB (L2-resident) table, measured now by the bench-only
    libnsm_bench_probe.so (not part of the product ABI): what `encode` / `scatter` are quoted against while the tables fit the L2."""
    path = os.path.join(ROOT, "paper_2210_13641_b200", "libnsm_bench_probe.so")
    try:
        lib = ctypes.CDLL(path)
        lib.nsm_bench_probe_l2.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        out = {}
        sec = ctypes.c_double()
        for _ in range(3):                                   # untimed: an idle GPU takes a few launches to reach its clocks
            lib.nsm_bench_probe_l2(48 << 20, 1 << 22, 0, ctypes.byref(sec))
        for name, red in (("gathers_per_s", 0), ("reductions_per_s", 1)):
            rc = lib.nsm_bench_probe_l2(48 << 20, 1 << 22, red, ctypes.byref(sec))
            if rc != 0:
                return dict(error=f"nsm_bench_probe_l2 rc={rc}")
            out[name] = (1 << 22) / sec.value
        out["how"] = "libnsm_bench_probe.so: 2^22 random 8-byte gathers / red.global.add.v2.f32 over a 48 MB table, best of 8 launches, this run"
        return out
    except OSError as e:
        return dict(error=repr(e))


def probe_mma():
    """Cycles per small tcgen05.mma (M = 128, K = 16) in a stream of 48 at N = 16 / 32 / 48 / 64, and the issue-to-completion
    latency of a single one, measured now by libnsm_bench_probe.so: the MLP kernels' bound (profiles/r2d)."""
    path = os.path.join(ROOT, "paper_2210_13641_b200", "libnsm_bench_probe.so")
    try:
        lib = ctypes.CDLL(path)
        lib.nsm_bench_probe_mma.argtypes = [ctypes.c_uint32, ctypes.c_uint32, ctypes.POINTER(ctypes.c_longlong)]
        cyc = ctypes.c_longlong()
        out = dict(cycles_per_mma={})
        for N in (16, 32, 48, 64):
            if lib.nsm_bench_probe_mma(N, 48, ctypes.byref(cyc)) != 0:
                return dict(error="nsm_bench_probe_mma failed")
            out["cycles_per_mma"][N] = cyc.value / 48.0
        if lib.nsm_bench_probe_mma(64, 1, ctypes.byref(cyc)) != 0:
            return dict(error="nsm_bench_probe_mma failed")
        out["single_mma_cycles"] = int(cyc.value)
        out["how"] = ("libnsm_bench_probe.so: one CTA, an elected lane issues 48 (1) tcgen05.mma.cta_group::1.kind::f16 M=128 K=16 and one "
                      "commit; SM cycles from the first issue to the mbarrier flip, best of 4, this run")
        return out
    except (OSError, AttributeError) as e:
        return dict(error=repr(e))


def mma_dispatch_floor(name, mma, fc, S, n_sms, sm_hz, two_term):
    """MMA instructions per 128-sample tile of the tcgen05 MLP kernels and the time their dispatch alone takes at the
    measured rate (one tensor core per SM, tiles spread over n_sms SMs)."""
    c = lambda N: mma["cycles_per_mma"][min((16, 32, 48, 64), key=lambda n: abs(n - N))]
    LF = fc.n_levels * fc.n_features
    two = fc.color_hidden_layers == 2
    if name == "mlp_fwd":
        t = 3 if two_term else 1
        groups = [(t * LF // 16, 64), (t * 4, 16), (t * 2, 64)] + ([(t * 4, 64)] if two else []) + [(t * 4, 16)]
    else:   # per layer: 8 wgrad k-steps over the 128 samples + the dgrad's K / 16
        groups = [(8, 16), (1, 64)] + ([(8, 64), (4, 64)] if two else []) + [(8, 32), (4, 32), (8, 16), (1, 64), (8, 64), (4, LF)]
    n = sum(g[0] for g in groups)
    cycles = sum(g[0] * c(g[1]) for g in groups)
    tiles = -(-int(S) // 128)
    floor_s = -(-tiles // n_sms) * cycles / sm_hz
    return dict(mmas_per_tile=n, dispatch_cycles_per_tile=cycles, tiles=tiles, floor_us=1e6 * floor_s)


def mlp_activation_bytes(name, fc, S):
    """HBM bytes one launch of a tcgen05 TRAINING MLP kernel has to move ("blobs"): the forward reads
    the two-term 16-bit encoder tile and writes the 16-bit activations the backward pass needs (hidden density layer,
    colour-MLP input padded to 32, one or two hidden colour layers) plus sigma and rgb; the backward reads those, the hi
    term of the encoder tile and dL/dsigma, dL/drgb, and writes dL/de in fp32 for the scatter."""
    LF = fc.n_levels * fc.n_features
    saved = 2 * (fc.density_hidden + 32 + fc.color_hidden * (2 if fc.color_hidden_layers == 2 else 1))
    if name == "mlp_fwd":
        return S * (4 * LF + saved + 16 + 4)
    return S * (2 * LF + saved + 16 + 4 + 4 * LF)


class Timer:
    def __init__(self, torch, dev, replicas):
        self.torch, self.dev, self.replicas = torch, dev, replicas
        self.stream = torch.cuda.current_stream(dev)
        self.flush_buf = None

    def timed(self, n_steps, step_fn, first, flush=False):
        """Seconds on the device for exactly n_steps steps, bracketed by a barrier + synchronize on both sides.  flush: the
        L2 is overwritten between steps and every step has its own event pair (tiny working sets only)."""
        torch = self.torch
        self.replicas.barrier()
        torch.cuda.synchronize(self.dev)
        if not flush:
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(self.stream)
            for i in range(n_steps):
                step_fn(first + i)
            ev1.record(self.stream)
            torch.cuda.synchronize(self.dev)
            t = ev0.elapsed_time(ev1) * 1e-3
        else:
            if self.flush_buf is None:
                self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)
            evs = []
            for i in range(n_steps):
                self.flush_buf.fill_(i & 0xff)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(self.stream)
                step_fn(first + i)
                b.record(self.stream)
                evs.append((a, b))
            torch.cuda.synchronize(self.dev)
            t = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
        self.replicas.barrier()
        return t


def measure_training(cfg, K, W, env, want_sampled=False, want_pose=False):
    """One training configuration: device-resident leg, end-to-end leg through the host entry point, per-kernel pass,
    roofline of its dominant kernel, oracle baseline.  Returns the dict of one `configs[]` entry."""
    torch, nsm, replicas, dev, rank, world, peaks, l2 = (env[k] for k in ("torch", "nsm", "replicas", "dev", "rank", "world", "peaks", "l2"))
    from workloads import configs
    t_gen = time.perf_counter()
    w = make_workload(cfg)
    t_gen = time.perf_counter() - t_gen
    fc = w.field
    f = nsm.Field(fc, dev)
    f.nsm_set_params(configs.init_params(fc.seed + rank, f.n_table, f.mlp_shapes()))
    if w.bits is not None:
        f.nsm_update_occupancy(nsm.NSM_OCC_SET, w.bits)
    # the batches are generated and uploaded before the timed region and never modified: declared ready, so the marcher of
    # step i+1 may run beside the table update of step i (include/nsm.h)
    flush = cfg == 1                          # per-step event pairs with an L2 flush in between: keep each step self-contained
    f.nsm_set_option(nsm.NSM_OPT_BATCH_READY, 0 if flush else 1)
    refresh = 16 if cfg == 3 else 0          # config 3: occupancy FROM_FIELD every 16 steps, inside the timed region
    dbatches = [nsm.DeviceBatch(b, dev) for b in w.batches]
    hbatches = [nsm.HostBatch(b) for b in w.batches]
    lam = w.lambda_d
    timer = Timer(torch, dev, replicas)

    def reset_field():                        # config 3 is a 100-step protocol from theta_0 and FULL occupancy
        f.nsm_set_params(configs.init_params(fc.seed + rank, f.n_table, f.mlp_shapes()), np.zeros(f.n_table + f.n_mlp, np.float32),
                         np.zeros(f.n_table + f.n_mlp, np.float32), 0)
        f.nsm_update_occupancy(nsm.NSM_OCC_FULL)

    def dev_step(i):
        if refresh and i > 0 and i % refresh == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step(dbatches[i % len(dbatches)], lam, want_stats=False)

    def e2e_step(i):
        if refresh and i > 0 and i % refresh == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step_host(hbatches[i % len(hbatches)], lam, want_stats=True)

    # ---- device-resident leg.  Config 3 times steps 0..K-1 of the protocol itself (its first 16 steps, at FULL
    # occupancy, are the expensive ones), after a warm-up run that is then rolled back; the others W warm-up steps.
    first = 0 if cfg == 3 else W
    for i in range(W):
        dev_step(i)
    if cfg == 3:
        reset_field()
    s0, l0 = f.nsm_total_samples(), f.nsm_launch_count()
    sampler = ClockSampler(dev.index).start() if rank == 0 else None
    t_dev = timer.timed(K, dev_step, first, flush)
    clocks = sampler.stop() if sampler else None
    samples_dev = f.nsm_total_samples() - s0
    launches = f.nsm_launch_count() - l0
    value, total_samples, t_max = replicas.aggregate_throughput(samples_dev, t_dev)

    # ---- end-to-end leg: HOST buffers through the C-ABI, H2D of the batch and D2H of the statistics every step
    if cfg == 3:
        reset_field()
    for i in range(min(W, 3)):
        e2e_step(i)
    if cfg == 3:
        reset_field()
    s1 = f.nsm_total_samples()
    t_e2e = timer.timed(K, e2e_step, first, flush)
    e2e_value, _, t_e2e_max = replicas.aggregate_throughput(f.nsm_total_samples() - s1, t_e2e)
    e2e = dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=hbatches[0].bytes_in(), d2h_bytes_per_step=2 * 8 + 4,
               ms_per_step=1e3 * t_e2e_max / K, api="nsm_train_step_host, pinned host batches, statistics read back every step")

    out = None
    sampled = None
    if want_sampled and cfg == 3:
        # row f1: the same steps with the batches drawn on the device from the keyframe store
        kfs = w.extra["keyframes"]
        for i in range(kfs.n):
            f.nsm_add_keyframe(kfs.store_frame(i))
        b0_ = w.batches[0]

        def sampled_step(i):
            if refresh and i > 0 and i % refresh == 0:
                f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
            f.nsm_train_step_sampled(b0_.n_rays, b0_.t_min, b0_.t_max, b0_.n_candidates, lam, want_stats=False)
        reset_field()
        for i in range(W):
            sampled_step(i)
        reset_field()
        s3 = f.nsm_total_samples()
        t_s = timer.timed(K, sampled_step, 0)
        v_s, _, _ = replicas.aggregate_throughput(f.nsm_total_samples() - s3, t_s)
        sampled = dict(value=v_s, unit=UNIT, ms_per_step=1e3 * t_s / K, keyframes=kfs.n, store_bytes=kfs.n * kfs.W * kfs.H * 5 * 4,
                       api="nsm_train_step_sampled")
        if want_pose:   # row f2: the same leg with the pose gradients computed and the keyframe poses stepped every step
            f.nsm_set_option(nsm.NSM_OPT_POSE_GRADIENTS, 1)

            def pose_step(i):
                sampled_step(i)
                f.nsm_apply_pose_step(0.0, 0.0)          # zero learning rates: the full update path, poses unchanged
            reset_field()
            for i in range(W):
                pose_step(i)
            reset_field()
            s4 = f.nsm_total_samples()
            t_p = timer.timed(K, pose_step, 0)
            v_p, _, _ = replicas.aggregate_throughput(f.nsm_total_samples() - s4, t_p)
            sampled["with_pose_gradients"] = dict(value=v_p, unit=UNIT, ms_per_step=1e3 * t_p / K,
                                                  api="nsm_train_step_sampled + nsm_apply_pose_step, NSM_OPT_POSE_GRADIENTS")
            f.nsm_set_option(nsm.NSM_OPT_POSE_GRADIENTS, 0)

    if rank == 0:
        # ---- per-kernel pass: CUDA events around every launch, one launch at a time on the field's stream (no PDL overlap, no
        # side stream), so `share` is a share of this SERIALISED pass, whose sum exceeds the pipelined step above
        if cfg == 3:
            reset_field()
        f.nsm_profile(True)
        s2 = f.nsm_total_samples()
        KP = min(K, 100)
        for i in range(KP):
            dev_step(first + i)
        torch.cuda.synchronize(dev)
        prof = f.nsm_profile_read()
        f.nsm_profile(False)
        refresh_info = None
        if refresh:
            # the refreshes inside that pass launched encode / mlp_fwd over the 128^3 cell centres: time the same number of
            # refreshes alone and take them out of the per-kernel table, so that it describes the training step
            n_ref = (KP - 1) // refresh
            f.nsm_profile(True)
            for _ in range(n_ref):
                f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
            torch.cuda.synchronize(dev)
            prof_r = f.nsm_profile_read()
            f.nsm_profile(False)
            prof = {k: (max(ms - prof_r.get(k, (0.0, 0))[0], 0.0), n - prof_r.get(k, (0.0, 0))[1]) for k, (ms, n) in prof.items()}
            refresh_info = dict(refreshes_in_timed_region=(K - 1) // refresh,
                                us_per_refresh=1e3 * sum(ms for ms, n in prof_r.values()) / max(n_ref, 1),
                                kernels={k: dict(us=1e3 * ms / n_ref, launches=n / n_ref) for k, (ms, n) in prof_r.items() if n},
                                note="nsm_update_occupancy(FROM_FIELD) every 16 steps INSIDE the timed region (value and ms_per_step include "
                                     "it); timed here separately, serialised, and removed from kernels[]")
        S_avg = (f.nsm_total_samples() - s2) / KP
        # touched-entry count U of a representative step (the step after the passes above)
        f.nsm_backward(dbatches[0], lam, want_stats=False)
        U = int(f.nsm_debug_last_step("touched").astype(bool).sum())
        f.nsm_apply_adam()
        b0 = w.batches[0]
        L, F = fc.n_levels, fc.n_features
        mac = f.n_mlp
        total_ms = sum(ms for ms, n in prof.values())
        kernels = []
        for name, (ms, n) in prof.items():
            if n == 0:
                continue
            model = kernel_model(name, S_avg, b0.n_rays, b0.n_candidates, L, F, U, mac)
            avg_s = ms * 1e-3 / n
            k = dict(kernel=name, launches_per_step=n / KP, avg_us=1e6 * avg_s, share_of_serialised_pass=ms / total_ms, bound=model["bound"])
            if "bytes" in model:
                k.update(achieved=model["bytes"] / avg_s / 1e9 if avg_s > 0 else 0.0, unit="GB/s", peak=peaks["hbm_gbs"],
                         algorithmic_bytes=model["bytes"])
            else:
                if name.startswith("mlp") and f.nsm_mlp_path().startswith("tcgen05"):
                    k["bound"] = "tensor"
                    peak = peaks["bf16_tflops"]          # fp16 and bf16 share the dense tensor rate (guide: ratio 1)
                else:
                    peak = FP32_ALU_TFLOPS
                k.update(achieved=model["flops"] / avg_s / 1e12 if avg_s > 0 else 0.0, unit="TFLOP/s", peak=peak,
                         algorithmic_flops=model["flops"])
            k["frac"] = k["achieved"] / k["peak"]
            if name in ("mlp_fwd", "mlp_bwd") and k["bound"] == "tensor" and "error" not in env["mma"] and avg_s > 0:
                # what bounds these kernels: the dispatch rate of their small MMAs (measured in this run), not tensor math
                d = mma_dispatch_floor(name, env["mma"], fc, S_avg, torch.cuda.get_device_properties(dev).multi_processor_count,
                                       1e6 * ((clocks or {}).get("sm_mhz") or 1965.0), two_term=True)
                d["frac_of_floor"] = d["floor_us"] / (1e6 * avg_s)
                k["mma_dispatch"] = d
                # ... and the activations that cross HBM between the forward and the backward kernel
                nb = mlp_activation_bytes(name, fc, S_avg)
                k["hbm"] = dict(algorithmic_bytes=nb, achieved=nb / avg_s / 1e9, unit="GB/s", peak=peaks["hbm_gbs"],
                                frac=nb / avg_s / 1e9 / peaks["hbm_gbs"],
                                note="operand-tile images read and written by this launch (encoder tile, saved activations, "
                                     "dL/de): the second bound of this kernel beside MMA dispatch")
            if name in ("encode", "scatter") and avg_s > 0 and "error" not in l2:
                # what bounds S4 / S12 while the tables fit the L2: its random-access rate (8 corners per sample and level)
                acc = 8 * L * S_avg / avg_s
                pk = l2["gathers_per_s"] if name == "encode" else l2["reductions_per_s"]
                k["l2_random"] = dict(achieved_accesses_per_s=acc, peak_accesses_per_s=pk, frac=acc / pk,
                                      note="corner REFERENCES per second (8 per sample and level) against the probe's rate of physical "
                                           "L2 accesses: x-neighbour pairs share one access and runs of samples in one coarse cell are "
                                           "merged, so the ratio can exceed 1")
            kernels.append(k)
        kernels.sort(key=lambda k: -k["share_of_serialised_pass"])
        top = kernels[0]
        roofline = dict(kernel=top["kernel"], bound=top["bound"], achieved=top["achieved"], peak=top["peak"], unit=top["unit"],
                        frac=top["frac"], traffic=NCU_TRAFFIC.get((cfg, top["kernel"])),
                        traffic_source=NCU_TRAFFIC_SOURCE if (cfg, top["kernel"]) in NCU_TRAFFIC else None,
                        avg_us=top["avg_us"], share_of_serialised_pass=top["share_of_serialised_pass"],
                        algorithmic=(f"{top.get('algorithmic_bytes', top.get('algorithmic_flops')):.6g} "
                                     f"{'B' if 'algorithmic_bytes' in top else 'flop'} per launch: SURVEY.md 8(d) figure x units "
                                     f"(S = {S_avg:.0f} live samples, U = {U} touched entries, F = {F})"),
                        peak_source=peaks["source"] if top["bound"] != "alu" else "derived: 148 SM x 128 FMA/clk x 2 x 1.965 GHz",
                        samples_per_launch=S_avg, touched_entries=U)
        # ---- CPU baseline: the oracle as it stands on the host cores, whole steps, bounded
        n_or, budget = {1: (20, 3.0), 2: (10, 8.0), 3: (1, 40.0), 4: (2, 12.0)}[cfg]
        cpu_baseline = oracle_baseline(cfg, w, n_or, budget)
        out = dict(config=workload_config(cfg, w, f, dict(parallelism=f"{world} independent replica(s)", generate_s=round(t_gen, 1))),
                   metric=METRIC, value=value, unit=UNIT, steps=K, warmup=W, ms_per_step=1e3 * t_max / K,
                   samples_per_step=total_samples / K / world, touched_entries=U, rays_per_s=world * K * b0.n_rays / t_max,
                   candidates_per_s=world * K * b0.n_rays * b0.n_candidates / t_max,
                   dtype="f32" if f.nsm_mlp_path() == "simt_fp32" else ("f16" if fc.mlp_precision == 1 else "bf16"),
                   clocks=clocks, e2e=e2e, gpu_launches=launches, roofline=roofline, kernels=kernels, cpu_baseline=cpu_baseline)
        if refresh_info:
            out["occupancy_refresh"] = refresh_info
        if sampled is not None:
            out["sampled"] = sampled
    f.close()
    replicas.barrier()
    return out, w, fc


def measure_render(K, W, env):
    """Config 5: forward-only full-frame render (rays/s) of a field trained 500 steps on config 3's data."""
    torch, nsm, replicas, dev, rank, world, peaks, l2 = (env[k] for k in ("torch", "nsm", "replicas", "dev", "rank", "world", "peaks", "l2"))
    from dataclasses import replace
    from workloads import configs
    w = make_workload(3)
    fc = replace(w.field, max_candidates=256, max_rays=1 << 16)
    f = nsm.Field(fc, dev)
    f.nsm_set_params(configs.init_params(fc.seed, f.n_table, f.mlp_shapes()))
    train_steps = 500
    db = [nsm.DeviceBatch(b, dev) for b in w.batches]
    for i in range(train_steps):
        if i > 0 and i % 16 == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step(db[i % len(db)], w.lambda_d, want_stats=False)
    f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD)
    bits = f.nsm_get_occupancy()
    occ = float(np.unpackbits(bits).mean())
    hv = configs.config5_views()
    views = [nsm.DeviceBatch(v, dev) for v in hv]
    hviews = [nsm.HostBatch(v) for v in hv]
    timer = Timer(torch, dev, replicas)
    n_rays = views[0].n_rays
    step = lambda i: f.nsm_render(views[i % 4], 1e-4)
    for i in range(max(W, 1)):
        step(i)
    l0 = f.nsm_launch_count()
    sampler = ClockSampler(dev.index).start() if rank == 0 else None
    t = timer.timed(K, step, 0)
    clocks = sampler.stop() if sampler else None
    launches = f.nsm_launch_count() - l0
    rays_s, _, t_max = replicas.aggregate_throughput(K * n_rays, t)
    outs = (torch.empty((n_rays, 3), dtype=torch.float32).pin_memory(), torch.empty(n_rays, dtype=torch.float32).pin_memory(),
            torch.empty(n_rays, dtype=torch.float32).pin_memory())
    e2e_step = lambda i: f.nsm_render_host(hviews[i % 4], 1e-4, outs)
    e2e_step(0)
    t_e2e = timer.timed(K, e2e_step, 0)
    e2e_v, _, t_e2e_max = replicas.aggregate_throughput(K * n_rays, t_e2e)
    out = None
    if rank == 0:
        f.nsm_profile(True)
        for i in range(min(K, 2)):
            step(i)
        torch.cuda.synchronize(dev)
        prof = f.nsm_profile_read()
        f.nsm_profile(False)
        total_ms = sum(ms for ms, n in prof.values())
        n_prof_views = min(K, 2)
        # live samples of one view (S is a device-side count per ray chunk): view 0 rendered chunk by chunk, counts read back
        M = fc.max_rays
        S_view = 0
        for a in range(0, n_rays, M):
            part = configs.RayBatch(hv[0].origins[a:a + M], hv[0].dirs[a:a + M], None, None, None, hv[0].t_min, hv[0].t_max, hv[0].n_candidates)
            f.nsm_render(nsm.DeviceBatch(part, dev), 1e-4)
            S_view += int(f.nsm_debug_last_step("counts").sum())
        L, F, mac = fc.n_levels, fc.n_features, f.n_mlp
        kernels = []
        for kname, (ms, n) in prof.items():
            if n == 0:
                continue
            per_view_s = ms * 1e-3 / n_prof_views
            k = dict(kernel=kname, total_ms=ms, launches=n, us_per_view=1e6 * per_view_s, share_of_serialised_pass=ms / total_ms)
            if kname == "encode":
                nbytes = 8 * L * F * 4 * S_view + 12 * S_view + 4 * L * F * S_view
                k.update(bound="hbm", algorithmic_bytes=nbytes, achieved=nbytes / per_view_s / 1e9, unit="GB/s", peak=peaks["hbm_gbs"])
                k["frac"] = k["achieved"] / k["peak"]
                if "error" not in l2:
                    acc = 8 * L * S_view / per_view_s
                    k["l2_random"] = dict(achieved_accesses_per_s=acc, peak_accesses_per_s=l2["gathers_per_s"], frac=acc / l2["gathers_per_s"],
                                          note="corner references per second against the probe's rate of physical L2 accesses (pairs and "
                                               "runs of equal coarse cells are merged: the ratio can exceed 1)")
            elif kname == "mlp_fwd":
                flops = 2 * mac * S_view
                k.update(bound="tensor", algorithmic_flops=flops, achieved=flops / per_view_s / 1e12, unit="TFLOP/s", peak=peaks["bf16_tflops"])
                k["frac"] = k["achieved"] / k["peak"]
                if "error" not in env["mma"]:
                    # 13 launches per view, each spreading its own tiles over the SMs: the floor is summed per launch
                    d = mma_dispatch_floor("mlp_fwd", env["mma"], fc, S_view / max(n / n_prof_views, 1),
                                           torch.cuda.get_device_properties(dev).multi_processor_count,
                                           1e6 * ((clocks or {}).get("sm_mhz") or 1965.0), two_term=False)
                    d["floor_us"] *= n / n_prof_views
                    d["frac_of_floor"] = d["floor_us"] / (1e6 * per_view_s)
                    k["mma_dispatch"] = d
            kernels.append(k)
        kernels.sort(key=lambda k: -k["share_of_serialised_pass"])
        top = kernels[0]
        roofline = None
        if "achieved" in top:
            roofline = dict(kernel=top["kernel"], bound=top["bound"], achieved=top["achieved"], peak=top["peak"], unit=top["unit"],
                            frac=top["frac"], traffic=None, us_per_view=top["us_per_view"],
                            share_of_serialised_pass=top["share_of_serialised_pass"], samples_per_view=S_view,
                            algorithmic=f"SURVEY.md 8(d) gather bytes x S = {S_view} live samples of one view (all evaluated: the "
                                        "transmittance cut is applied in the compositor)", peak_source=peaks["source"])
        theta = f.nsm_get_params()[0]
        cpu = oracle_render_baseline(fc, theta, bits, hv[0])
        out = dict(config=dict(workload=WORKLOADS[5], config=5, rays_per_view=n_rays, candidates_per_ray=256, train_steps=train_steps,
                               occupancy_fraction_after_training=occ, mlp_path=f.nsm_mlp_path(), l2=L2_NOTE[5]),
                   metric="render rays/sec (forward only) on 1 B200", value=rays_s, unit="rays/s", steps=K, warmup=max(W, 1),
                   ms_per_step=1e3 * t_max / K, dtype="f16", clocks=clocks,
                   e2e=dict(value=e2e_v, unit="rays/s", h2d_bytes_per_step=hviews[0].bytes_in(), d2h_bytes_per_step=n_rays * 20,
                            ms_per_step=1e3 * t_e2e_max / K, api="nsm_render_host, pinned host rays in, pinned host image out"),
                   gpu_launches=launches, samples_per_view=S_view, samples_per_s=rays_s * S_view / n_rays, roofline=roofline,
                   kernels=kernels, cpu_baseline=cpu)
    f.close()
    replicas.barrier()
    return out


def run_cuda(args):
    import torch
    import paper_2210_13641_b200 as nsm
    from paper_2210_13641_b200 import build as nsm_build, replicas

    rank, local_rank, world = replicas.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback (use --impl reference for the oracle)")
    nsm_build.build()
    dev = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(dev)
    env = dict(torch=torch, nsm=nsm, replicas=replicas, dev=dev, rank=rank, world=world, peaks=measured_peaks(),
               l2=probe_l2(dev.index) if rank == 0 else dict(error="rank != 0"),
               mma=probe_mma() if rank == 0 else dict(error="rank != 0"))
    t_all = time.perf_counter()
    head_cfg = args.config or HEADLINE
    K, W = args.steps, max(args.warmup, 3)
    if head_cfg == 5:
        head = measure_render(K, max(args.warmup, 1), env)
    else:
        head, _, _ = measure_training(head_cfg, K, W, env, want_sampled=args.sampled, want_pose=args.pose)
    subs = []
    if args.config is None and not args.only_headline:
        for c in (1, 2, 3, 5):
            ks, ws_ = SUB_STEPS[c]
            if c == 5:
                subs.append(measure_render(ks, ws_, env))
            else:
                r, _, _ = measure_training(c, ks, ws_, env, want_sampled=args.sampled, want_pose=args.pose)
                subs.append(r)
    if rank == 0:
        line = dict(metric=head["metric"], value=head["value"], unit=head["unit"], n_gpus=world, steps=head["steps"], warmup=head["warmup"],
                    ms_per_step=head["ms_per_step"], higher_is_better=True, scaling="weak", vs_baseline=None, dtype=head["dtype"],
                    data="synthetic", config=head["config"])
        for k in ("samples_per_step", "touched_entries", "rays_per_s", "candidates_per_s", "samples_per_view", "samples_per_s", "clocks", "e2e",
                  "gpu_launches", "roofline",
                  "kernels", "cpu_baseline", "occupancy_refresh", "sampled"):
            if k in head:
                line[k] = head[k]
        line["l2_probe"] = env["l2"]
        line["mma_probe"] = env["mma"]
        line["peaks"] = env["peaks"]
        if subs:
            line["configs"] = subs
            line["gpu_launches_all_configs"] = head["gpu_launches"] + sum(s["gpu_launches"] for s in subs)
        line["bench_wall_s"] = round(time.perf_counter() - t_all, 1)
        print(json.dumps(line))
    replicas.shutdown()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps of the headline configuration (default 40; config 3: 100; config 5: 4, one view each)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default 5; at least 3 are always run)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=None, choices=[1, 2, 3, 4, 5],
                    help="measure this BASELINE.json configuration alone (default: config 4 as the headline and configs 1, 2, 3, 5 under `configs`)")
    ap.add_argument("--only-headline", action="store_true", help="skip the `configs` array")
    ap.add_argument("--sampled", action="store_true", help="config 3: add the leg that draws the batches on the device from the keyframe "
                    "store (row f1; casts ten full 1200x680 keyframes on the host first, ~30 s)")
    ap.add_argument("--pose", action="store_true", help="with --sampled: add a leg with pose gradients and pose steps (row f2)")
    args = ap.parse_args()
    head = args.config or HEADLINE
    if args.steps is None:
        args.steps = 5 if args.impl == "reference" else SUB_STEPS[head][0]
    if args.warmup is None:
        args.warmup = 0 if args.impl == "reference" else SUB_STEPS[head][1]
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
