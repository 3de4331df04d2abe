#!/usr/bin/env python
"""bench.py — train samples/s (fwd+bwd+Adam) of nsm_train_step on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload: BASELINE.json configs[1] (the configuration the metric is quoted on): 4096 rays x 128
candidates through a 128^3 sphere-union occupancy bitfield at ~15 %, L=16 F=2 T=2^19 hash grid,
64-wide MLPs; a fresh pre-generated synthetic ray batch every step.
A "step" is one pass of the whole hot path (S1-S13).  One JSON line is printed by rank 0.

N > 1 runs N independent replicas (one field per GPU, no data-path collective; DESIGN.md
"Multi-GPU"), timed as the max over ranks; value = all ranks' samples / that time.
--impl reference times the float64 CPU oracle (oracle/) on the host cores instead.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "train samples/sec (fwd+bwd+Adam) on 1 B200; % of HBM/L2 and tensor-pipe peak"
UNIT = "samples/s"
N_BATCHES = 16          # distinct pre-generated batches, cycled
REF_RAYS = 1024         # rays per step in the bounded CPU sample


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_tflops=d["bf16_tflops"], bf16_tflops_sustained=d.get("bf16_tflops_sustained"),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, reasons = [], set()
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(name)
        if sm:
            out["sm_mhz"] = float(np.median(sm))
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


WORKLOADS = {
    1: "BASELINE.json configs[0]: tiny fp32 case, 256 rays x 32 samples, full occupancy, L=4 F=2 T=2^10, 16-wide MLPs",
    2: "BASELINE.json configs[1]: Instant-NGP-default field, 4096 rays x 128 candidates, 128^3 sphere-union occupancy, "
       "L=16 F=2 T=2^19, MLPs 32->64->16 / 31->64->64->3",
    3: "BASELINE.json configs[2]: keyframe-window mapping, 10 synthetic 1200x680 keyframes of the 8x6x3 m room, 2^14 rays x 128 "
       "candidates per step, occupancy FULL then FROM_FIELD every 16 steps, field as config 2",
    4: "BASELINE.json configs[3]: large-table stress, 2^12 rays x 512 candidates, L=16 F=4 T=2^22 N_max=8192 (719 MB of tables), "
       "256^3 occupancy at ~10 %, bf16 MLPs",
    5: "BASELINE.json configs[4]: full-frame render of 4 held-out 1200x680 views, 256 candidates/ray, cut 1e-4, field trained on "
       "config 3's data",
}


def make_workload(n_batches, cfg=2):
    from workloads import configs
    if cfg == 1:
        return configs.config1()
    if cfg == 2:
        return configs.config2(n_batches=n_batches)
    if cfg == 3:
        return configs.config3(n_batches=n_batches)
    if cfg == 4:
        return configs.config4(n_batches=min(n_batches, 8))
    raise ValueError(cfg)


def workload_config(w, extra=None, cfg=2):
    fc = w.field
    c = dict(workload=WORKLOADS[cfg],
             rays_per_step=w.batches[0].n_rays, candidates_per_ray=w.batches[0].n_candidates,
             occupancy_fraction=round(w.extra["occupancy_fraction"], 4) if "occupancy_fraction" in w.extra else None,
             lambda_d=w.lambda_d, table_params=None, mlp_precision=["fp32", "fp16", "bf16"][fc.mlp_precision],
             l2="not flushed: the tables (theta, gradient, Adam m and v: 16 B per parameter, 195 MB at config 2) plus the "
                "per-sample workspace exceed the 126 MB L2, and every step gets a fresh ray batch",
             batches=f"{len(w.batches)} distinct pre-generated batches, cycled")
    if extra:
        c.update(extra)
    return c


# ----------------------------------------------------------------------------- CPU oracle legs

def oracle_step_sample(w, n_rays):
    """The bounded CPU sample: the first n_rays rays of each batch."""
    from workloads import configs
    out = []
    for b in w.batches:
        out.append(configs.RayBatch(b.origins[:n_rays], b.dirs[:n_rays], b.rgb[:n_rays], b.depth[:n_rays],
                                    b.depth_var[:n_rays], b.t_min, b.t_max, b.n_candidates))
    return out


def time_oracle(w, steps, warmup, budget_s=None):
    """Time the oracle as it stands (-fopenmp build) on the host cores.  Returns samples/s etc."""
    from oracle import oracle as orc
    from workloads import configs
    fc = w.field
    nt, nm = orc.param_count(fc)
    theta0 = configs.init_params(fc.seed, nt, orc.mlp_shapes(fc))
    O = orc.Oracle(fc, theta0, omp=True)
    O.set_occupancy(w.bits)
    sample = oracle_step_sample(w, REF_RAYS)
    for i in range(warmup):
        O.train_step(sample[i % len(sample)], w.lambda_d)
    t0 = time.perf_counter()
    total, done = 0, 0
    for i in range(steps):
        st, _ = O.train_step(sample[(warmup + i) % len(sample)], w.lambda_d)
        total += st["n_samples"]
        done += 1
        if budget_s is not None and time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return dict(value=total / dt, seconds=dt, steps=done, samples=total, cores=O.num_threads())


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_workload(N_BATCHES, 2)
    r = time_oracle(w, args.steps, args.warmup, budget_s=150.0)   # stops early past 150 s; steps actually done are reported
    sample = f"{r['steps']} oracle steps, each on the first {REF_RAYS} of the 4096 rays of a config-2 batch ({r['samples']} live samples in {r['seconds']:.1f} s)"
    line = dict(impl="reference", metric=METRIC, value=r["value"], unit=UNIT, n_gpus=args.gpus, steps=r["steps"], warmup=args.warmup,
                ms_per_step=1e3 * r["seconds"] / max(r["steps"], 1), higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=workload_config(w, dict(rays_per_step=REF_RAYS)),
                cpu_baseline=dict(value=r["value"], unit=UNIT, cores=r["cores"], kind="oracle", sample=sample),
                e2e=dict(value=r["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- the CUDA arm

def kernel_model(name, S, R, K, L, F, LF, U, E, mac, n_mlp):
    """Algorithmic bytes / flops of one launch of a kernel class."""
    gather = 8 * L * F * 4 * S
    if name == "encode":
        return dict(bound="hbm", bytes=gather + 12 * S + 4 * LF * S)
    if name == "scatter":
        return dict(bound="hbm", bytes=2 * gather + 4 * LF * S + 12 * S)
    if name == "adam_table":
        return dict(bound="hbm", bytes=32 * F * U)
    if name == "mlp_fwd":
        return dict(bound="alu", flops=2 * mac * S)
    if name == "mlp_bwd":
        return dict(bound="alu", flops=4 * mac * S)
    if name == "composite":
        return dict(bound="hbm", bytes=S * (4 + 4 + 4 + 12) * 2 + S * (4 + 4 + 12) + R * 40)
    if name == "march":
        return dict(bound="alu", flops=40 * R * K)
    return dict(bound="hbm", bytes=0)


# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch from the `ncu --set full` capture of
# profiles/r1q_ncu_full.md (config 2; cold cache, as ncu flushes before every kernel).  bench.py cannot run ncu:
# these are recorded values, refreshed with each committed profile.
NCU_TRAFFIC_CFG2 = {"adam_table": 213411328, "scatter": 37968128, "encode": 40532736, "mlp_bwd": 11986432, "mlp_fwd": 3022336,
                    "adam_mlp": 6556160, "composite": 643584, "march": 381952}


def run_probe_l2():
    """The L2 random-access rates the encoder / scatter rooflines are quoted against (nsm_probe_l2)."""
    import torch
    import paper_2210_13641_b200 as nsm
    from paper_2210_13641_b200 import build as nsm_build
    nsm_build.build()
    torch.cuda.set_device(0)
    rows = []
    for mb in (12, 24, 48, 64, 96, 128, 195, 390):
        g = nsm.probe_l2(mb << 20, 1 << 22, False)
        r = nsm.probe_l2(mb << 20, 1 << 22, True)
        rows.append(dict(table_mb=mb, gathers_per_s=g, reductions_per_s=r))
    print(json.dumps(dict(probe="nsm_probe_l2: 2^22 random 8-byte gathers / red.global.add.v2.f32 per launch, best of 8", rows=rows)))
    return 0


# L2 random-access peaks from `python bench.py --probe-l2` on B200 (profiles/r1p_l2_probe.md): table resident in L2
L2_RANDOM_GATHERS_PER_S = 202e9
L2_RANDOM_REDUCTIONS_PER_S = 160e9


def run_render(args, nsm, replicas, dev, rank, world, peaks):
    """Config 5: forward-only full-frame render (rays/s, samples/s) of a field trained on config 3's data."""
    import torch
    from workloads import configs
    w = configs.config3(n_batches=100)
    fc = w.field
    from dataclasses import replace
    fc = replace(fc, max_candidates=256, max_rays=1 << 16)
    f = nsm.Field(fc, dev)
    f.nsm_set_params(configs.init_params(fc.seed, f.n_table, f.mlp_shapes()))
    train_steps = 500
    for i in range(train_steps):
        if i > 0 and i % 16 == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step(nsm.DeviceBatch(w.batches[i % len(w.batches)], dev), w.lambda_d, want_stats=False)
    f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD)
    occ = float(np.unpackbits(f.nsm_get_occupancy()).mean())
    views = [nsm.DeviceBatch(v, dev) for v in configs.config5_views()]
    hviews = [nsm.HostBatch(v) for v in configs.config5_views()]
    K, W = args.steps, max(args.warmup, 3)
    stream = torch.cuda.current_stream(dev)
    n_rays = views[0].n_rays

    def timed(fn, n):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        ev0.record(stream)
        for i in range(n):
            fn(i)
        ev1.record(stream)
        torch.cuda.synchronize(dev)
        return ev0.elapsed_time(ev1) * 1e-3

    step = lambda i: f.nsm_render(views[i % 4], 1e-4)
    for i in range(W):
        step(i)
    l0 = f.nsm_launch_count()
    sampler = ClockSampler(dev.index)
    t = timed(step, K)
    clocks = sampler.stop()
    launches = f.nsm_launch_count() - l0
    outs = (torch.empty((n_rays, 3), dtype=torch.float32).pin_memory(), torch.empty(n_rays, dtype=torch.float32).pin_memory(),
            torch.empty(n_rays, dtype=torch.float32).pin_memory())
    e2e = lambda i: f.nsm_render_host(hviews[i % 4], 1e-4, outs)
    e2e(0)
    t_e2e = timed(e2e, K)
    f.nsm_profile(True)
    for i in range(min(K, 4)):
        step(i)
    torch.cuda.synchronize(dev)
    prof = f.nsm_profile_read()
    f.nsm_profile(False)
    total_ms = sum(ms for ms, n in prof.values())
    kernels = sorted([dict(kernel=k, total_ms=ms, launches=n, share=ms / total_ms) for k, (ms, n) in prof.items() if n], key=lambda k: -k["share"])
    line = dict(metric="render rays/sec (forward only) on 1 B200", value=K * n_rays / t, unit="rays/s", n_gpus=world, steps=K, warmup=W,
                ms_per_step=1e3 * t / K, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f16", data="synthetic", config=dict(workload=WORKLOADS[5], rays_per_view=n_rays, train_steps=train_steps,
                                                           occupancy_fraction_after_training=occ, mlp_path=f.nsm_mlp_path()),
                clocks=clocks, e2e=dict(value=K * n_rays / t_e2e, unit="rays/s", h2d_bytes_per_step=hviews[0].bytes_in(),
                                        d2h_bytes_per_step=n_rays * 20, ms_per_step=1e3 * t_e2e / K),
                gpu_launches=launches, kernels=kernels)
    f.close()
    print(json.dumps(line))
    return 0


def run_cuda(args):
    import torch
    import paper_2210_13641_b200 as nsm
    from paper_2210_13641_b200 import build as nsm_build, replicas
    from workloads import configs

    rank, local_rank, world = replicas.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback (use --impl reference for the oracle)")
    nsm_build.build()
    dev = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(dev)
    peaks = measured_peaks()

    cfg = args.config
    if cfg == 5:
        return run_render(args, nsm, replicas, dev, rank, world, peaks)
    w = make_workload(N_BATCHES if cfg != 3 else 100, cfg)
    fc = w.field
    f = nsm.Field(fc, dev)
    theta0 = configs.init_params(fc.seed + rank, f.n_table, f.mlp_shapes())
    f.nsm_set_params(theta0)
    if w.bits is not None:
        f.nsm_update_occupancy(nsm.NSM_OCC_SET, w.bits)
    # the batches below are generated and uploaded before the timed region and never modified: declare them
    # ready, so the marcher of step i+1 may run beside the table update of step i (include/nsm.h)
    f.nsm_set_option(nsm.NSM_OPT_BATCH_READY, 1)
    refresh = 16 if cfg == 3 else 0          # config 3: occupancy FROM_FIELD every 16 steps (inside the timed region)
    dbatches = [nsm.DeviceBatch(b, dev) for b in w.batches]
    hbatches = [nsm.HostBatch(b) for b in w.batches]
    K, W = args.steps, max(args.warmup, 3)
    lam = w.lambda_d
    stream = torch.cuda.current_stream(dev)

    def timed(n_steps, step_fn, first):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        replicas.barrier()
        torch.cuda.synchronize(dev)
        ev0.record(stream)
        for i in range(n_steps):
            step_fn(first + i)
        ev1.record(stream)
        torch.cuda.synchronize(dev)
        replicas.barrier()
        return ev0.elapsed_time(ev1) * 1e-3

    # ---- device-resident leg: inputs already in HBM, no host sync inside the timed region
    def dev_step(i):
        if refresh and i > 0 and i % refresh == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step(dbatches[i % len(dbatches)], lam, want_stats=False)
    for i in range(W):
        dev_step(i)
    s0, l0 = f.nsm_total_samples(), f.nsm_launch_count()
    sampler = ClockSampler(dev.index) if rank == 0 else None
    t_dev = timed(K, dev_step, W)
    clocks = sampler.stop() if sampler else None
    samples_dev = f.nsm_total_samples() - s0
    launches = f.nsm_launch_count() - l0
    value, total_samples, t_max = replicas.aggregate_throughput(samples_dev, t_dev)

    # ---- end-to-end leg: HOST buffers through the C-ABI, H2D of the batch and D2H of the stats every step
    def e2e_step(i):
        if refresh and i > 0 and i % refresh == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step_host(hbatches[i % len(hbatches)], lam, want_stats=True)
    for i in range(W):
        e2e_step(i)
    s1 = f.nsm_total_samples()
    t_e2e = timed(K, e2e_step, W + K)
    samples_e2e = f.nsm_total_samples() - s1
    e2e_value, _, _ = replicas.aggregate_throughput(samples_e2e, t_e2e)
    h2d = hbatches[0].bytes_in()
    d2h = 2 * 8 + 4   # the stats read-back: two double accumulators and the sample count

    # ---- config 3 only: the same steps with the batches drawn on the device from the keyframe store (row F1)
    sampled = None
    if cfg == 3 and "keyframes" in w.extra:
        kfs = w.extra["keyframes"]
        for i in range(kfs.n):
            f.nsm_add_keyframe(kfs.store_frame(i))
        b0_ = w.batches[0]

        def sampled_step(i):
            if refresh and i > 0 and i % refresh == 0:
                f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
            f.nsm_train_step_sampled(b0_.n_rays, b0_.t_min, b0_.t_max, b0_.n_candidates, lam, want_stats=False)
        for i in range(W):
            sampled_step(i)
        s3 = f.nsm_total_samples()
        t_s = timed(K, sampled_step, W + 2 * K)
        v_s, _, _ = replicas.aggregate_throughput(f.nsm_total_samples() - s3, t_s)
        sampled = dict(value=v_s, unit=UNIT, ms_per_step=1e3 * t_s / K, keyframes=kfs.n,
                       store_bytes=kfs.n * kfs.W * kfs.H * 5 * 4, api="nsm_train_step_sampled")
        if args.pose:   # row f2: the same leg with the pose gradients computed and the keyframe poses stepped every step
            f.nsm_set_option(nsm.NSM_OPT_POSE_GRADIENTS, 1)

            def pose_step(i):
                sampled_step(i)
                f.nsm_apply_pose_step(0.0, 0.0)          # zero learning rates: the full update path, poses unchanged
            for i in range(W):
                pose_step(i)
            s4 = f.nsm_total_samples()
            t_p = timed(K, pose_step, W + 3 * K)
            v_p, _, _ = replicas.aggregate_throughput(f.nsm_total_samples() - s4, t_p)
            sampled["with_pose_gradients"] = dict(value=v_p, unit=UNIT, ms_per_step=1e3 * t_p / K,
                                                  api="nsm_train_step_sampled + nsm_apply_pose_step, NSM_OPT_POSE_GRADIENTS")

    line = None
    if rank == 0:
        # ---- per-kernel pass (CUDA events around every launch on the field's stream; separate from the headline timing)
        f.nsm_profile(True)
        s2 = f.nsm_total_samples()
        KP = min(K, 200)
        for i in range(KP):
            dev_step(W + 2 * K + i)
        torch.cuda.synchronize(dev)
        prof = f.nsm_profile_read()
        f.nsm_profile(False)
        S_avg = (f.nsm_total_samples() - s2) / KP
        # touched-entry count U of one representative step
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
            model = kernel_model(name, S_avg, b0.n_rays, b0.n_candidates, L, F, L * F, U, f.n_entries, mac, f.n_mlp)
            avg_s = ms * 1e-3 / n
            k = dict(kernel=name, launches_per_step=n / KP, avg_us=1e6 * avg_s, share=ms / total_ms, bound=model["bound"])
            if "bytes" in model:
                k.update(achieved=model["bytes"] / avg_s / 1e9 if avg_s > 0 else 0.0, unit="GB/s", peak=peaks["hbm_gbs"],
                         algorithmic_bytes=model["bytes"])
            else:
                path = f.nsm_mlp_path()
                if name.startswith("mlp") and path.startswith("tcgen05"):
                    k["bound"] = "tensor"
                    peak = peaks["bf16_tflops"]
                else:
                    peak = 148 * 128 * 2 * 1.965e9 / 1e12    # fp32 FMA lanes x 2 flop x max SM clock
                k.update(achieved=model["flops"] / avg_s / 1e12 if avg_s > 0 else 0.0, unit="TFLOP/s", peak=peak,
                         algorithmic_flops=model["flops"])
            k["frac"] = k["achieved"] / k["peak"]
            if name in ("encode", "scatter") and avg_s > 0:
                # what actually bounds S4 / S12 while the tables fit the L2: its random-access rate (8 corners per sample-level)
                acc = 8 * L * S_avg / avg_s
                pk = L2_RANDOM_GATHERS_PER_S if name == "encode" else L2_RANDOM_REDUCTIONS_PER_S
                k["l2_random"] = dict(achieved_accesses_per_s=acc, peak_accesses_per_s=pk, frac=acc / pk,
                                      peak_source="nsm_probe_l2, 48 MB table (profiles/r1p_l2_probe.md)")
            kernels.append(k)
        kernels.sort(key=lambda k: -k["share"])
        top = kernels[0]
        roofline = dict(kernel=top["kernel"], bound=top["bound"], achieved=top["achieved"], peak=top["peak"], unit=top["unit"],
                        frac=top["frac"], traffic=NCU_TRAFFIC_CFG2.get(top["kernel"]) if cfg == 2 else None,
                        traffic_source="profiles/r1q_ncu_full.md (ncu --set full, per launch, cold cache)" if cfg == 2 else None,
                        share_of_step=top["share"], avg_us=top["avg_us"],
                        peak_source=peaks["source"] if top["bound"] != "alu" else "derived: 148 SM x 128 FMA/clk x 2 x 1.965 GHz",
                        samples_per_launch=S_avg, touched_entries=U)
        # ---- CPU baseline: the oracle on the host cores, bounded sample
        cpu = time_oracle(w, steps=40, warmup=1, budget_s=12.0)
        cpu_baseline = dict(value=cpu["value"], unit=UNIT, cores=cpu["cores"], kind="oracle",
                            sample=f"{cpu['steps']} oracle steps, each on the first {REF_RAYS} of the 4096 rays of a config-2 batch "
                                   f"({cpu['samples']} live samples in {cpu['seconds']:.1f} s)")
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=1e3 * t_max / K,
                    higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32" if f.nsm_mlp_path() == "simt_fp32" else
                    ("f16" if fc.mlp_precision == 1 else "bf16"), data="synthetic",
                    config=workload_config(w, cfg=cfg, extra=dict(table_params=f.n_table, mlp_params=f.n_mlp, mlp_path=f.nsm_mlp_path(),
                                                   parallelism=f"{world} independent replica(s)",
                                                   samples_per_step=total_samples / K / world)),
                    rays_per_s=world * K * b0.n_rays / t_max, clocks=clocks, sampled=sampled,
                    e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                             ms_per_step=1e3 * t_e2e / K),
                    gpu_launches=launches, roofline=roofline, kernels=kernels, cpu_baseline=cpu_baseline)
    f.close()
    replicas.barrier()
    if rank == 0:
        print(json.dumps(line))
    replicas.shutdown()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 2000; 40 for --impl reference)")
    ap.add_argument("--warmup", type=int, default=None, help="untimed warm-up steps (default 20; 2 for --impl reference)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--pose", action="store_true", help="config 3: add a sampled leg with pose gradients and pose steps (row f2)")
    ap.add_argument("--probe-l2", action="store_true", help="print the random-gather / vector-reduction rates of nsm_probe_l2 "
                    "over table sizes from L2-resident to DRAM-resident (one JSON line) and exit")
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config to run (default 2 = configs[1], the one the metric is quoted on)")
    args = ap.parse_args()
    if args.probe_l2:
        return run_probe_l2()
    if args.steps is None:
        args.steps = 40 if args.impl == "reference" else {1: 2000, 2: 2000, 3: 100, 4: 200, 5: 3}[args.config]
    if args.warmup is None:
        args.warmup = 2 if args.impl == "reference" else 20
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
