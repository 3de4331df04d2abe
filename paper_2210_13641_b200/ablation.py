"""Row f3 of SURVEY.md 8(f): a synthetic replay of the paper's depth-loss ablation (metrics
PAPER.md:210: PSNR and depth L1) on data this repository can generate.

Three fields are trained on the same keyframe store (the synthetic room of config 3: noisy depth with 5 % gross
outliers that are flagged only by a large variance) through nsm_train_step_sampled:

    none      lambda_D = 0                      photometric loss only
    raw       Sigma_D := its mean over pixels   depth loss without the uncertainty weighting ("raw depth")
    weighted  Sigma_D as estimated              the paper's loss, Eq. 4

and evaluated on held-out views with nsm_render against the analytic ground truth: PSNR of the colour and L1 error of
the expected depth.  This is an experiment, not a parity test: every number comes from the CUDA path.

    python -m paper_2210_13641_b200.ablation [--steps 600] [--width 300 --height 170] [--rays 4096] [--seeds 0 1 2]

`--width 1200 --height 680 --rays 16384` is config 3's size.  `--seeds` repeats every variant with
different training seeds (parameter initialisation and ray draws) on the same scene and reports mean and standard
deviation, which is what separates a variant's effect from the run-to-run noise of atomic summation order and Adam.
"""
import argparse
import json
import time
from dataclasses import replace

import numpy as np


def psnr(image, truth, peak=1.0):
    """peak signal-to-noise ratio in dB, 10 log10(peak^2 / MSE) over all pixels and channels."""
    mse = float(np.mean((np.asarray(image, np.float64) - np.asarray(truth, np.float64)) ** 2))
    return 10.0 * np.log10(peak * peak / max(mse, 1e-12))


def depth_l1(depth, truth, valid=None):
    """L1 depth error, the mean of |D_hat - D_true| over the (valid) pixels, in the unit of the inputs."""
    d = np.abs(np.asarray(depth, np.float64) - np.asarray(truth, np.float64))
    if valid is not None:
        d = d[np.asarray(valid, bool)]
    return float(d.mean())


_psnr = psnr


def run(device="cuda:0", steps=600, width=300, height=170, n_keyframes=10, n_rays=4096, eval_every=200, n_views=2,
        seed=3, variants=("none", "raw", "weighted"), log=print, train_seed=None, eval_at=None, workload=None):
    """seed: the scene (room, keyframe poses, sensor noise); train_seed (default: seed): parameter initialisation and the
    sampler's ray draws.  eval_at: explicit list of evaluation steps (default: every eval_every).  workload: a config-3
    workload already generated for this scene (its keyframes are cast once and reused across train seeds)."""
    import torch

    import paper_2210_13641_b200 as nsm
    from workloads import configs, scenes

    w = workload or configs.config3(seed=seed, R=n_rays, K=128, n_keyframes=n_keyframes, n_batches=1, width=width, height=height)
    train_seed = seed if train_seed is None else train_seed
    eval_steps = set(eval_at) if eval_at else {s_ for s_ in range(eval_every, steps + 1, eval_every)}
    eval_steps.add(steps)
    kfs = w.extra["keyframes"]
    store = [kfs.store_frame(i) for i in range(n_keyframes)]
    inlier_var = np.concatenate([s["depth_var"][s["depth_var"] < 0.5].ravel() for s in store])
    raw_var = float(inlier_var.mean())
    held = scenes.KeyframeSet(w.extra["room"], seed + 5000, n_views, width, height)
    truth = [held.frame(i) for i in range(n_views)]
    views = [configs.RayBatch(t["o"], t["d"], None, None, None, 0.05, 10.5, 256) for t in truth]
    seen = kfs.frame(0)                                  # one TRAINING view, to tell fitting from generalisation
    seen_view = configs.RayBatch(seen["o"], seen["d"], None, None, None, 0.05, 10.5, 256)
    fc = replace(w.field, max_rays=max(n_rays, 1 << 15), max_candidates=256, seed=train_seed)
    dev = torch.device(device)
    results = {}
    for variant in variants:
        f = nsm.Field(fc, dev)
        f.nsm_set_params(configs.init_params(train_seed, f.n_table, f.mlp_shapes()))
        for s in store:
            kf = dict(s)
            if variant == "raw":
                kf["depth_var"] = np.full_like(s["depth_var"], raw_var)
            f.nsm_add_keyframe(kf)
        lam = 0.0 if variant == "none" else w.lambda_d
        dviews = [nsm.DeviceBatch(v, dev) for v in views]
        dseen = nsm.DeviceBatch(seen_view, dev)
        curve, train_s = [], 0.0
        for step in range(1, steps + 1):
            t0 = time.perf_counter()
            if step > 16 and step % 16 == 0:
                f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
            f.nsm_train_step_sampled(n_rays, 0.05, 10.5, 128, lam, want_stats=False)
            if step in eval_steps:
                torch.cuda.synchronize(dev)
                train_s += time.perf_counter() - t0
                ps, l1 = [], []
                for dv, t in zip(dviews, truth):
                    rgb, dep, opa = (x.cpu().numpy() for x in f.nsm_render(dv, 1e-4))
                    ps.append(_psnr(rgb, t["rgb"]))
                    l1.append(depth_l1(dep, t["range"]))
                rgb_s, dep_s, _ = (x.cpu().numpy() for x in f.nsm_render(dseen, 1e-4))
                curve.append(dict(step=step, seconds=train_s, psnr=float(np.mean(ps)), depth_l1_m=float(np.mean(l1)),
                                  psnr_seen=_psnr(rgb_s, seen["rgb"]),
                                  depth_l1_seen_m=depth_l1(dep_s, seen["range"])))
                c = curve[-1]
                log(f"{variant:9s} step {step:5d}  train {train_s:6.2f} s  held-out: PSNR {c['psnr']:6.2f} dB  depth L1 {100 * c['depth_l1_m']:7.2f} cm"
                    f"   training view: PSNR {c['psnr_seen']:6.2f} dB  depth L1 {100 * c['depth_l1_seen_m']:7.2f} cm")
            else:
                train_s += time.perf_counter() - t0
        results[variant] = curve
        f.close()
    return results


def aggregate(runs):
    """runs: list (one per train seed) of {variant: curve}.  Returns {variant: [dict(step, seconds, <metric>_mean, <metric>_std)]}."""
    out = {}
    for v in runs[0]:
        rows = []
        for i, c0 in enumerate(runs[0][v]):
            row = dict(step=c0["step"], seconds=float(np.mean([r[v][i]["seconds"] for r in runs])), n=len(runs))
            for k in ("psnr", "depth_l1_m", "psnr_seen", "depth_l1_seen_m"):
                vals = np.array([r[v][i][k] for r in runs], np.float64)
                row[k + "_mean"], row[k + "_std"] = float(vals.mean()), float(vals.std(ddof=1)) if len(vals) > 1 else 0.0
            rows.append(row)
        out[v] = rows
    return out


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--width", type=int, default=300)
    ap.add_argument("--height", type=int, default=170)
    ap.add_argument("--rays", type=int, default=4096)
    ap.add_argument("--keyframes", type=int, default=10)
    ap.add_argument("--eval-every", type=int, default=200)
    ap.add_argument("--eval-at", type=int, nargs="*", default=None, help="explicit evaluation steps")
    ap.add_argument("--scene-seed", type=int, default=3)
    ap.add_argument("--seeds", type=int, nargs="*", default=None, help="training seeds (default: the scene seed alone)")
    ap.add_argument("--outlier-fraction", type=float, default=0.05, help="share of pixels with a gross depth error flagged only by "
                    "their variance (BASELINE.json config 3: 0.05)")
    ap.add_argument("--json", default=None, help="write every curve to this file")
    a = ap.parse_args()
    from workloads import configs
    w = configs.config3(seed=a.scene_seed, R=a.rays, K=128, n_keyframes=a.keyframes, n_batches=1, width=a.width, height=a.height,
                        outlier_fraction=a.outlier_fraction)
    seeds = a.seeds if a.seeds else [a.scene_seed]
    runs = [run(steps=a.steps, width=a.width, height=a.height, n_rays=a.rays, n_keyframes=a.keyframes, eval_every=a.eval_every,
                seed=a.scene_seed, train_seed=ts, eval_at=a.eval_at, workload=w) for ts in seeds]
    agg = aggregate(runs)
    if a.json:
        with open(a.json, "w") as fh:
            json.dump(dict(args=vars(a), runs=runs, aggregate=agg), fh)
    pm = lambda r, k, sc=1.0: f"{sc * r[k + '_mean']:.2f} +- {sc * r[k + '_std']:.2f}"
    print(f"\n{len(seeds)} training seed(s) {seeds}, scene seed {a.scene_seed}, outlier fraction {a.outlier_fraction}, {a.keyframes} keyframes {a.width}x{a.height}, {a.rays} rays/step; mean +- sample std over the seeds")
    print("| variant | step | train s | held-out PSNR dB | held-out depth L1 cm | training-view PSNR dB | training-view depth L1 cm |\n|---|---:|---:|---:|---:|---:|---:|")
    for v, rows in agg.items():
        for r in rows:
            print(f"| {v} | {r['step']} | {r['seconds']:.2f} | {pm(r, 'psnr')} | {pm(r, 'depth_l1_m', 100)} | {pm(r, 'psnr_seen')} | {pm(r, 'depth_l1_seen_m', 100)} |")


if __name__ == "__main__":
    main()
