"""Row f3 of SURVEY.md 8(f): a synthetic replay of the paper's depth-loss ablation (metrics
PAPER.md:210: PSNR and depth L1) on data this repository can generate.

Three fields are trained on the same keyframe store (the synthetic room of config 3: noisy depth with 5 % gross
outliers that are flagged only by a large variance) through nsm_train_step_sampled:

    none      lambda_D = 0                      photometric loss only
    raw       Sigma_D := its mean over pixels   depth loss without the uncertainty weighting ("raw depth")
    weighted  Sigma_D as estimated              the paper's loss, Eq. 4

and evaluated on held-out views with nsm_render against the analytic ground truth: PSNR of the colour and L1 error of
the expected depth.  This is an experiment, not a parity test: every number comes from the CUDA path.

    python -m paper_2210_13641_b200.ablation [--steps 600] [--width 300 --height 170] [--rays 4096]
"""
import argparse
import time
from dataclasses import replace

import numpy as np


def _psnr(a, b):
    mse = float(np.mean((a.astype(np.float64) - b.astype(np.float64)) ** 2))
    return 10.0 * np.log10(1.0 / max(mse, 1e-12))


def run(device="cuda:0", steps=600, width=300, height=170, n_keyframes=10, n_rays=4096, eval_every=200, n_views=2,
        seed=3, variants=("none", "raw", "weighted"), log=print):
    import torch

    import paper_2210_13641_b200 as nsm
    from workloads import configs, scenes

    w = configs.config3(seed=seed, R=n_rays, K=128, n_keyframes=n_keyframes, n_batches=1, width=width, height=height)
    kfs = w.extra["keyframes"]
    store = [kfs.store_frame(i) for i in range(n_keyframes)]
    inlier_var = np.concatenate([s["depth_var"][s["depth_var"] < 0.5].ravel() for s in store])
    raw_var = float(inlier_var.mean())
    held = scenes.KeyframeSet(w.extra["room"], seed + 5000, n_views, width, height)
    truth = [held.frame(i) for i in range(n_views)]
    views = [configs.RayBatch(t["o"], t["d"], None, None, None, 0.05, 10.5, 256) for t in truth]
    seen = kfs.frame(0)                                  # one TRAINING view, to tell fitting from generalisation
    seen_view = configs.RayBatch(seen["o"], seen["d"], None, None, None, 0.05, 10.5, 256)
    fc = replace(w.field, max_rays=max(n_rays, 1 << 15), max_candidates=256)
    dev = torch.device(device)
    results = {}
    for variant in variants:
        f = nsm.Field(fc, dev)
        f.nsm_set_params(configs.init_params(seed, f.n_table, f.mlp_shapes()))
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
            if step % eval_every == 0 or step == steps:
                torch.cuda.synchronize(dev)
                train_s += time.perf_counter() - t0
                ps, l1 = [], []
                for dv, t in zip(dviews, truth):
                    rgb, dep, opa = (x.cpu().numpy() for x in f.nsm_render(dv, 1e-4))
                    ps.append(_psnr(rgb, t["rgb"]))
                    l1.append(float(np.mean(np.abs(dep.astype(np.float64) - t["range"].astype(np.float64)))))
                rgb_s, dep_s, _ = (x.cpu().numpy() for x in f.nsm_render(dseen, 1e-4))
                curve.append(dict(step=step, seconds=train_s, psnr=float(np.mean(ps)), depth_l1_m=float(np.mean(l1)),
                                  psnr_seen=_psnr(rgb_s, seen["rgb"]),
                                  depth_l1_seen_m=float(np.mean(np.abs(dep_s.astype(np.float64) - seen["range"].astype(np.float64))))))
                c = curve[-1]
                log(f"{variant:9s} step {step:5d}  train {train_s:6.2f} s  held-out: PSNR {c['psnr']:6.2f} dB  depth L1 {100 * c['depth_l1_m']:7.2f} cm"
                    f"   training view: PSNR {c['psnr_seen']:6.2f} dB  depth L1 {100 * c['depth_l1_seen_m']:7.2f} cm")
            else:
                train_s += time.perf_counter() - t0
        results[variant] = curve
        f.close()
    return results


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--steps", type=int, default=600)
    ap.add_argument("--width", type=int, default=300)
    ap.add_argument("--height", type=int, default=170)
    ap.add_argument("--rays", type=int, default=4096)
    ap.add_argument("--keyframes", type=int, default=10)
    ap.add_argument("--eval-every", type=int, default=200)
    a = ap.parse_args()
    res = run(steps=a.steps, width=a.width, height=a.height, n_rays=a.rays, n_keyframes=a.keyframes, eval_every=a.eval_every)
    print("\n| variant | step | train s | held-out PSNR dB | held-out depth L1 cm | training-view PSNR dB | training-view depth L1 cm |\n|---|---:|---:|---:|---:|---:|---:|")
    for v, curve in res.items():
        for c in curve:
            print(f"| {v} | {c['step']} | {c['seconds']:.2f} | {c['psnr']:.2f} | {100 * c['depth_l1_m']:.2f} | {c['psnr_seen']:.2f} | {100 * c['depth_l1_seen_m']:.2f} |")


if __name__ == "__main__":
    main()
