"""Row f2 in use: joint optimisation of keyframe poses and field (L_M(T, Theta)) on the synthetic room.

Half of the keyframes are handed to the store with perturbed poses (a few centimetres and a fraction of a degree, the
other half stay exact and anchor the gauge).  The field is trained with nsm_train_step_sampled; with --refine every
step is followed by nsm_apply_pose_step.  Reported: mean translation / rotation error of the perturbed keyframes over
training.  An experiment on the CUDA path, not a parity test.

    python -m paper_2210_13641_b200.pose_refine [--steps 3000] [--sigma-t 0.03] [--sigma-r-deg 0.5]
"""
import argparse
from dataclasses import replace

import numpy as np


def _rot(axis, ang):
    axis = axis / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(ang) * K + (1 - np.cos(ang)) * K @ K


def pose_errors(f, truth, idx):
    et, er = [], []
    for k in idx:
        R, t = f.nsm_get_keyframe_pose(k)
        et.append(np.linalg.norm(t.astype(np.float64) - truth[k][1]))
        c = (np.trace(R.astype(np.float64) @ truth[k][0].T) - 1.0) / 2.0
        er.append(np.degrees(np.arccos(np.clip(c, -1.0, 1.0))))
    return float(np.mean(et)), float(np.mean(er))


def run(device="cuda:0", steps=3000, width=300, height=170, n_keyframes=8, n_rays=4096, sigma_t=0.03, sigma_r_deg=0.5,
        refine=True, warm=300, lr_t=1e-3, lr_r=5e-4, seed=3, log=print, every=500):
    import torch

    import paper_2210_13641_b200 as nsm
    from workloads import configs

    w = configs.config3(seed=seed, R=n_rays, K=128, n_keyframes=n_keyframes, n_batches=1, width=width, height=height)
    kfs = w.extra["keyframes"]
    rng = np.random.default_rng(seed + 77)
    truth, store, moved = [], [], []
    for i in range(n_keyframes):
        s = kfs.store_frame(i)
        R0, t0 = np.asarray(s["R"], np.float64), np.asarray(s["t"], np.float64)
        truth.append((R0, t0))
        if i % 2 == 1:                                     # perturb every other keyframe
            s = dict(s)
            s["R"] = _rot(rng.normal(size=3), np.radians(sigma_r_deg) * rng.uniform(0.5, 1.5)) @ R0
            s["t"] = t0 + sigma_t * rng.normal(size=3)
            moved.append(i)
        store.append(s)
    fc = replace(w.field, max_rays=n_rays)
    f = nsm.Field(fc, torch.device(device))
    f.nsm_set_params(configs.init_params(seed, f.n_table, f.mlp_shapes()))
    f.nsm_set_option(nsm.NSM_OPT_POSE_GRADIENTS, 1 if refine else 0)
    for s in store:
        f.nsm_add_keyframe(s)
    curve = [dict(step=0, **dict(zip(("trans_m", "rot_deg"), pose_errors(f, truth, moved))))]
    log(f"step     0  translation error {100 * curve[0]['trans_m']:6.2f} cm  rotation error {curve[0]['rot_deg']:.3f} deg")
    for step in range(1, steps + 1):
        if step > 16 and step % 16 == 0:
            f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD, sync=False)
        f.nsm_train_step_sampled(n_rays, 0.05, 10.5, 128, w.lambda_d, want_stats=False)
        if refine and step > warm:                         # let the field take shape before the poses move
            f.nsm_apply_pose_step(lr_t, lr_r)
        if step % every == 0 or step == steps:
            e = pose_errors(f, truth, moved)
            curve.append(dict(step=step, trans_m=e[0], rot_deg=e[1]))
            log(f"step {step:5d}  translation error {100 * e[0]:6.2f} cm  rotation error {e[1]:.3f} deg")
    f.close()
    return curve


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--steps", type=int, default=3000)
    ap.add_argument("--sigma-t", type=float, default=0.03)
    ap.add_argument("--sigma-r-deg", type=float, default=0.5)
    ap.add_argument("--lr-t", type=float, default=1e-3)
    ap.add_argument("--lr-r", type=float, default=5e-4)
    ap.add_argument("--no-refine", action="store_true")
    a = ap.parse_args()
    run(steps=a.steps, sigma_t=a.sigma_t, sigma_r_deg=a.sigma_r_deg, refine=not a.no_refine, lr_t=a.lr_t, lr_r=a.lr_r)


if __name__ == "__main__":
    main()
