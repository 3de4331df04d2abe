"""Pins of the oracle's ray-batch sampler (row F1, oracle/nsm_oracle.h orc_sample_batch) against
what the pinhole model and the mathematics fix: closed forms, a float64 reprojection loop, an independent numpy
ray generator, hand-evaluated integers and chi-square uniformity.  CPU only."""
import numpy as np
import pytest

from oracle import oracle as orc
from workloads import scenes


def make_kf(W, H, fx, fy, R=None, t=(0.0, 0.0, 0.0), depth=None, var=None, rgb=None, seed=0):
    rng = np.random.default_rng(seed)
    return dict(width=W, height=H, fx=fx, fy=fy, cx=(W - 1) / 2.0, cy=(H - 1) / 2.0,
                R=np.eye(3) if R is None else R, t=np.asarray(t, np.float64),
                rgb=rng.uniform(0, 1, (H, W, 3)).astype(np.float32) if rgb is None else rgb,
                depth=rng.uniform(0.5, 4.0, (H, W)).astype(np.float32) if depth is None else depth,
                depth_var=rng.uniform(1e-4, 1e-2, (H, W)).astype(np.float32) if var is None else var)


def rot(axis, ang):
    axis = np.asarray(axis, float) / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(ang) * K + (1 - np.cos(ang)) * K @ K


def mix32(x):
    x ^= x >> 16; x = (x * 0x7feb352d) & 0xffffffff
    x ^= x >> 15; x = (x * 0x846ca68b) & 0xffffffff
    x ^= x >> 16
    return x


def hash32(seed, step, r, k):
    h = mix32((seed & 0xffffffff) ^ 0x9e3779b9)
    for w in (seed >> 32, step, r, k):
        h = mix32(h ^ w)
    return h


def test_indices_hand_evaluated():
    """kf and pix are the multiply-shift maps of the two selector hashes, in exact Python integers."""
    kfs = [make_kf(31, 17, 20.0, 20.0, seed=i) for i in range(5)] + [make_kf(13, 7, 9.0, 9.0, seed=9)]
    out = orc.sample_batch(kfs, seed=0x1234567890ab, draw=7, n_rays=500)
    for r in range(500):
        kf = (hash32(0x1234567890ab, 7, r, 0xffff0001) * len(kfs)) >> 32
        k = kfs[kf]
        pix = (hash32(0x1234567890ab, 7, r, 0xffff0002) * (k["width"] * k["height"])) >> 32
        assert (out["kf"][r], out["pix"][r]) == (kf, pix)
        v, u = divmod(pix, k["width"])
        assert np.array_equal(out["rgb"][r], k["rgb"][v, u])
    assert out["kf"].max() == 5 and out["pix"].max() < 31 * 17


def test_principal_point_is_the_forward_axis_and_dirs_are_unit():
    R = rot([0.3, -1.0, 0.5], 1.1)
    t = np.array([1.5, -2.0, 0.25])
    kf = make_kf(33, 21, 40.0, 35.0, R=R, t=t)          # odd sizes: the principal point is a pixel centre
    out = orc.sample_batch([kf], 1, 1, 4000)
    centre = 10 * 33 + 16
    hit = out["pix"] == centre
    assert hit.any()
    assert np.array_equal(out["dirs"][hit][0], R[:, 2].astype(np.float32))
    assert np.abs(np.linalg.norm(out["dirs"].astype(np.float64), axis=1) - 1.0).max() <= 3e-7
    assert np.array_equal(out["origins"], np.broadcast_to(t.astype(np.float32), (4000, 3)))


def test_reprojection_closes_in_float64():
    """o + range * d, projected back through the pinhole model in float64, lands on the pixel it came from at the
    z-depth stored for it: fixes the rotation convention (camera-to-world, row-major), the axis signs and the
    z-depth -> range conversion.  A transposed R, a swapped u/v or a missing |(xc, yc, 1)| all fail."""
    R = rot([1.0, 2.0, -0.5], 2.3)
    t = np.array([4.0, 3.0, 1.5])
    kf = make_kf(64, 48, 55.0, 50.0, R=R, t=t, seed=3)
    out = orc.sample_batch([kf], 2, 3, 3000)
    P = out["origins"].astype(np.float64) + out["depth"].astype(np.float64)[:, None] * out["dirs"].astype(np.float64)
    Pc = (P - t) @ R                                   # world -> camera: R^T (P - t)
    u = Pc[:, 0] / Pc[:, 2] * kf["fx"] + kf["cx"]
    v = Pc[:, 1] / Pc[:, 2] * kf["fy"] + kf["cy"]
    pu, pv = out["pix"] % 64, out["pix"] // 64
    assert np.abs(u - pu).max() <= 2e-4 and np.abs(v - pv).max() <= 2e-4
    z = kf["depth"][pv, pu].astype(np.float64)
    assert np.abs(Pc[:, 2] - z).max() <= 1e-6 * z.max()


def test_plane_closed_form_and_variance_ratio():
    """A fronto-parallel plane at z = D is seen at range D sqrt(1 + xc^2 + yc^2); the variance scales with its square."""
    W, H, f, D = 41, 31, 30.0, 2.5
    kf = make_kf(W, H, f, f, depth=np.full((H, W), D, np.float32), var=np.full((H, W), 0.04, np.float32))
    out = orc.sample_batch([kf], 3, 1, 2000)
    u, v = (out["pix"] % W).astype(np.float64), (out["pix"] // W).astype(np.float64)
    n2 = ((u - kf["cx"]) / f) ** 2 + ((v - kf["cy"]) / f) ** 2 + 1.0
    assert np.abs(out["depth"] - D * np.sqrt(n2)).max() <= 3e-7 * D * np.sqrt(n2.max())
    assert np.abs(out["depth_var"] - np.float64(np.float32(0.04)) * n2).max() <= 3e-7 * 0.04 * n2.max()
    # invalid depth stays invalid (reading R13: depth <= 0 masks the depth term)
    kf0 = make_kf(W, H, f, f, depth=np.zeros((H, W), np.float32))
    assert not orc.sample_batch([kf0], 3, 1, 100)["depth"].any()


def test_against_the_workload_generator_rays():
    """The synthetic-room keyframes were ray-cast with an independent float64 numpy ray generator
    (workloads.scenes.KeyframeSet.rays); the sampler's rays, colours, ranges and variances agree with its frames."""
    room = scenes.Room(3)
    kfs = scenes.KeyframeSet(room, 3, 2, width=60, height=34)
    store = [kfs.store_frame(i) for i in range(2)]
    out = orc.sample_batch(store, 11, 5, 1500)
    for i in range(2):
        sel = out["kf"] == i
        fr = kfs.frame(i)
        pix = out["pix"][sel]
        assert np.abs(out["dirs"][sel] - fr["d"][pix]).max() <= 5e-7
        assert np.array_equal(out["origins"][sel], fr["o"][pix])
        assert np.array_equal(out["rgb"][sel], fr["rgb"][pix])
        assert np.abs(out["depth"][sel] - fr["depth"][pix]).max() <= 3e-7 * fr["depth"].max()
        assert np.abs(out["depth_var"][sel] - fr["var"][pix]).max() <= 1e-6 * fr["var"].max()


def test_uniform_over_keyframes_and_pixels_and_draws_differ():
    n_kf, W, H, R = 7, 16, 8, 70000
    kfs = [make_kf(W, H, 10.0, 10.0, seed=i) for i in range(n_kf)]
    a = orc.sample_batch(kfs, 42, 1, R)
    exp = R / n_kf
    chi_kf = ((np.bincount(a["kf"], minlength=n_kf) - exp) ** 2 / exp).sum()
    assert chi_kf < 22.5                                 # chi^2(6) 99.9 %
    exp = R / (W * H)
    chi_px = ((np.bincount(a["pix"], minlength=W * H) - exp) ** 2 / exp).sum()
    assert chi_px < 181.0                                # chi^2(127) 99.9 %
    joint = np.bincount(a["kf"].astype(np.int64) * 4 + (a["pix"] & 3), minlength=n_kf * 4)
    exp = R / (n_kf * 4)
    assert ((joint - exp) ** 2 / exp).sum() < 56.9       # chi^2(27) 99.9 %: keyframe and pixel draws are independent
    b = orc.sample_batch(kfs, 42, 2, R)
    assert (a["pix"] != b["pix"]).mean() > 0.98 and (a["kf"] != b["kf"]).mean() > 0.8
    c = orc.sample_batch(kfs, 42, 1, R)
    assert all(np.array_equal(a[k], c[k]) for k in a)    # counter-based: same draw, same batch
