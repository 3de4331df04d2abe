"""Pins of the oracle's pose gradients (row f2; Eq. 3 is minimised over the poses T too): central finite
differences of the oracle's own loss under a translation of a ray's origin and a rotation of its direction, plus two
structural cases.  CPU only."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from workloads import configs


def tiny(sh_degree=3, seed=0, R=10, K=16):
    w = configs.config1()
    fc = replace(w.field, sh_degree=sh_degree, max_rays=R, max_candidates=K)
    b = w.batches[0]
    b = replace(b, origins=b.origins[:R].copy(), dirs=b.dirs[:R].copy(), rgb=b.rgb[:R].copy(), depth=b.depth[:R].copy(),
                depth_var=b.depth_var[:R].copy(), n_candidates=K)
    n_table, n_mlp = orc.param_count(fc)
    theta = configs.init_params(seed, n_table, orc.mlp_shapes(fc)).astype(np.float64)
    theta[:n_table] *= 3e3                       # tables that matter: the field varies across cells
    theta[n_table:] *= 1.5
    return fc, b, theta


def loss(fc, theta, b, lam=0.3):
    O = orc.Oracle(fc, theta.copy())
    return O.train_step(b, lam, apply_adam=False)[0]["loss"]


def rot(axis, ang):
    K = np.zeros((3, 3))
    a = np.eye(3)[axis]
    K[0, 1], K[0, 2], K[1, 0], K[1, 2], K[2, 0], K[2, 1] = -a[2], a[1], a[2], -a[0], -a[1], a[0]
    return np.eye(3) + np.sin(ang) * K + (1 - np.cos(ang)) * K @ K


def fd_check(name, analytic, perturb, h, n, tol):
    """analytic[i]: claimed derivative; perturb(i, s) -> batch perturbed by s*h along coordinate i."""
    ok = skipped = 0
    worst = 0.0
    scale = np.abs(analytic).max()
    for i in range(n):
        lp, l0, lm = perturb(i, +1), perturb(i, 0), perturb(i, -1)
        fd = (lp - lm) / (2 * h)
        curv = abs(lp - 2 * l0 + lm) / h          # a kink of the piecewise-trilinear field inside the stencil
        if curv > 0.02 * scale:
            skipped += 1
            continue
        worst = max(worst, abs(fd - analytic[i]) / scale)
        ok += 1
    assert ok >= 0.5 * n, (name, ok, skipped)
    assert worst <= tol, (name, worst)
    return ok, skipped


@pytest.mark.parametrize("sh_degree", [1, 3, 4])
def test_translation_and_rotation_gradients_by_finite_differences(sh_degree):
    fc, b, theta = tiny(sh_degree)
    O = orc.Oracle(fc, theta.copy())
    _, tr = O.train_step(b, 0.3, apply_adam=False, trace=("g_o", "tau"))
    R = b.n_rays
    h = 2.0 ** -13      # small against the finest cell (extent 5 / 32): few stencils straddle a kink of the trilinear field

    def shift(i, s):
        r, c = divmod(i, 3)
        o = b.origins.copy()
        o[r, c] += np.float32(s * h)
        return loss(fc, theta, replace(b, origins=o))

    def turn(i, s):
        r, k = divmod(i, 3)
        d = b.dirs.astype(np.float64).copy()
        d[r] = rot(k, s * h) @ d[r]
        return loss(fc, theta, replace(b, dirs=d.astype(np.float32)))

    fd_check("g_o", tr["g_o"].reshape(-1), shift, h, 3 * R, 1e-2)
    fd_check("tau", tr["tau"].reshape(-1), turn, h, 3 * R, 1e-2)
    assert np.abs(tr["g_o"]).max() > 0 and np.abs(tr["tau"]).max() > 0


def test_constant_tables_leave_only_the_direction_encoding():
    """With every table entry equal the encoding does not depend on x: dL/do = 0 exactly and dL/dx = 0; the rotation
    gradient is then the SH path alone and vanishes too when Y is the constant Y_00 (sh_degree = 1)."""
    for n, expect_tau in ((1, False), (3, True)):
        fc, b, theta = tiny(n)
        n_table, _ = orc.param_count(fc)
        theta[:n_table] = 0.37
        O = orc.Oracle(fc, theta.copy())
        _, tr = O.train_step(b, 0.3, apply_adam=False, trace=("g_o", "tau", "dx"))
        assert np.abs(tr["dx"]).max() <= 1e-12 and np.abs(tr["g_o"]).max() <= 1e-12
        assert (np.abs(tr["tau"]).max() > 1e-9) == expect_tau


def test_translation_gradient_is_the_sum_of_the_sample_gradients():
    """dL/do_r = (1/extent) sum_s dL/dx_s over the ray's samples; a whole-batch translation is the sum over rays."""
    fc, b, theta = tiny(3)
    O = orc.Oracle(fc, theta.copy())
    _, tr = O.train_step(b, 0.3, apply_adam=False, trace=("g_o", "dx", "s_ray"))
    acc = np.zeros_like(tr["g_o"])
    np.add.at(acc, tr["s_ray"], tr["dx"] * float(np.float32(1.0) / np.float32(fc.aabb_extent)))   # S0's fp32 inv_extent
    assert np.abs(acc - tr["g_o"]).max() <= 1e-12 * max(1.0, np.abs(acc).max())
    h = 2.0 ** -13
    for c in range(3):
        o = b.origins.copy()
        lp = loss(fc, theta, replace(b, origins=(o + np.float32(h) * np.eye(3, dtype=np.float32)[c])))
        lm = loss(fc, theta, replace(b, origins=(o - np.float32(h) * np.eye(3, dtype=np.float32)[c])))
        fd, an = (lp - lm) / (2 * h), tr["g_o"][:, c].sum()
        assert abs(fd - an) <= 0.03 * np.abs(tr["g_o"]).sum(0).max() + 1e-9, (c, fd, an)


def test_pose_step_exponential_map_and_adam():
    """The update R <- exp(-[w]x) R against scipy's matrix exponential, orthonormality, the first Adam step's closed form
    (delta = lr sign(g)), torch.optim.Adam on the 6-vector over several steps, and the world-frame convention: the
    update by w turns every world direction d = R d_cam by exp(-[w]x), which is what tau = dL/d(omega) is the gradient of."""
    import scipy.linalg
    import torch
    rng = np.random.default_rng(5)
    R0 = rot(0, 0.4) @ rot(1, -0.9) @ rot(2, 0.2)
    t0 = rng.normal(size=3)
    g = rng.normal(size=6) * np.array([1, 1e-3, 10, 1e-2, 1, 5])
    R, t, m, v = R0.copy(), t0.copy(), np.zeros(6), np.zeros(6)
    cnt = orc.pose_step(R, t, m, v, 0, g, 1e-3, 2e-3)
    assert cnt == 1
    assert np.abs(t - (t0 - 1e-3 * np.sign(g[:3]))).max() <= 1e-12          # Adam step 1: -lr sign(g)
    w = 2e-3 * np.sign(g[3:])
    K = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])
    assert np.abs(R - scipy.linalg.expm(-K) @ R0).max() <= 1e-13
    assert np.abs(R @ R.T - np.eye(3)).max() <= 1e-13 and abs(np.linalg.det(R) - 1) <= 1e-13
    # several steps against torch.optim.Adam on the raw 6-vector with per-group learning rates
    p_t = torch.zeros(3, dtype=torch.float64, requires_grad=True)
    p_r = torch.zeros(3, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([dict(params=[p_t], lr=1e-3), dict(params=[p_r], lr=2e-3)], betas=(0.9, 0.99), eps=1e-15)
    R, t, m, v, cnt = R0.copy(), t0.copy(), np.zeros(6), np.zeros(6), 0
    Racc = R0.copy()
    for k in range(6):
        gk = rng.normal(size=6)
        prev_r = p_r.detach().numpy().copy()
        p_t.grad, p_r.grad = torch.tensor(gk[:3]), torch.tensor(gk[3:])
        opt.step()
        cnt = orc.pose_step(R, t, m, v, cnt, gk, 1e-3, 2e-3)
        assert np.abs(t - (t0 + p_t.detach().numpy())).max() <= 1e-12
        dw = -(p_r.detach().numpy() - prev_r)                                # this step's delta_omega
        Kk = np.array([[0, -dw[2], dw[1]], [dw[2], 0, -dw[0]], [-dw[1], dw[0], 0]])
        Racc = scipy.linalg.expm(-Kk) @ Racc
        assert np.abs(R - Racc).max() <= 1e-12
    # tiny and zero rotations stay finite and exact to first order
    R, t, m, v = R0.copy(), t0.copy(), np.zeros(6), np.zeros(6)
    orc.pose_step(R, t, m, v, 0, np.array([0, 0, 0, 1e-30, 0, 0.0]), 1e-3, 1e-20)
    assert np.isfinite(R).all() and np.abs(R - R0).max() <= 1e-15


def test_pose_step_descends_the_loss():
    """Moving one keyframe's rays by a small se(3) step against (g_o sums | tau sums) lowers the oracle's loss by the
    first-order amount -|g|^2 step (the sums ARE the keyframe gradient, in the convention the update uses)."""
    fc, b, theta = tiny(3)
    O = orc.Oracle(fc, theta.copy())
    st, tr = O.train_step(b, 0.3, apply_adam=False, trace=("g_o", "tau"))
    G = np.concatenate([tr["g_o"].sum(0), tr["tau"].sum(0)])
    # all rays as one rigid body rotating about a common centre c: o <- c + E (o - c), d <- E d, then o <- o - eps g_t
    c = b.origins.astype(np.float64).mean(0)
    # gradient of that motion: translation = sum g_o; rotation = sum (tau + (o - c) x g_o)
    G[3:] += np.cross(b.origins.astype(np.float64) - c, tr["g_o"]).sum(0)
    eps = 2.0 ** -12 / np.abs(G).max()
    w = eps * G[3:]
    K = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])
    import scipy.linalg
    E = scipy.linalg.expm(-K)
    o2 = c + (b.origins.astype(np.float64) - c) @ E.T - eps * G[:3]
    d2 = b.dirs.astype(np.float64) @ E.T
    l2 = loss(fc, theta, replace(b, origins=o2.astype(np.float32), dirs=d2.astype(np.float32)))
    predicted = -eps * (G ** 2).sum()
    assert l2 < st["loss"]
    assert abs((l2 - st["loss"]) - predicted) <= 0.15 * abs(predicted), (l2 - st["loss"], predicted)


# ---------------------------------------------------------------- coarse-to-fine pose gradients (reading R26)

def _ray_loss(fc, theta, b, r, xs_coarse, xs_fine, n_coarse, d_sh, t, delta, lam):
    """Ray r's term of L (Eqs. 3, 4, 7 with R rays in the batch) restated through the oracle's public stage functions, with
    the encoding levels l < n_coarse evaluated at xs_coarse and the others at xs_fine, and the SH encoding at d_sh."""
    F = fc.n_features
    n_table, _ = orc.param_count(fc)
    e_c, _, _ = orc.encode(fc, theta, xs_coarse, want_index=False)
    e_f, _, _ = orc.encode(fc, theta, xs_fine, want_index=False)
    e = np.concatenate([e_c[:, :n_coarse * F], e_f[:, n_coarse * F:]], axis=1)
    Y = orc.sh(fc.sh_degree, d_sh[None])[0]
    sig, rgb = [], []
    for i in range(len(e)):
        s_, c_ = orc.field_eval(fc, theta[n_table:], e[i], Y)
        sig.append(s_); rgb.append(c_)
    C, D, _ = orc.composite(np.array(sig), np.array(rgb), t, delta, fc.bg)
    R = b.n_rays
    L_rgb = ((C - b.rgb[r].astype(np.float64)) ** 2).sum() / R
    L_d = (D - float(b.depth[r])) ** 2 / float(b.depth_var[r]) / R
    return L_rgb + lam * L_d


@pytest.mark.parametrize("n_coarse", [1, 2, 3])
def test_masked_pose_gradients_differentiate_the_coarse_levels_only(n_coarse):
    """pose_levels = n: g_o and tau must be the derivative of the loss when ONLY the levels l < n see the moved ray, the
    finer levels keeping the unmoved positions (and the SH encoding seeing the rotated direction in full).  Checked by
    central differences of a per-ray loss rebuilt from orc.encode / field_eval / sh / composite with spliced encodings."""
    lam = 0.3
    fc, b, theta = tiny(3, seed=1)
    fc_m = replace(fc, pose_levels=n_coarse)
    assert n_coarse < fc.n_levels
    O = orc.Oracle(fc_m, theta.copy())
    _, tr = O.train_step(b, lam, apply_adam=False, trace=("g_o", "tau", "s_ray", "s_x", "s_t", "s_delta"))
    _, tr_all = orc.Oracle(fc, theta.copy()).train_step(b, lam, apply_adam=False, trace=("g_o", "tau"))
    assert np.abs(tr["g_o"] - tr_all["g_o"]).max() > 1e-3 * np.abs(tr_all["g_o"]).max()      # the mask does something
    ext = float(np.float32(fc.aabb_extent))
    amin = np.asarray(fc.aabb_min, np.float64)
    h = 2.0 ** -11
    ok = 0
    scale_o, scale_t = np.abs(tr["g_o"]).max(), np.abs(tr["tau"]).max()
    for r in range(b.n_rays):
        sel = tr["s_ray"] == r
        if sel.sum() == 0:
            continue
        x0, t, delta = tr["s_x"][sel].astype(np.float64), tr["s_t"][sel], tr["s_delta"][sel]
        o, d = b.origins[r].astype(np.float64), b.dirs[r].astype(np.float64)
        f = lambda xc, dsh: _ray_loss(fc, theta, b, r, xc.astype(np.float32), x0.astype(np.float32), n_coarse, dsh, t, delta, lam)
        for c in range(3):
            step = np.eye(3)[c] * h / ext
            lp, l0, lm = f(x0 + step, d), f(x0, d), f(x0 - step, d)
            if abs(lp - 2 * l0 + lm) / h > 0.02 * scale_o:          # a cell boundary inside the stencil
                continue
            assert abs((lp - lm) / (2 * h) - tr["g_o"][r, c]) <= 2e-2 * scale_o, (r, c)
            ok += 1
        for k in range(3):
            xs = lambda s_: ((o + t[:, None].astype(np.float64) * (rot(k, s_ * h) @ d) - amin) / ext)
            lp, l0, lm = f(xs(+1), rot(k, h) @ d), f(x0, d), f(xs(-1), rot(k, -h) @ d)
            if abs(lp - 2 * l0 + lm) / h > 0.02 * scale_t:
                continue
            assert abs((lp - lm) / (2 * h) - tr["tau"][r, k]) <= 2e-2 * scale_t, (r, k)
            ok += 1
    assert ok >= 3 * b.n_rays                                          # at least half of the 6 R derivatives were testable


def test_pose_levels_zero_and_all_levels_are_the_unmasked_gradients():
    fc, b, theta = tiny(3)
    ref = orc.Oracle(fc, theta.copy()).train_step(b, 0.3, apply_adam=False, trace=("g_o", "tau", "grad"))[1]
    for n in (0, fc.n_levels, fc.n_levels + 5):
        tr = orc.Oracle(replace(fc, pose_levels=n), theta.copy()).train_step(b, 0.3, apply_adam=False, trace=("g_o", "tau", "grad"))[1]
        assert np.array_equal(tr["g_o"], ref["g_o"]) and np.array_equal(tr["tau"], ref["tau"])
    # the mask never touches the parameter gradients
    tr = orc.Oracle(replace(fc, pose_levels=1), theta.copy()).train_step(b, 0.3, apply_adam=False, trace=("grad",))[1]
    assert np.array_equal(tr["grad"], ref["grad"])
