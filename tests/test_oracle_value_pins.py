"""Pins for the oracle's VALUE PATH (S4 interpolation .. S15) against closed forms, invariants,
library routines and brute force.  CPU only."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from tests.helpers import make_oracle, random_batch, tiny_field
from workloads import configs


# ---------------------------------------------------------------- S4 interpolation

def test_partition_of_unity_and_vertex_and_affine():
    fc = configs.config1().field
    res, off = orc.level_table(fc)
    nt, nm = orc.param_count(fc)
    rng = np.random.default_rng(0)
    x = rng.uniform(0, 1, (300, 3)).astype(np.float32)
    # constant tables => constant features (sum of the 8 weights is 1)
    th = np.zeros(nt + nm)
    th[:nt] = 0.37
    e, _, _ = orc.encode(fc, th, x)
    assert np.allclose(e, 0.37, atol=1e-14)
    # affine data on the dense levels is reproduced exactly by trilinear interpolation
    th = rng.normal(size=nt + nm)
    A = np.array([[0.3, -1.1, 0.7], [2.0, 0.25, -0.5]])
    for l in (0, 1):
        N = int(res[l])
        idx = np.arange((N + 1) ** 3)
        v = np.stack([idx % (N + 1), (idx // (N + 1)) % (N + 1), idx // (N + 1) ** 2], 1) / N
        for f in range(2):
            th[(int(off[l]) + idx) * 2 + f] = v @ A[f] + 0.1 * (f + 1)
    e, _, _ = orc.encode(fc, th, x)
    for l in (0, 1):
        for f in range(2):
            assert np.allclose(e[:, 2 * l + f], x.astype(np.float64) @ A[f] + 0.1 * (f + 1), atol=1e-6)
    # a point on a vertex returns that vertex's entry
    N = int(res[1])
    v = np.array([[3, 5, 2]])
    e, slots, _ = orc.encode(fc, th, (v / N).astype(np.float32))
    slot = 3 + (N + 1) * (5 + (N + 1) * 2)
    assert np.allclose(e[0, 2:4], th[(int(off[1]) + slot) * 2:(int(off[1]) + slot) * 2 + 2], atol=1e-14)


def test_encoding_continuous_across_cell_faces():
    fc = configs.FieldConfig(n_levels=4, log2_table_size=10, n_min=4, n_max=32)
    nt, nm = orc.param_count(fc)
    th = np.random.default_rng(1).normal(size=nt + nm)
    for N in (4, 8, 16, 32):
        face = np.float32(3.0 / N)
        lo = np.nextafter(face, np.float32(0))
        x = np.array([[lo, 0.3, 0.6], [face, 0.3, 0.6]], np.float32)
        e, _, _ = orc.encode(fc, th, x)
        assert np.allclose(e[0], e[1], atol=1e-4)


# ---------------------------------------------------------------- S6 spherical harmonics

def test_sh_constants_and_l1_band():
    d = np.array([[0.36, -0.48, 0.8]])
    Y = orc.sh(4, d)[0]
    assert np.isclose(Y[0], 1 / (2 * np.sqrt(np.pi)), atol=1e-15)
    k = np.sqrt(3 / (4 * np.pi))
    assert np.allclose(Y[1:4], k * np.array([d[0, 1], d[0, 2], d[0, 0]]), atol=1e-14)   # (y, z, x)


def test_sh_addition_theorem_and_orthonormality():
    rng = np.random.default_rng(2)
    d = configs.unit_dirs(rng, 50)
    n = 5
    Y = orc.sh(n, d)
    for l in range(n):
        assert np.allclose((Y[:, l * l:(l + 1) ** 2] ** 2).sum(1), (2 * l + 1) / (4 * np.pi), atol=1e-13)
    # Gauss-Legendre in z times uniform phi integrates products of degree <= 2(n-1) exactly
    z, wz = np.polynomial.legendre.leggauss(16)
    phi = (np.arange(32) + 0.5) * 2 * np.pi / 32
    zz, pp = np.meshgrid(z, phi, indexing="ij")
    s = np.sqrt(1 - zz ** 2)
    dirs = np.stack([s * np.cos(pp), s * np.sin(pp), zz], -1).reshape(-1, 3)
    wq = np.repeat(wz, 32) * (2 * np.pi / 32)
    Yq = orc.sh(n, dirs)
    gram = (Yq * wq[:, None]).T @ Yq
    assert np.allclose(gram, np.eye(n * n), atol=1e-12)


def test_sh_matches_scipy_complex_harmonics():
    scipy_special = pytest.importorskip("scipy.special")
    rng = np.random.default_rng(3)
    d = configs.unit_dirs(rng, 20)
    theta = np.arccos(d[:, 2])
    phi = np.arctan2(d[:, 1], d[:, 0])
    Y = orc.sh(4, d)
    for l in range(4):
        for m in range(0, l + 1):
            if hasattr(scipy_special, "sph_harm_y"):
                c = scipy_special.sph_harm_y(l, m, theta, phi)
            else:
                c = scipy_special.sph_harm(m, l, phi, theta)
            if m == 0:
                assert np.allclose(Y[:, l * l + l], c.real, atol=1e-12)
            else:   # scipy carries the Condon-Shortley phase (-1)^m; the spec does not
                assert np.allclose(Y[:, l * l + l + m], (-1) ** m * np.sqrt(2) * c.real, atol=1e-12)
                assert np.allclose(Y[:, l * l + l - m], (-1) ** m * np.sqrt(2) * c.imag, atol=1e-12)


# ---------------------------------------------------------------- S5 / S7 MLPs

def _split_mlp(fc, theta_mlp):
    out, o = {}, 0
    for name, n_out, n_in in orc.mlp_shapes(fc):
        out[name] = theta_mlp[o:o + n_out * n_in].reshape(n_out, n_in)
        o += n_out * n_in
    return out


@pytest.mark.parametrize("fc", [configs.config1().field, configs.FieldConfig()])
def test_mlp_reduces_to_matmul(fc):
    nt, nm = orc.param_count(fc)
    rng = np.random.default_rng(4)
    thm = rng.normal(scale=0.3, size=nm)
    W = _split_mlp(fc, thm)
    for _ in range(5):
        e = rng.normal(size=fc.n_levels * fc.n_features)
        Y = rng.normal(size=fc.sh_degree ** 2)
        sig, rgb = orc.field_eval(fc, thm, e, Y)
        g = W["W_d2"] @ np.maximum(W["W_d1"] @ e, 0)
        assert np.isclose(sig, np.exp(np.clip(g[0], -15, 15)), rtol=1e-13)
        h = np.maximum(W["W_c1"] @ np.concatenate([g[fc.geo_offset:fc.geo_offset + fc.geo_count], Y]), 0)
        if "W_c2" in W:
            h = np.maximum(W["W_c2"] @ h, 0)
        assert np.allclose(rgb, 1 / (1 + np.exp(-(W["W_c3"] @ h))), rtol=1e-13)


def test_mlp_identity_passthrough_and_clamp():
    fc = tiny_field(n_levels=4, n_features=2, density_hidden=8, density_out=8, geo_offset=0,
                    geo_count=8, sh_degree=1, color_hidden=9, color_hidden_layers=1)
    shapes = orc.mlp_shapes(fc)
    mats = {n: np.zeros((o, i)) for n, o, i in shapes}
    mats["W_d1"][:] = np.eye(8)
    mats["W_d2"][:] = np.eye(8)
    mats["W_c1"][:] = np.eye(9)
    mats["W_c3"][:, :3] = np.eye(3)
    thm = np.concatenate([mats[n].ravel() for n, _, _ in shapes])
    e = np.array([0.5, 1.5, 2.5, 0.1, 0.2, 0.3, 0.4, 0.6])
    sig, rgb = orc.field_eval(fc, thm, e, np.array([0.0]))
    assert np.isclose(sig, np.exp(0.5)) and np.allclose(rgb, 1 / (1 + np.exp(-e[:3])))
    e[0] = 40.0
    assert np.isclose(orc.field_eval(fc, thm, e, np.array([0.0]))[0], np.exp(15.0))


# ---------------------------------------------------------------- S8 compositing closed forms

def test_constant_density_slab_and_invariants():
    w = configs.config1()
    m = orc.march(w.field, None, w.batches[0], jitter=True, step=1)
    K = 32
    t, d = m["s_t"][:K], m["s_delta"][:K]
    sigma = 2.3
    C, D, O = orc.composite(np.full(K, sigma), np.full((K, 3), 0.25), t, d)
    length = float(np.sum(d.astype(np.float64)))
    assert np.isclose(O, 1 - np.exp(-sigma * length), atol=1e-12)        # telescoping, Eqs. 5-6
    assert np.isclose(O, 1 - np.exp(-sigma * (1.8 - float(t[0]))), atol=1e-5)
    assert np.allclose(C, 0.25 * O, atol=1e-12)
    rng = np.random.default_rng(5)
    sig = rng.uniform(0, 30, K)
    C, D, O = orc.composite(sig, rng.uniform(0, 1, (K, 3)), t, d, bg=(0.2, 0.4, 0.6))
    assert 0 <= O <= 1 and t[0] * O - 1e-12 <= D <= t[-1] * O + 1e-12
    # sigma == 0 => background, zero depth
    C, D, O = orc.composite(np.zeros(K), np.ones((K, 3)), t, d, bg=(0.2, 0.4, 0.6))
    assert np.allclose(C, [0.2, 0.4, 0.6], atol=1e-7) and D == 0 and O == 0
    # no samples
    C, D, O = orc.composite(np.zeros(0), np.zeros((0, 3)), t[:0], d[:0], bg=(0.2, 0.4, 0.6))
    assert np.allclose(C, [0.2, 0.4, 0.6], atol=1e-7) and D == 0 and O == 0


def test_opaque_shell_depth_equals_distance():
    K = 32
    t = np.linspace(0.1, 1.7, K).astype(np.float32)
    d = np.full(K, 0.05, np.float32)
    sig = np.zeros(K)
    sig[11] = 1e6
    rgb = np.random.default_rng(6).uniform(0, 1, (K, 3))
    C, D, O = orc.composite(sig, rgb, t, d)
    assert np.isclose(D, float(t[11]), atol=1e-12) and np.allclose(C, rgb[11], atol=1e-12) and np.isclose(O, 1)


def test_composite_matches_eq5_eq6_written_with_cumsum():
    rng = np.random.default_rng(7)
    K = 40
    sig = rng.uniform(0, 20, K)
    rgb = rng.uniform(0, 1, (K, 3))
    t = np.sort(rng.uniform(0.1, 3, K)).astype(np.float32)
    d = rng.uniform(0.01, 0.1, K).astype(np.float32)
    a = sig * d.astype(np.float64)
    T = np.exp(-np.concatenate([[0], np.cumsum(a)[:-1]]))                 # Eq. 6
    wgt = T * (1 - np.exp(-a))                                             # Eq. 5 weights
    C, D, O = orc.composite(sig, rgb, t, d, bg=(0.1, 0.2, 0.3))
    Tend = np.exp(-a.sum())
    assert np.allclose(C, wgt @ rgb + Tend * np.float32([0.1, 0.2, 0.3]), atol=1e-12)
    assert np.isclose(D, wgt @ t.astype(np.float64), atol=1e-12) and np.isclose(O, wgt.sum(), atol=1e-12)


# ---------------------------------------------------------------- S9 loss special cases

def _loss(O, b, lam):
    return O.train_step(b, lam, apply_adam=False, trace=("grad", "C", "D_hat"))


def test_loss_special_cases():
    fc = tiny_field()
    b = random_batch(1, 8, 8)
    O = make_oracle(fc, 0, table_scale=0.5)
    s1, t1 = _loss(O, b, 1.0)
    s0, t0 = _loss(O, b, 0.0)
    s2, t2 = _loss(O, b, 2.0)
    R = 8
    assert np.isclose(s0["loss"], s0["loss_rgb"])
    assert np.isclose(s0["loss_rgb"], ((t0["C"] - b.rgb) ** 2).sum() / R, rtol=1e-12)       # Eq. 7
    assert np.isclose(s1["loss_depth"], (((t1["D_hat"] - b.depth) ** 2) / b.depth_var.astype(np.float64)).sum() / R, rtol=1e-12)  # Eq. 4
    assert np.isclose(s2["loss"] - s1["loss"], s1["loss"] - s0["loss"], rtol=1e-10)          # linear in lambda (Eq. 3)
    assert np.allclose(t2["grad"] - t1["grad"], t1["grad"] - t0["grad"], atol=1e-13)
    # Sigma_D == 1 => plain L2 depth loss
    b1 = replace(b, depth_var=np.ones(8, np.float32))
    s, t = _loss(O, b1, 1.0)
    assert np.isclose(s["loss_depth"], ((t["D_hat"] - b.depth) ** 2).sum() / R, rtol=1e-12)
    # Sigma_D -> inf, invalid depth or variance => no depth term, gradients equal the lambda=0 ones
    for var, dep in ((np.full(8, np.inf), b.depth), (np.full(8, 1e30), b.depth), (b.depth_var, np.zeros(8)),
                     (np.zeros(8), b.depth), (np.full(8, -1.0), b.depth)):
        bb = replace(b, depth_var=var.astype(np.float32), depth=np.asarray(dep, np.float32))
        s, t = _loss(O, bb, 1.0)
        assert s["loss_depth"] < 1e-25
        assert np.allclose(t["grad"], t0["grad"], atol=1e-25 + 1e-20)


def test_empty_occupancy_loss_is_background_loss():
    fc = tiny_field(bg=(0.3, 0.5, 0.7))
    b = random_batch(2, 8, 8)
    O = make_oracle(fc)
    O.set_occupancy(np.zeros(8 ** 3 // 8, np.uint8))
    s, t = O.train_step(b, 0.7, apply_adam=False, trace=("grad", "touched"))
    want = (((np.float32([0.3, 0.5, 0.7]) - b.rgb) ** 2).sum() + 0.7 * (b.depth.astype(np.float64) ** 2 / b.depth_var).sum()) / 8
    assert s["n_samples"] == 0 and np.isclose(s["loss"], want, rtol=1e-12)
    assert not t["grad"].any() and not t["touched"].any()


# ---------------------------------------------------------------- S10-S12 gradients

def _total_loss(fc, theta, bits, b, lam):
    O = orc.Oracle(fc, theta)
    O.theta = theta.copy()
    O.set_occupancy(bits)
    return O.train_step(b, lam, apply_adam=False)[0]["loss"]


@pytest.mark.parametrize("layers,bg", [(1, (0, 0, 0)), (2, (0.2, 0.5, 0.9))])
def test_gradients_central_finite_differences(layers, bg):
    """Every MLP weight and every touched table entry of a tiny field (8 rays x 8 samples)."""
    fc = tiny_field(color_hidden_layers=layers, bg=bg, geo_offset=1 if layers == 2 else 0,
                    geo_count=15 if layers == 2 else 16)
    b = random_batch(3, 8, 8)
    O = make_oracle(fc, 1, table_scale=0.3)
    theta = O.theta.copy()
    theta[O.n_table:] *= 1.5
    O.theta = theta.copy()
    s, t = O.train_step(b, 0.6, apply_adam=False, trace=("grad", "touched"))
    g = t["grad"]
    touched_params = np.repeat(t["touched"].astype(bool), fc.n_features)
    assert not g[:O.n_table][~touched_params].any()            # untouched entries: exactly zero
    idx = np.concatenate([np.nonzero(touched_params)[0], O.n_table + np.arange(O.n_mlp)])
    bad, checked = 0, 0
    for i in idx:
        h = 1e-6 * max(1.0, abs(theta[i]))
        tp, tm = theta.copy(), theta.copy()
        tp[i] += h
        tm[i] -= h
        lp, lm = _total_loss(fc, tp, None, b, 0.6), _total_loss(fc, tm, None, b, 0.6)
        fd = (lp - lm) / (2 * h)
        # second difference flags a ReLU kink inside the stencil: skip those parameters
        curv = abs(lp - 2 * s["loss"] + lm) / h
        if curv > 1e-4 * max(abs(fd), 1e-6) + 1e-9:
            continue
        checked += 1
        if abs(fd - g[i]) > 1e-6 * max(abs(fd), abs(g[i])) + 2e-9:
            bad += 1
    assert checked > 0.8 * len(idx) and bad == 0, (checked, len(idx), bad)


def _torch_restatement(fc, O, b, lam, tr):
    """Independent float64 autograd restatement: gathers fed with the oracle's integer indices and
    fp32 fractions, matmuls, cumsum; everything else re-derived from Eqs. 3-7."""
    dt = torch.float64
    theta = torch.tensor(O.theta, dtype=dt, requires_grad=True)
    L, F = fc.n_levels, fc.n_features
    nt = O.n_table
    tab = theta[:nt].reshape(-1, F)
    slots = torch.tensor(tr["slots"].astype(np.int64))                     # [S,L,8]
    w = torch.tensor(tr["w"].astype(np.float64))                           # [S,L,3]
    off = torch.tensor(O.offset[:-1].astype(np.int64))
    S = slots.shape[0]
    feats = []
    for l in range(L):
        acc = 0
        for corner in range(8):
            om = 1
            for c in range(3):
                om = om * (w[:, l, c] if (corner >> c) & 1 else 1 - w[:, l, c])
            acc = acc + om[:, None] * tab[off[l] + slots[:, l, corner]]
        feats.append(acc)
    e = torch.cat(feats, 1)
    mats, o = {}, nt
    for name, n_out, n_in in orc.mlp_shapes(fc):
        mats[name] = theta[o:o + n_out * n_in].reshape(n_out, n_in)
        o += n_out * n_in
    g = torch.relu(e @ mats["W_d1"].T) @ mats["W_d2"].T
    sigma = torch.exp(torch.clamp(g[:, 0], -15, 15))
    ray = torch.tensor(tr["s_ray"].astype(np.int64))
    Y = torch.tensor(orc.sh(fc.sh_degree, b.dirs.astype(np.float64)))[ray]
    h = torch.relu(torch.cat([g[:, fc.geo_offset:fc.geo_offset + fc.geo_count], Y], 1) @ mats["W_c1"].T)
    if "W_c2" in mats:
        h = torch.relu(h @ mats["W_c2"].T)
    rgb = torch.sigmoid(h @ mats["W_c3"].T)
    a = sigma * torch.tensor(tr["s_delta"].astype(np.float64))
    R = b.n_rays
    # exclusive per-ray cumulative sum of a via a global cumsum minus the value at the ray start
    cs = torch.cumsum(a, 0)
    excl = cs - a
    offs = torch.tensor(tr["offsets"].astype(np.int64))
    start = torch.where(offs[:-1] < S, excl[torch.clamp(offs[:-1], max=max(S - 1, 0))], torch.zeros(R, dtype=dt))
    T = torch.exp(-(excl - start[ray]))
    wgt = T * (1 - torch.exp(-a))
    C = torch.zeros(R, 3, dtype=dt).index_add(0, ray, wgt[:, None] * rgb)
    D = torch.zeros(R, dtype=dt).index_add(0, ray, wgt * torch.tensor(tr["s_t"].astype(np.float64)))
    Osum = torch.zeros(R, dtype=dt).index_add(0, ray, wgt)
    C = C + (1 - Osum)[:, None] * torch.tensor(np.float32(fc.bg).astype(np.float64))
    dep = torch.tensor(b.depth.astype(np.float64))
    var = torch.tensor(b.depth_var.astype(np.float64))
    mask = (dep > 0) & (var > 0) & torch.isfinite(var)
    Lrgb = ((C - torch.tensor(b.rgb.astype(np.float64))) ** 2).sum() / R
    Ld = (torch.where(mask, (D - dep) ** 2 / torch.where(mask, var, torch.ones_like(var)), torch.zeros_like(D))).sum() / R
    loss = Lrgb + lam * Ld
    loss.backward()
    return loss.item(), theta.grad.numpy(), C.detach().numpy(), D.detach().numpy()


@pytest.mark.parametrize("which", ["cfg1", "cfg1b", "cfg2small"])
def test_gradients_match_torch_autograd_restatement(which):
    if which == "cfg2small":
        w = configs.config2(R=512, K=64, occ_res=32, field_overrides=dict(log2_table_size=14, n_max=256, bg=(0.1, 0.2, 0.3)))
    else:
        w = configs.config1(variant_b=(which == "cfg1b"))
    fc, b = w.field, w.batches[0]
    O = make_oracle(fc, 3, table_scale=0.2)
    O.set_occupancy(w.bits)
    s, tr = O.train_step(b, w.lambda_d, apply_adam=False,
                         trace=("grad", "slots", "w", "s_ray", "s_t", "s_delta", "offsets", "C", "D_hat", "touched"))
    loss, grad, C, D = _torch_restatement(fc, O, b, w.lambda_d, tr)
    assert np.isclose(loss, s["loss"], rtol=1e-12)
    assert np.allclose(C, tr["C"], atol=1e-12) and np.allclose(D, tr["D_hat"], atol=1e-12)
    scale = np.abs(grad).max()
    assert np.abs(grad - tr["grad"]).max() <= 1e-10 * scale
    # structural touched set == set of referenced slots
    ref = np.zeros(O.n_entries, bool)
    ref[(O.offset[:-1].astype(np.int64)[None, :, None] + tr["slots"]).reshape(-1)] = True
    assert np.array_equal(ref, tr["touched"].astype(bool))


# ---------------------------------------------------------------- S13 Adam

def test_adam_matches_torch_optim_and_closed_form():
    rng = np.random.default_rng(8)
    n = 257
    th0 = rng.normal(size=n)
    theta, m, v = th0.copy(), np.zeros(n), np.zeros(n)
    p = torch.tensor(th0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([p], lr=1e-2, betas=(0.9, 0.99), eps=1e-15, weight_decay=0)
    for step in range(1, 8):
        g = rng.normal(size=n) * 10.0 ** rng.integers(-8, 2, n)
        orc.adam(theta, m, v, g, step, 1e-2, 0.9, 0.99, 1e-15)
        p.grad = torch.tensor(g)
        opt.step()
        assert np.allclose(theta, p.detach().numpy(), rtol=0, atol=1e-12)
        if step == 1:   # closed form at step 1: -lr g/(|g| + eps)
            assert np.allclose(theta - th0, -1e-2 * g / (np.abs(g) + 1e-15), atol=1e-15)


def test_sparse_adam_leaves_untouched_entries_bit_unchanged_and_dense_mode_is_textbook():
    w = configs.config1(variant_b=True)
    fc, b = w.field, w.batches[0]
    O = make_oracle(fc, 4, table_scale=0.3)
    O.m[:] = 0.01
    O.v[:] = 1e-4
    th0, m0, v0 = O.theta.copy(), O.m.copy(), O.v.copy()
    s, tr = O.train_step(b, 0.1, trace=("grad", "touched"))
    tp = np.repeat(tr["touched"].astype(bool), fc.n_features)
    assert 0 < tp.sum() < tp.size
    nt = O.n_table
    for a, a0 in ((O.theta, th0), (O.m, m0), (O.v, v0)):
        assert np.array_equal(a[:nt][~tp], a0[:nt][~tp])
        assert not np.any(a[:nt][tp] == a0[:nt][tp])
        assert not np.any(a[nt:] == a0[nt:])
    assert O.step == 1 and s["step"] == 1
    # dense mode: every parameter gets the textbook update with g = 0 where untouched
    Od = make_oracle(replace(fc, sparse_table_adam=0), 4, table_scale=0.3)
    Od.m[:] = 0.01
    Od.v[:] = 1e-4
    Od.train_step(b, 0.1)
    p = torch.tensor(th0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([p], lr=float(np.float32(1e-2)), betas=(float(np.float32(0.9)), float(np.float32(0.99))),
                           eps=float(np.float32(1e-15)))
    p.grad = torch.tensor(tr["grad"])
    opt.state[p] = dict(step=torch.tensor(0.0), exp_avg=torch.tensor(m0.copy()), exp_avg_sq=torch.tensor(v0.copy()))
    opt.step()
    assert np.allclose(Od.theta, p.detach().numpy(), atol=1e-12)
    assert np.array_equal(Od.theta[:nt][tp], O.theta[:nt][tp])


# ---------------------------------------------------------------- S14 / S15

def test_occupancy_from_field_zero_tables_and_set_roundtrip():
    fc = tiny_field(occ_res=8, occ_sigma_threshold=0.5)
    O = make_oracle(fc)
    O.theta[:O.n_table] = 0.0                       # e == 0 => g == 0 => sigma == exp(0) == 1
    bits, sig = O.occupancy_from_field(want_sigma=True)
    assert np.all(sig == 1.0) and np.all(bits == 0xFF)
    O2 = make_oracle(replace(fc, occ_sigma_threshold=1.0))
    O2.theta[:O2.n_table] = 0.0
    assert not O2.occupancy_from_field().any()      # strict '>' threshold
    # general field: bit i <=> sigma(cell centre i) > thr, sigma from encode + field_eval
    O3 = make_oracle(replace(fc, occ_sigma_threshold=1.0), 5, table_scale=0.5)
    bits, sig = O3.occupancy_from_field(want_sigma=True)
    G = 8
    idx = np.arange(G ** 3)
    x = np.stack([(idx % G + 0.5) / G, ((idx // G) % G + 0.5) / G, (idx // G ** 2 + 0.5) / G], 1).astype(np.float32)
    e, _, _ = orc.encode(fc, O3.theta, x, want_index=False)
    s_ref = np.array([orc.field_eval(fc, O3.theta[O3.n_table:], e[i], np.zeros(4))[0] for i in idx])
    assert np.allclose(sig, s_ref, rtol=1e-13)
    assert np.array_equal(np.unpackbits(bits, bitorder="little").astype(bool), sig > 1.0)
    assert 0 < (sig > 1.0).sum() < G ** 3


def test_render_cut_zero_equals_training_forward_and_cut_bound():
    w = configs.config1()
    fc, b = replace(w.field, bg=(0.2, 0.3, 0.4)), w.batches[0]
    O = make_oracle(fc, 6, table_scale=0.5)
    O.theta[O.n_table:] *= 3.0                      # make some rays opaque
    s, tr = O.train_step(b, 0.0, jitter=False, apply_adam=False, trace=("C", "D_hat", "O"))
    rgb, dep, opa, n = O.render(b, cut=0.0)
    assert n == s["n_samples"]
    assert np.allclose(rgb, tr["C"], atol=1e-13) and np.allclose(dep, tr["D_hat"], atol=1e-13) and np.allclose(opa, tr["O"], atol=1e-13)
    cut = 1e-2
    rgb2, dep2, opa2, n2 = O.render(b, cut=cut)
    assert n2 < n                                   # termination actually happens
    assert np.abs(rgb2 - rgb).max() <= cut * 1.4 + 1e-12
    assert np.abs(dep2 - dep).max() <= cut * b.t_max + 1e-12
    assert np.all(opa2 <= opa + 1e-12)
