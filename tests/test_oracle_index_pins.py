"""Pins for the oracle's INDEX PATH (S0-S4 integers and fp32 quantities) against what the
mathematics fixes, not against the oracle itself.  CPU only."""
from dataclasses import replace
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as orc
from tests.helpers import make_oracle, random_batch, tiny_field
from workloads import configs


def exact_resolution(n_min, n_max, L, l):
    """floor(n_min * (n_max/n_min)^(l/(L-1))) in exact integer arithmetic:
    the largest n with n^(L-1) * n_min^l <= n_min^(L-1) * n_max^l."""
    if L == 1 or l == 0:
        return n_min
    rhs = n_min ** (L - 1) * n_max ** l
    lo, hi = n_min, n_max
    while lo < hi:
        mid = (lo + hi + 1) // 2
        if mid ** (L - 1) * n_min ** l <= rhs:
            lo = mid
        else:
            hi = mid - 1
    return lo


GOLDEN = {}
with open(__file__.replace("test_oracle_index_pins.py", "golden/level_tables.txt")) as fh:
    for line in fh:
        if line.startswith("#") or not line.strip():
            continue
        key, vals = line.split(":")
        GOLDEN[key.strip()] = [int(v) for v in vals.split()]


@pytest.mark.parametrize("name,L,F,log2T,n_min,n_max", [
    ("cfg1", 4, 2, 10, 4, 32), ("cfg2", 16, 2, 19, 16, 2048), ("cfg4", 16, 4, 22, 16, 8192)])
def test_level_tables_exact_and_golden(name, L, F, log2T, n_min, n_max):
    fc = configs.FieldConfig(n_levels=L, n_features=F, log2_table_size=log2T, n_min=n_min, n_max=n_max)
    res, off = orc.level_table(fc)
    # exact big-integer evaluation of the geometric progression (catches the 127/1023/8191 trap)
    assert [int(r) for r in res] == [exact_resolution(n_min, n_max, L, l) for l in range(L)]
    assert [int(r) for r in res] == GOLDEN[name + ".res"]       # SURVEY.md section 8 size table
    T = 1 << log2T
    E = [min((n + 1) ** 3, T) for n in GOLDEN[name + ".res"]]
    assert [int(o) for o in off] == [sum(E[:i]) for i in range(L + 1)]
    assert int(off[-1]) == GOLDEN[name + ".entries"][0]
    nt, _ = orc.param_count(fc)
    assert nt == F * GOLDEN[name + ".entries"][0]


def test_exact_power_levels_cfg4():
    fc = configs.FieldConfig(n_levels=16, n_features=4, log2_table_size=22, n_min=16, n_max=8192)
    res, _ = orc.level_table(fc)
    assert (res[5], res[10], res[15]) == (128, 1024, 8192)      # 16 * 512^(l/15)


def test_mlp_param_counts():
    # MLP weight counts 752 / 9344 / 11392
    assert orc.param_count(configs.config1().field)[1] == 752
    assert orc.param_count(configs.FieldConfig())[1] == 9344
    assert orc.param_count(configs.FieldConfig(n_features=4, log2_table_size=22, n_max=8192))[1] == 11392


def test_jitter_stream_uniform_and_distinct():
    n = 1 << 16
    hs = np.array([orc.hash32(5, 1 + (i >> 14), (i >> 7) & 127, i & 127) for i in range(n)], np.uint64)
    assert len(np.unique(hs)) > n - 8                    # birthday bound: ~0.5 collisions expected
    u = (hs >> np.uint64(8)).astype(np.float64) / 2 ** 24
    hist, _ = np.histogram(u, bins=64, range=(0, 1))
    chi2 = ((hist - n / 64) ** 2 / (n / 64)).sum()
    assert chi2 < 120                                     # 63 dof: P(chi2 > 120) ~ 1e-5
    # neighbouring counters decorrelate
    a = np.array([orc.jitter_u(5, 1, 0, k) for k in range(4096)])
    assert abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 0.06
    assert orc.jitter_u(5, 1, 0, 0) != orc.jitter_u(5, 2, 0, 0) != orc.jitter_u(6, 1, 0, 0)
    assert 0.0 <= a.min() and a.max() < 1.0


def test_march_t_in_bin_and_delta_telescopes():
    w = configs.config1()
    b = w.batches[0]
    m = orc.march(w.field, None, b, jitter=True, step=1)
    K, R = b.n_candidates, b.n_rays
    assert m["S"] == R * K and np.all(m["counts"] == K)       # full occupancy, AABB contains all
    assert np.array_equal(m["offsets"], np.arange(R + 1) * K)
    assert np.array_equal(m["s_ray"], np.repeat(np.arange(R), K))
    assert np.array_equal(m["s_k"], np.tile(np.arange(K), R))
    dt = (b.t_max - b.t_min) / K
    t = m["s_t"].reshape(R, K).astype(np.float64)
    k = np.arange(K)
    assert np.all(t >= b.t_min + k * dt - 1e-6) and np.all(t <= b.t_min + (k + 1) * dt + 1e-6)
    d = m["s_delta"].reshape(R, K).astype(np.float64)
    # Eq. 5: delta_i = d_{i+1} - d_i on the candidate lattice; the last runs to t_max
    assert np.allclose(d[:, :-1], t[:, 1:] - t[:, :-1], atol=2e-7)
    assert np.allclose(d.sum(1), b.t_max - t[:, 0], atol=1e-5)
    # x = (o + t d - aabb_min)/extent
    x = m["s_x"].reshape(R, K, 3).astype(np.float64)
    p = b.origins[:, None, :].astype(np.float64) + t[..., None] * b.dirs[:, None, :].astype(np.float64)
    assert np.allclose(x, (p + 2.0) / 5.0, atol=1e-6)
    # no jitter: u == 0.5 exactly
    m0 = orc.march(w.field, None, b, jitter=False)
    assert np.allclose(m0["s_t"].reshape(R, K)[0], b.t_min + (k + 0.5) * dt, atol=1e-6)


def test_march_halfspace_closed_form_and_empty():
    G = 16
    fc = tiny_field(aabb_min=(0, 0, 0), aabb_extent=1.0, occ_res=G)
    cells = np.arange(G ** 3)
    mask = (cells % G) < G // 2                               # gx < G/2  <=>  x < 0.5
    bits = np.packbits(mask.astype(np.uint8), bitorder="little")
    K = 64
    o = np.array([[0.1, 0.3, 0.7], [0.9, 0.2, 0.2], [0.25, 0.5, 0.5], [0.6, 0.5, 0.5]], np.float32)
    d = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, 0, 1]], np.float32)
    b = configs.RayBatch(o, d, t_min=0.0, t_max=1.0, n_candidates=K)
    m = orc.march(fc, bits, b, jitter=False)
    tk = (np.arange(K) + 0.5) / K
    want = [np.sum(0.1 + tk < 0.5), np.sum((0.9 - tk < 0.5) & (0.9 - tk >= 0)),
            np.sum(0.5 + tk < 1.0), 0]
    assert list(m["counts"]) == want
    assert m["S"] == sum(want) and np.array_equal(m["offsets"], np.concatenate([[0], np.cumsum(want)]))
    # (ray, k) order and k values of ray 1: the candidates with 0 <= x < 0.5
    k1 = m["s_k"][m["s_ray"] == 1]
    assert np.array_equal(k1, np.nonzero((0.9 - tk < 0.5) & (0.9 - tk >= 0))[0])
    empty = orc.march(fc, np.zeros(G ** 3 // 8, np.uint8), b, jitter=False)
    assert empty["S"] == 0 and not empty["counts"].any()


def test_march_sphere_bits_agree_with_geometry():
    """Every live sample's fp32 x lies in a set cell, and every in-cube candidate in a set cell
    is live (checked from the returned t via the sphere geometry, away from cell boundaries)."""
    w = configs.config2(R=256, K=64, occ_res=32)
    b = w.batches[0]
    m = orc.march(w.field, w.bits, b, jitter=True, step=3)
    G = 32
    x = m["s_x"]
    assert np.all((x >= 0) & (x < 1))
    g = np.minimum((x * G).astype(np.int64), G - 1)
    cell = g[:, 0] + G * (g[:, 1] + G * g[:, 2])
    mask = np.unpackbits(w.bits, bitorder="little")
    assert np.all(mask[cell] == 1)
    assert m["S"] == m["counts"].sum() and np.all(np.diff(m["offsets"]) == m["counts"])
    # order: (ray, k) lexicographic, strictly increasing
    key = m["s_ray"].astype(np.int64) * 64 + m["s_k"]
    assert np.all(np.diff(key) > 0)
    # completeness via a full-occupancy march of the same batch
    full = orc.march(w.field, None, b, jitter=True, step=3)
    gf = np.minimum((full["s_x"] * G).astype(np.int64), G - 1)
    live = mask[gf[:, 0] + G * (gf[:, 1] + G * gf[:, 2])] == 1
    assert live.sum() == m["S"]
    assert np.array_equal(full["s_t"][live], m["s_t"])


def test_dense_slots_are_a_bijection_and_hashed_slots_in_range():
    w = configs.config1()
    fc = w.field
    res, off = orc.level_table(fc)
    th = np.zeros(orc.param_count(fc)[0] + orc.param_count(fc)[1])
    for l in (0, 1):                                           # dense: 125 and 729 entries
        N = int(res[l])
        v = np.stack(np.meshgrid(np.arange(N + 1), np.arange(N + 1), np.arange(N + 1), indexing="ij"), -1).reshape(-1, 3)
        interior = v[(v < N).all(1)]
        x = (interior / N).astype(np.float32)                  # exact: N is a power of two
        _, slots, wts = orc.encode(fc, th, x)
        assert np.all(wts[:, l] == 0)
        seen = set()
        for corner in range(8):
            vv = interior + [(corner >> 0) & 1, (corner >> 1) & 1, (corner >> 2) & 1]
            want = vv[:, 0] + (N + 1) * (vv[:, 1] + (N + 1) * vv[:, 2])
            assert np.array_equal(slots[:, l, corner], want)
            seen |= set(want.tolist())
        assert seen == set(range((N + 1) ** 3))
    rng = np.random.default_rng(0)
    _, slots, _ = orc.encode(fc, th, rng.uniform(0, 1, (2000, 3)).astype(np.float32))
    assert slots[:, 2:].max() < 1024 and slots[:, 2:].min() >= 0


def test_hash_constants_hand_computed():
    """Hashed level: vertex (0,0,0)->0, (1,0,0)->1, (0,1,0)->2654435761 mod T, (0,0,1)->805459861 mod T,
    and a general vertex against Python integers."""
    fc = configs.FieldConfig(n_levels=2, log2_table_size=10, n_min=16, n_max=64)   # level 1 hashed
    res, _ = orc.level_table(fc)
    N, T = int(res[1]), 1024
    th = np.zeros(sum(orc.param_count(fc)))
    _, slots, _ = orc.encode(fc, th, np.zeros((1, 3), np.float32))
    s = slots[0, 1]
    assert s[0] == 0 and s[1] == 1 and s[2] == 2654435761 % T and s[4] == 805459861 % T
    assert s[7] == (1 ^ 2654435761 ^ 805459861) % T
    v = (37, 51, 22)
    x = (np.array(v) / N).astype(np.float32)[None]             # N = 64
    _, slots, _ = orc.encode(fc, th, x)
    for corner in range(8):
        vv = [v[c] + ((corner >> c) & 1) for c in range(3)]
        want = ((vv[0] * 1) & 0xFFFFFFFF) ^ ((vv[1] * 2654435761) & 0xFFFFFFFF) ^ ((vv[2] * 805459861) & 0xFFFFFFFF)
        assert slots[0, 1, corner] == want % T


def test_fraction_w_is_exact_remainder():
    fc = configs.FieldConfig()
    res, _ = orc.level_table(fc)
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 1, (500, 3)).astype(np.float32)
    _, _, w = orc.encode(fc, np.zeros(sum(orc.param_count(fc))), x)
    for l, N in enumerate(res):
        pos = (x * np.float32(N)).astype(np.float32)
        c0 = np.minimum(np.floor(pos), N - 1)
        assert np.array_equal(w[:, l], (pos.astype(np.float64) - c0).astype(np.float32))
        assert np.all((w[:, l] >= 0) & (w[:, l] <= 1))
