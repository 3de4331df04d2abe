"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO arithmetic of the method: it only produces arrays (rays, targets, depth,
variance, occupancy bits, initial parameters) that are handed, as arrays, to both the oracle
and the CUDA path.  It imports neither.  Everything is generated on the host in float64 with
numpy.random.Generator(PCG64(seed)) and cast to fp32.

The paper evaluates on Replica and Cube-Diorama; neither is available, so
these generators stand in for them with the benchmark's shapes (1200x680 pinhole, fx=fy=600,
room-scale scenes, dense noisy depth with per-pixel variance and gross outliers,
PAPER.md:124, 240).
"""
from dataclasses import dataclass, field, replace

import numpy as np

from . import scenes


@dataclass
class FieldConfig:
    aabb_min: tuple = (0.0, 0.0, 0.0)
    aabb_extent: float = 1.0
    n_levels: int = 16
    n_features: int = 2
    log2_table_size: int = 19
    n_min: int = 16
    n_max: int = 2048
    occ_res: int = 128
    density_hidden: int = 64
    density_out: int = 16
    geo_offset: int = 1
    geo_count: int = 15
    sh_degree: int = 4
    color_hidden: int = 64
    color_hidden_layers: int = 2
    mlp_precision: int = 1            # 0 fp32, 1 fp16, 2 bf16 (GPU only; the oracle is float64)
    bg: tuple = (0.0, 0.0, 0.0)
    occ_sigma_threshold: float = 0.01
    lr: float = 1e-2
    beta1: float = 0.9
    beta2: float = 0.99
    eps: float = 1e-15
    sparse_table_adam: int = 1
    seed: int = 0
    max_rays: int = 4096
    max_candidates: int = 128
    occ_cascades: int = 1             # F4: nested occupancy grids (1 = the single grid of S2)
    pose_levels: int = 0              # F2: levels that carry the pose gradient (0 = all); oracle config / GPU option


@dataclass
class RayBatch:
    origins: np.ndarray               # [R,3] fp32
    dirs: np.ndarray                  # [R,3] fp32, unit
    rgb: np.ndarray = None            # [R,3] fp32 in [0,1]
    depth: np.ndarray = None          # [R] fp32 range along the ray; <=0 => no depth term
    depth_var: np.ndarray = None      # [R] fp32 variance Sigma_D
    t_min: float = 0.05
    t_max: float = 1.8
    n_candidates: int = 32

    @property
    def n_rays(self):
        return int(self.origins.shape[0])


@dataclass
class Workload:
    name: str
    field: FieldConfig
    lambda_d: float
    bits: np.ndarray = None           # None => FULL
    batches: list = field(default_factory=list)
    extra: dict = field(default_factory=dict)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def unit_dirs(rng, n):
    d = rng.standard_normal((n, 3))
    return d / np.linalg.norm(d, axis=1, keepdims=True)


def init_params(seed, n_table, mlp_shapes):
    """theta_0 in the canonical flat layout: tables U(-1e-4, 1e-4), then each MLP matrix
    Xavier-uniform with bound sqrt(6/(fan_in+fan_out)) (BASELINE.json config 1; R18).
    mlp_shapes: [(name, n_out, n_in)] supplied by the caller."""
    rng = np.random.Generator(np.random.PCG64([seed, 0x7e7a]))
    parts = [rng.uniform(-1e-4, 1e-4, int(n_table)).astype(np.float32)]
    for _, n_out, n_in in mlp_shapes:
        bound = np.sqrt(6.0 / (n_in + n_out))
        parts.append(rng.uniform(-bound, bound, int(n_out) * int(n_in)).astype(np.float32))
    return np.concatenate(parts)


def lognormal_var(rng, n, mu=-2.0, sigma=1.0):
    return np.exp(rng.normal(mu, sigma, n))


# ------------------------------------------------------------------------------- config 1

def config1(variant_b=False, seed=0, R=256, K=32):
    """Tiny fp32 case (BASELINE.json configs[0]).  AABB [-2,3]^3 so all R*K candidates are
    inside (R19); variant 1b uses AABB [0,1]^3 to exercise clipping."""
    rng = np.random.Generator(np.random.PCG64(seed))
    fc = FieldConfig(aabb_min=(0.0, 0.0, 0.0) if variant_b else (-2.0, -2.0, -2.0),
                     aabb_extent=1.0 if variant_b else 5.0,
                     n_levels=4, n_features=2, log2_table_size=10, n_min=4, n_max=32, occ_res=32,
                     density_hidden=16, density_out=16, geo_offset=0, geo_count=16, sh_degree=2,
                     color_hidden=16, color_hidden_layers=1, mlp_precision=0, seed=seed,
                     max_rays=R, max_candidates=K)
    o = rng.uniform(0.0, 1.0, (R, 3))
    d = unit_dirs(rng, R)
    b = RayBatch(_f32(o), _f32(d), _f32(rng.uniform(0, 1, (R, 3))), _f32(rng.uniform(0.3, 1.5, R)),
                 _f32(lognormal_var(rng, R)), 0.05, 1.8, K)
    return Workload("cfg1b" if variant_b else "cfg1", fc, 0.1, None, [b])


# ------------------------------------------------------------------------------- config 2

def config2(seed=2, R=4096, K=128, n_batches=1, occ_res=128, field_overrides=None):
    """Instant-NGP-default field, 128^3 sphere-union occupancy at >= 15 % (BASELINE.json configs[1])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    fc = FieldConfig(seed=seed, max_rays=R, max_candidates=K, occ_res=occ_res, mlp_precision=1)
    if field_overrides:
        fc = replace(fc, **field_overrides)
    centres, radii, bits, frac = scenes.sphere_union_occupancy(rng, occ_res, 0.15)
    batches = []
    for i in range(n_batches):
        brng = np.random.Generator(np.random.PCG64([seed, 1000 + i]))
        o = np.zeros((0, 3))
        while o.shape[0] < R:
            cand = brng.uniform(0.05, 0.95, (2 * R, 3))
            inside = scenes.inside_any_sphere(cand, centres, radii)
            o = np.concatenate([o, cand[~inside]])
        o = o[:R]
        d = unit_dirs(brng, R)
        hit = scenes.ray_sphere_union(_f32(o).astype(np.float64), _f32(d).astype(np.float64),
                                      centres, radii)
        depth = np.where(np.isfinite(hit), hit * (1.0 + 0.01 * brng.standard_normal(R)), 0.0)
        batches.append(RayBatch(_f32(o), _f32(d), _f32(brng.uniform(0, 1, (R, 3))), _f32(depth),
                                _f32(lognormal_var(brng, R)), 0.02, float(np.sqrt(3.0)), K))
    return Workload("cfg2", fc, 1.0, bits, batches,
                    dict(occupancy_fraction=frac, n_spheres=len(radii)))


# --------------------------------------------------------------------------- configs 3, 4, 5

def config3(seed=3, R=1 << 14, K=128, n_keyframes=10, n_batches=4, width=1200, height=680,
            first_batch=0, field_overrides=None, outlier_fraction=0.05):
    """Keyframe-window mapping in the synthetic room (BASELINE.json configs[2]).  Batches are
    drawn uniformly over all (keyframe, pixel) pairs, seeded per step."""
    room = scenes.Room(seed)
    kfs = scenes.KeyframeSet(room, seed, n_keyframes, width, height, outlier_fraction)
    fc = FieldConfig(aabb_min=(0.0, 0.0, 0.0), aabb_extent=8.0, seed=seed, max_rays=R,
                     max_candidates=K, mlp_precision=1)
    t_min, t_max = 0.05, 10.5
    fc.occ_sigma_threshold = float(np.float32(0.01 / ((t_max - t_min) / K)))
    if field_overrides:
        fc = replace(fc, **field_overrides)
    batches = [kfs.draw_batch(step, R, t_min, t_max, K, RayBatch)
               for step in range(first_batch, first_batch + n_batches)]
    return Workload("cfg3", fc, 1.0, None, batches, dict(room=room, keyframes=kfs))


def config4(seed=4, R=1 << 12, K=512, n_keyframes=25, n_batches=1, occ_res=256, width=1200,
            height=680, field_overrides=None):
    """Large-table stress (BASELINE.json configs[3]): F=4, T=2^22, N_max=8192, bf16 MLPs,
    256^3 occupancy = the ~10 % of cells nearest to a surface."""
    room = scenes.Room(seed)
    kfs = scenes.KeyframeSet(room, seed, n_keyframes, width, height)
    fc = FieldConfig(aabb_min=(0.0, 0.0, 0.0), aabb_extent=8.0, n_features=4, log2_table_size=22,
                     n_max=8192, occ_res=occ_res, seed=seed, max_rays=R, max_candidates=K,
                     mlp_precision=2)
    if field_overrides:
        fc = replace(fc, **field_overrides)
    bits, frac = scenes.near_surface_occupancy(room, fc.occ_res, 8.0, 0.10)
    batches = [kfs.draw_batch(step, R, 0.05, 10.5, K, RayBatch) for step in range(n_batches)]
    return Workload("cfg4", fc, 1.0, bits, batches,
                    dict(room=room, keyframes=kfs, occupancy_fraction=frac))


def config5_views(seed=3, n_views=4, width=1200, height=680, K=256, stride=1):
    """Held-out full-frame views of config 3's room for nsm_render (BASELINE.json configs[4]).
    stride>1 gives the pixel-strided subset the oracle renders."""
    room = scenes.Room(seed)
    kfs = scenes.KeyframeSet(room, seed + 5000, n_views, width, height)
    views = []
    for i in range(n_views):
        o, d = kfs.rays(i)
        o = o.reshape(height, width, 3)[::stride, ::stride].reshape(-1, 3)
        d = d.reshape(height, width, 3)[::stride, ::stride].reshape(-1, 3)
        views.append(RayBatch(_f32(o), _f32(d), None, None, None, 0.05, 10.5, K))
    return views
