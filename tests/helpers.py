"""Shared test helpers: small field configs and oracle construction (tests only)."""
from dataclasses import replace

import numpy as np

from oracle import oracle as orc
from workloads import configs


def tiny_field(**kw):
    """cfg 1 scaled down: L=2, T=2^6 (level 0 dense 5^3=125>64 -> hashed? no: n_min=2 -> 27 dense)."""
    base = dict(aabb_min=(-2.0, -2.0, -2.0), aabb_extent=5.0, n_levels=2, n_features=2,
                log2_table_size=6, n_min=2, n_max=8, occ_res=8, density_hidden=8, density_out=16,
                geo_offset=0, geo_count=16, sh_degree=2, color_hidden=8, color_hidden_layers=1,
                mlp_precision=0, seed=7, max_rays=8, max_candidates=8)
    base.update(kw)
    return configs.FieldConfig(**base)


def make_oracle(fc, seed=0, table_scale=None, omp=False):
    nt, nm = orc.param_count(fc)
    th = configs.init_params(seed, nt, orc.mlp_shapes(fc))
    if table_scale is not None:
        th[:nt] *= table_scale / 1e-4
    return orc.Oracle(fc, th, omp=omp)


def random_batch(seed, R, K, t_min=0.05, t_max=1.8, origin_lo=0.0, origin_hi=1.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    o = rng.uniform(origin_lo, origin_hi, (R, 3)).astype(np.float32)
    d = configs.unit_dirs(rng, R).astype(np.float32)
    return configs.RayBatch(o, d, rng.uniform(0, 1, (R, 3)).astype(np.float32),
                            rng.uniform(0.3, 1.5, R).astype(np.float32),
                            np.exp(rng.normal(-2, 1, R)).astype(np.float32), t_min, t_max, K)
