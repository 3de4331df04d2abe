"""Helpers shared by the GPU parity test modules: a CUDA field and an oracle built from the same seeded theta_0
(R18: parameters are always uploaded, never regenerated), and the tolerance rules of DESIGN.md section 5."""
import numpy as np

from oracle import oracle as orc
from workloads import configs

# the encoder output is fp32 on the CUDA-core path and a two-term 16-bit expansion on the tensor-core path
E_TOL = {"simt_fp32": 1e-4, "tcgen05_f16": 1e-4, "tcgen05_bf16": 1e-4}   # two-term (hi + lo) tiles


def tol_for(fc, path):
    """BASELINE.json north_star: 1e-4 on the fp32 configuration, 2e-2 where the configuration asks
    for fp16/bf16 MLPs.  While such a configuration still runs on the fp32 CUDA-core path it is held
    to 1e-3 (fp32 with the cancellation of up to 512 samples per ray in S10 and of colliding hash
    slots in S12)."""
    if fc.mlp_precision == 0:
        return 1e-4
    return 1e-3 if path == "simt_fp32" else 2e-2


def assert_close(name, got, ref, tol, scale=None):
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (name, got.shape, ref.shape)
    if ref.size == 0:
        return
    s = np.abs(ref).max() if scale is None else scale
    err = np.abs(got - ref) - tol * np.maximum(np.abs(ref), s)
    assert err.max() <= 0, f"{name}: max excess {err.max():.3e}, scale {s:.3e}, worst at {np.argmax(err)}"


def make_pair(nsm, w, seed=0, table_scale=0.1, mlp_scale=1.0, omp=False):
    fc = w.field
    f = nsm.Field(fc, "cuda:0")
    theta0 = configs.init_params(seed, f.n_table, f.mlp_shapes())
    theta0[:f.n_table] *= table_scale / 1e-4
    theta0[f.n_table:] *= mlp_scale
    f.nsm_set_params(theta0)
    O = orc.Oracle(fc, theta0, omp=omp)
    assert (O.n_table, O.n_mlp) == (f.n_table, f.n_mlp)
    assert np.array_equal(O.res, f.res) and np.array_equal(O.offset, f.offset)          # P1: S0 tables
    if w.bits is not None:
        f.nsm_update_occupancy(nsm.NSM_OCC_SET, w.bits)
        O.set_occupancy(w.bits)
    return f, O, theta0


