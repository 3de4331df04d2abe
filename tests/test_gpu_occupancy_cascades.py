"""GPU parity of the rest of row f4 (readings R23 / R25): nested occupancy cascades in the marcher (index
path: bit-exact), FROM_FIELD and the strided refresh over all cascades, and the stochastic partial refresh
(nsm_update_occupancy_stochastic) against orc_occupancy_stochastic_update."""
from dataclasses import replace

import numpy as np
import pytest

from oracle import oracle as orc
from tests.gpu_common import make_pair, tol_for
from workloads import configs

pytestmark = pytest.mark.gpu


def cascade_workload(C, G=32, R=1024, K=128, precision=None):
    """config-3-style room data on a field with C occupancy cascades; the AABB is the cube [0,8]^3 around the 8x6x3 m room,
    so the room's contents sit around the cube's centre region in x, y and below it in z: all cascades see geometry."""
    w = configs.config3(R=R, K=K, n_keyframes=3, n_batches=4, width=300, height=170)
    fc = replace(w.field, occ_res=G, occ_cascades=C, occ_sigma_threshold=1.0)
    if precision is not None:
        fc = replace(fc, mlp_precision=precision)
    return replace(w, field=fc)


@pytest.mark.parametrize("C", [2, 4])
def test_marcher_with_cascades_is_bit_exact(nsm, C):
    """SET random bits on every cascade: counts, offsets, the (ray, k) list and t, delta, x word for word (P1 / P2)."""
    w = cascade_workload(C)
    f, O, _ = make_pair(nsm, w, seed=31, table_scale=0.5)
    n = orc.n_occ_cells(w.field)
    assert f.n_occ_cells == n == C * 32 ** 3
    rng = np.random.Generator(np.random.PCG64(40 + C))
    bits = rng.integers(0, 256, n // 8, dtype=np.uint8) & rng.integers(0, 256, n // 8, dtype=np.uint8)   # ~25 % set
    f.nsm_update_occupancy(nsm.NSM_OCC_SET, bits)
    assert np.array_equal(f.nsm_get_occupancy(), bits)
    O.set_occupancy(bits)
    for b in w.batches[:2]:
        st = f.nsm_backward(nsm.DeviceBatch(b), w.lambda_d)
        so, tr = O.train_step(b, w.lambda_d, apply_adam=False, trace=("counts", "offsets", "s_ray", "s_k", "s_t", "s_delta", "s_x"))
        assert st["n_samples"] == so["n_samples"] and 0 < so["n_samples"] < b.n_rays * b.n_candidates
        for k in ("counts", "offsets", "s_ray", "s_k"):
            assert np.array_equal(f.nsm_debug_last_step(k), tr[k]), k
        for k in ("s_t", "s_delta", "s_x"):
            assert np.array_equal(f.nsm_debug_last_step(k).view(np.uint32), tr[k].view(np.uint32)), k
        # the samples really come from several cascades
        _, casc = orc.occupancy_cell(w.field, tr["s_x"][:: max(1, len(tr["s_x"]) // 4000)])
        assert len(np.unique(casc)) >= 2
        tol = tol_for(w.field, f.nsm_mlp_path())
        assert abs(st["loss"] - so["loss"]) <= tol * abs(so["loss"])
    f.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_from_field_strided_and_stochastic_refresh_over_cascades(nsm, precision):
    """After a few training steps: FROM_FIELD over all C G^3 cells, two strided decay updates and four stochastic updates,
    each against the oracle fed the GPU's parameters: grid within tolerance, bits equal outside the tolerance band, and
    the marcher bit-exact on the GPU's own bits afterwards."""
    C, G = 3, 32
    w = cascade_workload(C, G, precision=precision)
    f, O, _ = make_pair(nsm, w, seed=33, table_scale=0.5)
    tol = tol_for(w.field, f.nsm_mlp_path())
    thr = float(np.float32(w.field.occ_sigma_threshold))
    n = C * G ** 3

    def sync_params():
        th, _, _, step = f.nsm_get_params()
        O.theta, O.step = th.astype(np.float64), step

    def check(tag):
        grid = f.nsm_get_occupancy_grid().astype(np.float64)
        assert grid.shape == (n,)
        assert np.abs(grid - O.occ_grid).max() <= tol * max(O.occ_grid.max(), thr), (tag, np.abs(grid - O.occ_grid).max())
        bits_g = np.unpackbits(f.nsm_get_occupancy(), bitorder="little")[:n].astype(bool)
        bits_o = np.unpackbits(O.bits, bitorder="little")[:n].astype(bool)
        band = np.abs(O.occ_grid - thr) <= tol * thr + tol * np.abs(O.occ_grid)
        assert np.array_equal(bits_g[~band], bits_o[~band]), tag
        O.occ_grid = grid.copy()                                 # keep the two histories together (max is not linear)
        return bits_g

    for b in w.batches[:3]:
        f.nsm_train_step(nsm.DeviceBatch(b), w.lambda_d, want_stats=False)
    sync_params()
    with pytest.raises(nsm.NsmError):
        f.nsm_update_occupancy_stochastic(100, 0.9)              # unseeded grid
    f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD)
    O.occupancy_from_field(want_sigma=True)
    bits_g = check("from_field")
    per_cascade = bits_g.reshape(C, -1).mean(axis=1)
    assert np.all(per_cascade > 0.01) and np.all(per_cascade < 0.99), per_cascade
    for u in range(2):
        f.nsm_train_step(nsm.DeviceBatch(w.batches[u]), w.lambda_d, want_stats=False)
        sync_params()
        f.nsm_update_occupancy_decay(4, 0.9)
        O.occupancy_decay_update(4, 0.9)
        check(f"strided {u}")
    for u, (n_draws, decay) in enumerate(((20000, 0.95), (20000, 0.95), (777, 0.5), (50000, 1.0))):
        f.nsm_train_step(nsm.DeviceBatch(w.batches[u % 4]), w.lambda_d, want_stats=False)
        sync_params()
        f.nsm_update_occupancy_stochastic(n_draws, decay)
        _, cells, x, sig = O.occupancy_stochastic_update(n_draws, decay, want_draws=True)
        if u == 0:
            assert len(np.unique(cells)) < n_draws                 # some cells are drawn twice: the atomic maximum is exercised
        bits_g = check(f"stochastic {u}")
    assert 0.02 < bits_g.mean() < 0.98
    # the marcher runs on the GPU's bits
    O.set_occupancy(f.nsm_get_occupancy())
    st = f.nsm_backward(nsm.DeviceBatch(w.batches[0]), w.lambda_d)
    so, tr = O.train_step(w.batches[0], w.lambda_d, apply_adam=False, trace=("counts",))
    assert st["n_samples"] == so["n_samples"] and np.array_equal(f.nsm_debug_last_step("counts"), tr["counts"])
    f.close()


def test_stochastic_refresh_with_every_cell_drawn_and_no_memory(nsm):
    """decay = 0 wipes the grid; with ~20 draws per cell every cell is drawn (checked), so every cell's value is the
    maximum over its own draws: the GPU grid against the oracle's within tolerance on all C G^3 cells, and that maximum
    is at least the smallest density drawn in the cell (the atomic maximum over ~20 duplicates per cell)."""
    C, G = 2, 16
    w = cascade_workload(C, G, R=512)
    f, O, _ = make_pair(nsm, w, seed=35, table_scale=0.5)
    tol = tol_for(w.field, f.nsm_mlp_path())
    n = C * G ** 3
    f.nsm_update_occupancy(nsm.NSM_OCC_FROM_FIELD)
    O.occupancy_from_field(want_sigma=True)
    f.nsm_update_occupancy_stochastic(20 * n, 0.0)
    _, cells, _, sig = O.occupancy_stochastic_update(20 * n, 0.0, want_draws=True)
    assert len(np.unique(cells)) == n
    grid = f.nsm_get_occupancy_grid().astype(np.float64)
    assert np.abs(grid - O.occ_grid).max() <= tol * O.occ_grid.max()
    lo = np.full(n, np.inf); np.minimum.at(lo, cells.astype(np.int64), sig)
    assert np.all(O.occ_grid >= lo) and np.all(O.occ_grid >= 0)
    f.close()


def test_cascade_config_validation(nsm):
    w = cascade_workload(2)
    with pytest.raises(nsm.NsmError):
        nsm.Field(replace(w.field, occ_cascades=9), "cuda:0")
    with pytest.raises(nsm.NsmError):
        nsm.Field(replace(w.field, occ_cascades=8, occ_res=1024), "cuda:0")      # 2^33 cells
