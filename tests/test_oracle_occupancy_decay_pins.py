"""Pins of the oracle's decayed partial occupancy refresh (row f4; paper silent, after [17]): reduction to S14's FROM_FIELD,
exact coverage of the strided subsets, geometric decay of unvisited cells, a closed form on a constant field.  CPU only."""
from dataclasses import replace

import numpy as np

from oracle import oracle as orc
from workloads import configs


def small(seed=0, G=16, zero_tables=False):
    w = configs.config1()
    fc = replace(w.field, occ_res=G, occ_sigma_threshold=1.0)
    n_table, n_mlp = orc.param_count(fc)
    theta = configs.init_params(seed, n_table, orc.mlp_shapes(fc)).astype(np.float64)
    theta[:n_table] *= 0.0 if zero_tables else 5e3
    return fc, theta


def test_one_subset_no_memory_is_from_field():
    fc, theta = small()
    A, B = orc.Oracle(fc, theta.copy()), orc.Oracle(fc, theta.copy())
    bits_ref, sig = A.occupancy_from_field(want_sigma=True)
    bits, vis = B.occupancy_decay_update(1, 0.0, want_sigma=True)
    assert np.array_equal(bits, bits_ref) and np.array_equal(vis, sig) and np.array_equal(B.occ_grid, sig)
    assert 0.02 < np.unpackbits(bits).mean() < 0.98           # a non-trivial field


def test_subsets_cover_every_cell_exactly_once_and_unvisited_cells_decay():
    fc, theta = small(1)
    O = orc.Oracle(fc, theta.copy())
    _, sig = orc.Oracle(fc, theta.copy()).occupancy_from_field(want_sigma=True)
    n_sub, decay, cells = 5, 0.8, fc.occ_res ** 3
    visits = np.zeros(cells, int)
    when = np.full(cells, -1)
    for u in range(n_sub):
        bits, vis = O.occupancy_decay_update(n_sub, decay, want_sigma=True)
        seen = vis >= 0
        assert np.array_equal(np.nonzero(seen)[0] % n_sub, np.full(seen.sum(), u % n_sub))
        assert np.array_equal(vis[seen], sig[seen])           # the visited cells get the field's density at their centre
        visits += seen
        when[seen] = u
    assert np.all(visits == 1)
    # after n_sub updates: grid = sigma * decay^(age), age = updates since the visit (the field did not change)
    age = (n_sub - 1) - when
    assert np.abs(O.occ_grid - sig * decay ** age).max() <= 1e-12 * sig.max()
    bits = np.unpackbits(O.bits, bitorder="little")[:cells].astype(bool)
    assert np.array_equal(bits, O.occ_grid > float(np.float32(fc.occ_sigma_threshold)))
    # a second round: running maximum of the decayed old value and the new one (equal field: max = sigma again at the visit)
    g_before = O.occ_grid.copy()
    O.occupancy_decay_update(n_sub, decay)
    v0 = np.arange(cells) % n_sub == 0
    assert np.abs(O.occ_grid[v0] - sig[v0]).max() <= 1e-12 * sig.max()
    assert np.abs(O.occ_grid[~v0] - decay * g_before[~v0]).max() <= 1e-15 * sig.max()


def test_constant_field_closed_form_and_seeding_by_a_full_refresh():
    """Zero tables: sigma = exp(0) = 1 in every cell.  Seeded by FROM_FIELD (grid = 1), k updates with n_sub subsets leave
    grid = decay^(age) with age in [0, n_sub): bits follow decay^age > thr."""
    fc, theta = small(2, zero_tables=True)
    fc = replace(fc, occ_sigma_threshold=0.5)
    O = orc.Oracle(fc, theta.copy())
    _, sig = O.occupancy_from_field(want_sigma=True)
    assert np.abs(sig - 1.0).max() <= 1e-12 and np.array_equal(O.occ_grid, sig)
    n_sub, decay = 4, 0.7
    for u in range(7):
        O.occupancy_decay_update(n_sub, decay)
    c = np.arange(fc.occ_res ** 3)
    last = 6 - ((6 - c % n_sub) % n_sub)                      # index of the last update that visited c
    want = decay ** (6 - last)
    assert np.abs(O.occ_grid - want).max() <= 1e-12
    bits = np.unpackbits(O.bits, bitorder="little")[:c.size].astype(bool)
    assert np.array_equal(bits, want > 0.5) and 0 < bits.mean() < 1
