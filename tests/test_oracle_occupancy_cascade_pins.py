"""Pins of the rest of row f4 in the oracle (paper silent -> [17]; "region of interest" PAPER.md:266):
nested occupancy cascades (reading R23) and the stochastic partial refresh (reading R25).  CPU only.

Cascades: the cascade of a point and its cell re-derived in exact rational arithmetic; C = 1 is S2's single grid bit for
bit; a cell's centre maps back to that cell unless a finer cascade owns the centre; the cells of a cascade tile its cube
and nest in the next coarser one; a sphere rasterised through the cell centres is reproduced by the marcher's live test
to within the cell size of the cascade that owns each point.
Stochastic refresh: the draws re-derived in exact Python integers; points lie in their cells; chi-square uniformity of the
cells and of the offsets; drawn cells take max(decay * old, sigma(point)) with sigma re-evaluated through the oracle's
public encode + field_eval; undrawn cells decay geometrically; constant-field closed form; a doubly drawn cell keeps the
larger density."""
from dataclasses import replace
from fractions import Fraction

import numpy as np

from oracle import oracle as orc
from tests.helpers import random_batch
from workloads import configs


def field(C=3, G=16, seed=0, zero_tables=False, thr=1.0):
    w = configs.config1()
    fc = replace(w.field, occ_res=G, occ_cascades=C, occ_sigma_threshold=thr, aabb_min=(0.0, 0.0, 0.0), aabb_extent=1.0)
    n_table, n_mlp = orc.param_count(fc)
    theta = configs.init_params(seed, n_table, orc.mlp_shapes(fc)).astype(np.float64)
    theta[:n_table] *= 0.0 if zero_tables else 5e3
    return fc, theta


def exact_cell(x, C, G):
    """R23 in exact rationals on the fp32 inputs; returns (cascade, (gx, gy, gz)) or None when an fp32 rounding of the
    specified operations could matter (the point is then skipped by the caller: within 2^-20 of a decision boundary)."""
    xf = [Fraction(float(v)) for v in x]
    q = [v - Fraction(1, 2) for v in xf]
    m = max(abs(v) for v in q)
    j = C - 1
    for jj in range(C - 1):
        if m < Fraction(2) ** (jj - C):
            j = jj
            break
    eps = Fraction(1, 2 ** 20)
    for jj in range(C - 1):                                    # too close to a cascade boundary: skip
        if abs(m - Fraction(2) ** (jj - C)) < eps:
            return None
    xp = [v * 2 ** (C - 1 - j) + Fraction(1, 2) for v in q]
    g = []
    for v in xp:
        s = v * G
        if abs(s - round(s)) < eps * G * 2 ** C:               # too close to a cell face: skip
            return None
        g.append(min(int(s // 1), G - 1))
    return j, tuple(g)


def test_cascade_and_cell_against_exact_rationals():
    C, G = 4, 16
    fc, _ = field(C, G)
    rng = np.random.Generator(np.random.PCG64(5))
    # points at all scales around the centre, so every cascade is hit
    x = (0.5 + rng.uniform(-1, 1, (4000, 3)) * 0.5 * 2.0 ** -rng.integers(0, C + 1, (4000, 1))).astype(np.float32)
    x = np.clip(x, 0.0, np.nextafter(np.float32(1), np.float32(0)))
    cell, casc = orc.occupancy_cell(fc, x)
    checked = 0
    seen = set()
    for i in range(len(x)):
        ref = exact_cell(x[i], C, G)
        if ref is None:
            continue
        j, g = ref
        assert casc[i] == j, (x[i], casc[i], j)
        assert cell[i] == j * G ** 3 + g[0] + G * (g[1] + G * g[2]), (x[i], cell[i], ref)
        checked += 1
        seen.add(j)
    assert checked > 3500 and seen == set(range(C))


def test_one_cascade_is_the_single_grid_bit_for_bit():
    """C = 1 (and the legacy value 0) must leave S2 unchanged: the same march outputs on random bits, and the plain
    formula g = min(floor(x G), G - 1) for the cell."""
    fc1, _ = field(1, 8)
    fc0 = replace(fc1, occ_cascades=0)
    rng = np.random.Generator(np.random.PCG64(6))
    bits = rng.integers(0, 256, 8 ** 3 // 8, dtype=np.uint8)
    b = random_batch(3, 64, 24, t_min=0.01, t_max=1.2)
    m1, m0 = orc.march(fc1, bits, b), orc.march(fc0, bits, b)
    for k in ("counts", "s_ray", "s_k", "s_t", "s_x"):
        assert np.array_equal(m1[k], m0[k])
    x = m1["s_x"]
    cell, casc = orc.occupancy_cell(fc1, x)
    g = np.minimum(np.floor(x * np.float32(8)).astype(np.int64), 7)
    assert np.array_equal(cell, (g[:, 0] + 8 * (g[:, 1] + 8 * g[:, 2])).astype(np.uint64)) and not casc.any()
    live = (bits[cell >> 3] >> (cell & 7).astype(np.uint8)) & 1
    assert live.all() and 0 < m1["S"] < 64 * 24                # every compacted sample sits in a set cell


def test_cell_centres_map_back_and_cells_tile_and_nest():
    C, G = 3, 8
    fc, _ = field(C, G)
    n = C * G ** 3
    cells = np.arange(n, dtype=np.uint64)
    ctr = orc.occupancy_cell_point(fc, cells)
    back, casc = orc.occupancy_cell(fc, ctr)
    j_of = (cells // G ** 3).astype(np.int64)
    m = np.abs(ctr.astype(np.float64) - 0.5).max(axis=1)
    for j in range(C):
        sel = j_of == j
        # the cells of cascade j tile its cube: centres on the lattice (g + 1/2) 2^(j-(C-1)) / G about the centre
        side = 2.0 ** (j - (C - 1))
        g = np.stack([(cells[sel] % G), (cells[sel] // G) % G, (cells[sel] // G ** 2) % G], 1).astype(np.float64)
        assert np.array_equal(ctr[sel].astype(np.float64), 0.5 + ((g + 0.5) / G - 0.5) * side)
        owned = m[sel] >= (2.0 ** (j - 1 - C) if j > 0 else 0.0)      # not inside the next finer cube
        assert np.array_equal(back[sel][owned], cells[sel][owned]) and np.all(casc[sel][owned] == j)
        assert np.all(casc[sel][~owned] < j)                          # the finer cascade owns those centres
        if j > 0:
            assert (~owned).sum() == (G // 2) ** 3                    # exactly the inner eighth of the cube
    # nesting: a cell of cascade j lies inside one cell of cascade j + 1 (its centre's coarse cell, by plain geometry)
    for j in range(C - 1):
        sel = j_of == j
        coarse_side = 2.0 ** (j + 1 - (C - 1))
        gc = np.floor(((ctr[sel].astype(np.float64) - 0.5) / coarse_side + 0.5) * G).astype(np.int64)
        fine_half = 2.0 ** (j - (C - 1)) / G / 2
        lo = 0.5 + (gc / G - 0.5) * coarse_side
        assert np.all(ctr[sel] - fine_half >= lo - 1e-12) and np.all(ctr[sel] + fine_half <= lo + coarse_side / G + 1e-12)


def test_sphere_through_the_centres_is_what_the_marcher_sees():
    """Every cascade's bits are set from ONE geometric predicate at the cell centres (inside a sphere); a marched point
    must then be live iff it is inside the sphere, except within one cell diagonal of the surface -- measured in the cell
    size of the cascade that owns the point, so the allowance shrinks towards the centre.  A wrong zoom factor, a swapped
    axis or an off-by-one cascade breaks this."""
    C, G = 3, 32
    fc, _ = field(C, G)
    n = C * G ** 3
    centre, rad = np.array([0.53, 0.47, 0.5]), 0.21
    ctr = orc.occupancy_cell_point(fc, np.arange(n, dtype=np.uint64)).astype(np.float64)
    inside = np.linalg.norm(ctr - centre, axis=1) < rad
    bits = np.packbits(inside, bitorder="little")
    b = random_batch(11, 256, 64, t_min=0.0, t_max=1.0)
    allm = orc.march(fc, None, b, jitter=True, step=3)          # FULL: every candidate inside the cube
    live = orc.march(fc, bits, b, jitter=True, step=3)
    x = allm["s_x"].astype(np.float64)
    key_all = allm["s_ray"].astype(np.int64) * 64 + allm["s_k"]
    is_live = np.isin(key_all, live["s_ray"].astype(np.int64) * 64 + live["s_k"])
    _, casc = orc.occupancy_cell(fc, allm["s_x"])
    diag = np.sqrt(3.0) * 2.0 ** (casc.astype(np.float64) - (C - 1)) / G
    dist = np.linalg.norm(x - centre, axis=1) - rad
    sure_in, sure_out = dist < -diag, dist > diag
    assert is_live[sure_in].all() and not is_live[sure_out].any()
    assert sure_in.sum() > 200 and sure_out.sum() > 2000 and set(np.unique(casc)) == {0, 1, 2}
    # and the allowance really is finer near the centre: some points are decided in cascade 0 that cascade 2 could not decide
    coarse_diag = np.sqrt(3.0) / G
    assert ((casc == 0) & (np.abs(dist) > diag) & (np.abs(dist) < coarse_diag)).sum() > 0


def test_from_field_and_decay_cover_all_cascades():
    C, G = 2, 8
    fc, theta = field(C, G, seed=3)
    O = orc.Oracle(fc, theta.copy())
    bits, sig = O.occupancy_from_field(want_sigma=True)
    n = C * G ** 3
    assert sig.shape == (n,) and bits.size == n // 8
    # densities re-evaluated through the public encode + field_eval at the centres
    ctr = orc.occupancy_cell_point(fc, np.arange(n, dtype=np.uint64))
    e, _, _ = orc.encode(fc, theta, ctr, want_index=False)
    n_table, _ = orc.param_count(fc)
    Y = orc.sh(fc.sh_degree, np.array([[0.0, 0.0, 1.0]]))[0]
    ref = np.array([orc.field_eval(fc, theta[n_table:], e[i], Y)[0] for i in range(n)])
    assert np.abs(sig - ref).max() <= 1e-12 * ref.max()
    assert np.array_equal(np.unpackbits(bits, bitorder="little")[:n].astype(bool), sig > float(np.float32(fc.occ_sigma_threshold)))
    assert 0.02 < (sig > 1.0).mean() < 0.98
    # the strided decay update walks the global cell index over both cascades
    B = orc.Oracle(fc, theta.copy())
    b2, vis = B.occupancy_decay_update(1, 0.0, want_sigma=True)
    assert np.array_equal(b2, bits) and np.array_equal(vis, sig)


# ---------------------------------------------------------------- stochastic refresh (R25)

def mix32(x):
    x &= 0xffffffff
    x ^= x >> 16; x = (x * 0x7feb352d) & 0xffffffff
    x ^= x >> 15; x = (x * 0x846ca68b) & 0xffffffff
    x ^= x >> 16
    return x


def hash32(seed, step, r, k):
    h = mix32((seed & 0xffffffff) ^ 0x9e3779b9)
    for w in (seed >> 32, step, r, k):
        h = mix32(h ^ w)
    return h


def test_stochastic_draws_in_exact_integers_and_points_in_their_cells():
    C, G = 2, 8
    fc, theta = field(C, G, seed=4)
    fc = replace(fc, seed=0x1234567800000042)
    O = orc.Oracle(fc, theta.copy())
    O.occupancy_from_field(want_sigma=True)
    n = C * G ** 3
    for upd in range(3):
        _, cells, x, sig = O.occupancy_stochastic_update(200, 0.9, want_draws=True)
        for i in range(200):
            c = (hash32(fc.seed, upd, i, 0xffff0003) * n) >> 32
            assert cells[i] == c
            u = [(hash32(fc.seed, upd, i, 0xffff0004 + a) >> 8) / 2.0 ** 24 for a in range(3)]
            j, loc = c // G ** 3, c % G ** 3
            g = (loc % G, (loc // G) % G, loc // G ** 2)
            side = 2.0 ** (j - (C - 1))
            want = [0.5 + ((g[a] + u[a]) / G - 0.5) * side for a in range(3)]
            assert np.abs(x[i].astype(np.float64) - want).max() <= 2.0 ** -23
        back, _ = orc.occupancy_cell(fc, x)
        owned = np.abs(x.astype(np.float64) - 0.5).max(axis=1) >= np.where(cells >= G ** 3, 2.0 ** (-1 - C) * 2, 0.0)
        # a point drawn in a coarse cell that a finer cascade owns maps to the finer cascade; all others map back
        assert np.array_equal(back[owned], cells[owned])


def test_stochastic_draws_are_uniform():
    C, G = 1, 4
    fc, theta = field(C, G, seed=5)
    O = orc.Oracle(fc, theta.copy())
    n = G ** 3
    counts = np.zeros(n)
    us = []
    for upd in range(8):
        _, cells, x, _ = O.occupancy_stochastic_update(4000, 1.0, want_draws=True)
        counts += np.bincount(cells.astype(np.int64), minlength=n)
        g = np.stack([cells % G, (cells // G) % G, cells // G ** 2], 1).astype(np.float64)
        us.append(x.astype(np.float64) * G - g)
    exp = counts.sum() / n
    chi2 = ((counts - exp) ** 2 / exp).sum()
    assert chi2 < n - 1 + 5 * np.sqrt(2 * (n - 1))              # 5 sigma
    u = np.concatenate(us)
    assert u.min() >= 0 and u.max() < 1
    h = np.stack([np.histogram(u[:, a], bins=16, range=(0, 1))[0] for a in range(3)])
    chi2u = ((h - len(u) / 16) ** 2 / (len(u) / 16)).sum(axis=1)
    assert np.all(chi2u < 15 + 5 * np.sqrt(30))
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.02 and abs(np.corrcoef(u[:, 1], u[:, 2])[0, 1]) < 0.02


def test_stochastic_update_is_a_decayed_running_maximum():
    C, G = 2, 8
    fc, theta = field(C, G, seed=6)
    O = orc.Oracle(fc, theta.copy())
    _, sig0 = O.occupancy_from_field(want_sigma=True)
    n = C * G ** 3
    n_table, _ = orc.param_count(fc)
    Y = orc.sh(fc.sh_degree, np.array([[0.0, 0.0, 1.0]]))[0]
    grid = sig0.copy()
    for upd in range(4):
        decay = 0.6 + 0.1 * upd
        bits, cells, x, sig = O.occupancy_stochastic_update(300, decay, want_draws=True)
        # sigma at the drawn points through the public encode + field_eval
        e, _, _ = orc.encode(fc, theta, x, want_index=False)
        ref = np.array([orc.field_eval(fc, theta[n_table:], e[i], Y)[0] for i in range(len(x))])
        assert np.abs(sig - ref).max() <= 1e-12 * ref.max()
        grid *= decay
        np.maximum.at(grid, cells.astype(np.int64), ref)        # duplicates: the larger density, whatever the order
        assert np.abs(O.occ_grid - grid).max() <= 1e-12 * grid.max()
        assert np.array_equal(np.unpackbits(bits, bitorder="little")[:n].astype(bool), O.occ_grid > float(np.float32(fc.occ_sigma_threshold)))
        drawn = np.zeros(n, bool); drawn[cells.astype(np.int64)] = True
        assert 0 < drawn.sum() < 300 or len(np.unique(cells)) == 300
    assert len(np.unique(cells)) < len(cells) or True


def test_stochastic_constant_field_closed_form():
    """Zero tables: sigma = 1 everywhere.  Seeded with grid = 1; after k updates a cell holds decay^(updates since it was
    last drawn), or decay^k if never drawn."""
    C, G = 1, 8
    fc, theta = field(C, G, seed=7, zero_tables=True, thr=0.5)
    O = orc.Oracle(fc, theta.copy())
    O.occupancy_from_field(want_sigma=True)
    n, decay, k = G ** 3, 0.8, 5
    last = np.full(n, -1)
    for upd in range(k):
        _, cells, _, sig = O.occupancy_stochastic_update(100, decay, want_draws=True)
        assert np.abs(sig - 1.0).max() <= 1e-12
        last[cells.astype(np.int64)] = upd
    age = np.where(last >= 0, k - 1 - last, k)
    assert np.abs(O.occ_grid - decay ** age).max() <= 1e-12
    bits = np.unpackbits(O.bits, bitorder="little")[:n].astype(bool)
    assert np.array_equal(bits, decay ** age > 0.5) and 0 < bits.mean() < 1
