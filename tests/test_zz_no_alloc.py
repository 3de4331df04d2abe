"""GPU test of nsm_march_static (include/nsm.h "S1-S3 alone, allocating nothing"): the marcher behind an entry point
whose scratch memory (the chained scan's counters and status words) is a file-scope device array, for callers that
cannot call cudaMalloc.  Its output against the existing path's (the field's own step, read back with
nsm_debug_last_step) on the same inputs: S1-S3 is the index path, so the comparison is word for word (P1 / P2), on
calls made in a row, back to back, with different ray counts.  Collected last on purpose (the file name): the suite
runs with pytest -x."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from workloads import configs

pytestmark = pytest.mark.gpu

ITEMS = ("counts", "offsets", "s_ray", "s_k", "s_t", "s_delta", "s_x")


def field_path(nsm, f, batch, lambda_d=1.0):
    """S1-S3 as the field's own step runs them (nsm_backward, no Adam: the jitter step index stays Adam step + 1)."""
    st = f.nsm_backward(nsm.DeviceBatch(batch), lambda_d)
    out = {k: f.nsm_debug_last_step(k) for k in ITEMS}
    assert st["n_samples"] == int(out["offsets"][-1]) == len(out["s_ray"])
    return out


def assert_same(tag, got, ref):
    for k in ITEMS:
        assert got[k].shape == ref[k].shape, (tag, k, got[k].shape, ref[k].shape)
        assert np.array_equal(np.ascontiguousarray(got[k]).view(np.uint32), np.ascontiguousarray(ref[k]).view(np.uint32)), (tag, k)


def head(batch, n):
    return configs.RayBatch(batch.origins[:n], batch.dirs[:n], batch.rgb[:n], batch.depth[:n], batch.depth_var[:n],
                            batch.t_min, batch.t_max, batch.n_candidates)


@pytest.mark.parametrize("C", [1, 2])
def test_calls_in_a_row_match_the_field_path(nsm, C):
    """Sphere-union occupancy (C = 1) or random bits on two cascades (C = 2), jittered candidates.  Three calls are
    enqueued back to back with no synchronise in between: 4096 rays, then 3001 rays (a ragged last block, fewer scan
    words than the call before left behind), then 4096 rays again into the buffers of the second call."""
    w = configs.config2(R=4096, K=128, n_batches=2, occ_res=64)
    fc = replace(w.field, occ_cascades=C)
    f = nsm.Field(fc, "cuda:0")
    theta0 = configs.init_params(5, f.n_table, f.mlp_shapes())
    f.nsm_set_params(theta0)
    bits = w.bits
    if C > 1:
        rng = np.random.Generator(np.random.PCG64(50 + C))
        n = f.n_occ_cells
        bits = rng.integers(0, 256, n // 8, dtype=np.uint8) & rng.integers(0, 256, n // 8, dtype=np.uint8)
    f.nsm_update_occupancy(nsm.NSM_OCC_SET, bits)
    b0, b1 = w.batches[0], head(w.batches[1], 3001)
    ref0, ref1 = field_path(nsm, f, b0), field_path(nsm, f, b1)
    assert 0 < len(ref1["s_ray"]) < len(ref0["s_ray"]) < 4096 * 128
    step = f.nsm_get_params()[3] + 1

    d_bits = torch.as_tensor(bits).to("cuda:0")
    db0, db1 = nsm.DeviceBatch(b0), nsm.DeviceBatch(b1)
    out_a = nsm.MarchBuffers(4096, 4096 * 128, "cuda:0")
    out_b = nsm.MarchBuffers(4096, 4096 * 128, "cuda:0")
    torch.cuda.synchronize()
    nsm.nsm_march_static(fc, db0, d_bits, out_a, step)
    nsm.nsm_march_static(fc, db1, d_bits, out_b, step)
    assert_same("first call", out_a.read(4096), ref0)
    assert_same("second call", out_b.read(3001), ref1)
    # third call: buffers that hold the previous call's result; no device memory is taken or given back around it
    free_before = torch.cuda.mem_get_info()[0]
    nsm.nsm_march_static(fc, db0, d_bits, out_b, step)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    assert_same("third call", out_b.read(4096), ref0)
    # a different step index is a different jitter stream: the entry point really takes it from its argument
    nsm.nsm_march_static(fc, db0, d_bits, out_a, step + 1)
    other = out_a.read(4096)
    assert not np.array_equal(other["s_t"][:1000], ref0["s_t"][:1000])
    f.close()


def test_every_cell_live_and_no_jitter(nsm):
    """bits = NULL (every cell live; the field's FULL mode) with the clipping cube of config 1b and jitter off."""
    w = configs.config1(variant_b=True, R=250, K=40)
    fc = replace(w.field)
    fc.jitter = 0                                    # read by make_config and nsm_march_static alike (default 1)
    f = nsm.Field(fc, "cuda:0")
    f.nsm_set_params(configs.init_params(1, f.n_table, f.mlp_shapes()))
    ref = field_path(nsm, f, w.batches[0], w.lambda_d)
    out = nsm.MarchBuffers(250, 250 * 40, "cuda:0")
    for call in range(2):
        nsm.nsm_march_static(fc, nsm.DeviceBatch(w.batches[0]), None, out, f.nsm_get_params()[3] + 1)
        assert_same(f"call {call}", out.read(250), ref)
    assert 0 < len(ref["s_ray"]) < 250 * 40          # the cube clips
    f.close()


def test_the_maximum_ray_count(nsm):
    """NSM_MARCH_STATIC_MAX_RAYS rays in one call (every status word of the scratch array in use, 65536 blocks in the
    look-back chain) against the field path, twice in a row."""
    R, K = nsm.NSM_MARCH_STATIC_MAX_RAYS, 2
    w = configs.config1(variant_b=True, R=256, K=K)
    fc = replace(w.field, max_rays=R, max_candidates=K, occ_res=32)
    rng = np.random.Generator(np.random.PCG64(77))
    batch = configs.RayBatch(rng.uniform(-0.2, 1.2, (R, 3)).astype(np.float32), configs.unit_dirs(rng, R).astype(np.float32),
                             rng.uniform(0, 1, (R, 3)).astype(np.float32), rng.uniform(0.3, 1.5, R).astype(np.float32),
                             np.full(R, 0.01, np.float32), 0.05, 1.8, K)
    bits = rng.integers(0, 256, 32 ** 3 // 8, dtype=np.uint8)
    f = nsm.Field(fc, "cuda:0")
    f.nsm_set_params(configs.init_params(2, f.n_table, f.mlp_shapes()))
    f.nsm_update_occupancy(nsm.NSM_OCC_SET, bits)
    ref = field_path(nsm, f, batch)
    step = f.nsm_get_params()[3] + 1
    f.close()
    assert 0 < len(ref["s_ray"]) < R * K
    out = nsm.MarchBuffers(R, R * K, "cuda:0")
    db, d_bits = nsm.DeviceBatch(batch), torch.as_tensor(bits).to("cuda:0")
    for call in range(2):
        nsm.nsm_march_static(fc, db, d_bits, out, step)
        assert_same(f"call {call}", out.read(R), ref)


def test_sizes_beyond_the_maximum_are_rejected(nsm):
    """One ray more than the scratch array serves, too many candidates, too small an output capacity: NSM_ERR_CAPACITY
    with a message that names the limit, and nothing is launched (the outputs keep their contents)."""
    w = configs.config1(variant_b=True, R=64, K=8)
    fc = w.field
    out = nsm.MarchBuffers(64, 64 * 8, "cuda:0")
    out.counts.fill_(7)
    R = nsm.NSM_MARCH_STATIC_MAX_RAYS + 1
    big = configs.RayBatch(np.zeros((R, 3), np.float32), np.tile(np.float32([0, 0, 1]), (R, 1)), None, None, None, 0.05, 1.8, 8)
    with pytest.raises(nsm.NsmError) as ei:
        nsm.nsm_march_static(fc, nsm.DeviceBatch(big), None, out, 1)
    assert ei.value.status == 4 and str(nsm.NSM_MARCH_STATIC_MAX_RAYS) in str(ei.value)          # NSM_ERR_CAPACITY
    small = nsm.DeviceBatch(w.batches[0])
    small.n_candidates = 4097
    with pytest.raises(nsm.NsmError) as ei:
        nsm.nsm_march_static(fc, small, None, out, 1)
    assert ei.value.status == 4 and "4096" in str(ei.value)
    small.n_candidates = 9                                                                     # 64 * 9 > capacity
    with pytest.raises(nsm.NsmError) as ei:
        nsm.nsm_march_static(fc, small, None, out, 1)
    assert ei.value.status == 4 and "capacity" in str(ei.value)
    with pytest.raises(nsm.NsmError) as ei:
        nsm.nsm_march_static(replace(fc, occ_res=48), nsm.DeviceBatch(w.batches[0]), None, out, 1)
    assert ei.value.status == 1                                                                # NSM_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert bool((out.counts == 7).all())
