"""CPU pins of the two metrics of row f3 ("PSNR ... and L1 depth error"), the functions
paper_2210_13641_b200.ablation reports: closed forms on known images, no GPU."""
import numpy as np
import pytest

from paper_2210_13641_b200.ablation import aggregate, depth_l1, psnr


def test_psnr_closed_forms():
    rng = np.random.Generator(np.random.PCG64(0))
    img = rng.uniform(0.1, 0.9, (17, 23, 3)).astype(np.float32)
    # a constant offset d: MSE = d^2, PSNR = -20 log10(d); d = 0.1 -> 20 dB, d = 0.01 -> 40 dB
    assert psnr(img + np.float32(0.1), img) == pytest.approx(20.0, abs=1e-4)
    assert psnr(img - np.float32(0.01), img) == pytest.approx(40.0, abs=1e-3)
    # black against white: MSE = 1 -> 0 dB; peak scales as 20 log10(peak)
    assert psnr(np.zeros((4, 4, 3)), np.ones((4, 4, 3))) == pytest.approx(0.0, abs=1e-12)
    assert psnr(np.zeros((4, 4, 3)), np.ones((4, 4, 3)), peak=255.0) == pytest.approx(20 * np.log10(255.0), abs=1e-9)
    # symmetric, and one wrong pixel of N: MSE = e^2 / N
    a = np.zeros((10, 10)); b = a.copy(); b[3, 4] = 0.5
    assert psnr(a, b) == psnr(b, a) == pytest.approx(10 * np.log10(1.0 / (0.25 / 100)), abs=1e-9)
    # uniform noise of half-width h: MSE = h^2 / 3 (large sample)
    n = rng.uniform(-0.05, 0.05, (400, 400))
    assert psnr(0.5 + n, np.full((400, 400), 0.5)) == pytest.approx(10 * np.log10(3.0 / 0.05 ** 2), abs=0.05)
    # identical images: finite (floored MSE), very large
    assert 100.0 < psnr(img, img) < 130.0


def test_depth_l1_closed_forms():
    d = np.linspace(0.5, 4.0, 101).reshape(1, -1)
    assert depth_l1(d + 0.25, d) == pytest.approx(0.25, abs=1e-12)
    assert depth_l1(d - 0.25, d) == pytest.approx(0.25, abs=1e-12)              # absolute value
    e = np.zeros_like(d); e[0, :50] = 0.1; e[0, 50:] = -0.3
    assert depth_l1(d + e, d) == pytest.approx((50 * 0.1 + 51 * 0.3) / 101, abs=1e-12)   # a mean, not a sum or an RMS
    valid = np.zeros_like(d, bool); valid[0, :50] = True
    assert depth_l1(d + e, d, valid) == pytest.approx(0.1, abs=1e-12)            # the mask selects pixels
    assert depth_l1(d.astype(np.float32), d.astype(np.float32)) == 0.0


def test_aggregate_mean_and_sample_std():
    mk = lambda p, l: dict(weighted=[dict(step=10, seconds=1.0, psnr=p, depth_l1_m=l, psnr_seen=p + 1, depth_l1_seen_m=l / 2)])
    agg = aggregate([mk(20.0, 0.10), mk(22.0, 0.14), mk(24.0, 0.12)])
    r = agg["weighted"][0]
    assert r["n"] == 3 and r["step"] == 10
    assert r["psnr_mean"] == pytest.approx(22.0) and r["psnr_std"] == pytest.approx(2.0)          # ddof = 1
    assert r["depth_l1_m_mean"] == pytest.approx(0.12) and r["depth_l1_m_std"] == pytest.approx(0.02)
    one = aggregate([mk(20.0, 0.10)])["weighted"][0]
    assert one["psnr_std"] == 0.0
