"""Input generators: deterministic, chunkable, shaped as BASELINE.json says."""
import numpy as np

import workloads as W


def test_five_configs_match_baseline_shapes():
    shapes = [c.shape for c in W.CONFIG_LIST]
    assert shapes == [(24,) * 3, (48,) * 3, (96,) * 3, (72,) * 3, (128, 128, 192)]
    assert [c.nbands for c in W.CONFIG_LIST] == [8, 64, 256, 128, 384]
    assert [c.complex for c in W.CONFIG_LIST] == [False, False, False, True, False]
    assert W.get(3).min_bytes == 2 * 96 ** 3 * 256 * 8 + 8 * 96 ** 3
    assert abs(W.get(1).h[0] - 0.37794522) < 1e-7


def test_bands_are_independently_reproducible():
    c = W.get(4).with_bands(6)
    a = W.make_psi(c)
    b = W.make_psi(c, [4, 1])
    assert a.dtype == np.complex128 and a.flags.c_contiguous
    assert np.array_equal(a[4], b[0]) and np.array_equal(a[1], b[1])
    assert not np.array_equal(a[0], a[1])
    assert np.array_equal(W.make_veff(c), W.make_veff(W.get(4)))


def test_value_distributions():
    c1 = W.get(1)
    v = W.make_veff(c1)
    assert v.min() >= -1 and v.max() <= 0
    c2 = W.get(2).with_bands(2)
    psi = W.make_psi(c2)
    assert abs(psi[:, 0, 0, 0]).max() < abs(psi[:, 24, 24, 24]).max() + 5  # envelope decays
    assert np.abs(psi[:, 0]).max() < np.abs(psi[:, 20:28]).max()
    v2 = W.make_veff(c2)
    assert v2.max() <= 0 and v2.min() < -1
    v3 = W.make_veff(W.get(3).with_bands(1))
    assert -2 <= v3.min() and v3.max() <= 0.5 and v3.std() < 0.3   # smoothed
    v5 = W.make_veff(W.get(5))
    assert v5.shape == (128, 128, 192)
    assert v5[0, 0, -1] - v5[0, 0, 0] > 0.5                        # ramp along z
