"""Pins of the oracle's synchronised-scale cast and boundary-hit counts (O9: f2, f3; PAPER.md:310 Alg. 1 l.4-5, :277)."""
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(__file__)


def test_hand_worked_boundary_hits():
    rows = [l.split("|") for l in open(os.path.join(HERE, "golden", "boundary_hits_example.txt")) if l.strip() and not l.startswith("#")]
    x = np.array([[float(r[0]) for r in rows]], np.float32)
    x = np.concatenate([x, np.zeros((1, 16 - x.shape[1]), np.float32)], axis=1)       # (zeros are not hits)
    codes, sinv, (up, lo) = oracle.quantize_scaled(x, np.array([448.0], np.float32), oracle.E4M3)
    assert sinv[0] == 1.0
    assert codes[0, :len(rows)].tolist() == [int(r[1], 16) for r in rows]
    assert up == sum(r[2].strip() == "U" for r in rows) == 3 and lo == sum(r[2].strip() == "L" for r in rows) == 2


@pytest.mark.parametrize("fmt", [oracle.E4M3, oracle.E5M2])
@pytest.mark.parametrize("scaling", [oracle.SCALE_TENSOR, oracle.SCALE_BLOCK128])
def test_own_amax_is_the_plain_quantizer_and_counts_match_the_decoded_table(fmt, scaling):
    rng = np.random.default_rng(17 + fmt + 2 * scaling)
    x = (rng.normal(0, 1, (200, 272)) * np.exp(rng.normal(0, 4, (200, 272)))).astype(np.float32)
    x[3, 5] = 0.0
    a = oracle.amax(x, scaling)
    if scaling == oracle.SCALE_TENSOR:
        assert a[0] == np.abs(x).max()
    else:
        assert a[1] == np.abs(x[:128, 128:256]).max() and a[-1] == np.abs(x[128:, 256:]).max()
    c0, s0 = oracle.quantize(x, fmt, scaling)
    c1, s1, (up, lo) = oracle.quantize_scaled(x, a, fmt, scaling)
    assert np.array_equal(c0, c1) and np.array_equal(s0, s1)
    tab = np.abs(oracle.fp8_table(fmt)[c1])
    sub = np.min(np.abs(oracle.fp8_table(fmt))[np.abs(oracle.fp8_table(fmt)) > 0])
    assert up == int((tab == oracle.fp8_max(fmt)).sum()) and up >= len(a) - 1
    assert lo == int(((tab <= sub) & (x != 0)).sum()) and lo > 0
    # an agreed amax twice the local one: every value halves, nothing reaches the top of the format
    c2, s2, (up2, lo2) = oracle.quantize_scaled(x, 2 * a, fmt, scaling)
    assert np.all(np.abs(oracle.fp8_table(fmt)[c2]) <= oracle.fp8_max(fmt) / 2) and up2 == 0 and lo2 >= lo
    assert np.array_equal(s2, 2 * s1)
    # an agreed amax far below the local one: the large values saturate
    c3, _, (up3, _) = oracle.quantize_scaled(x, 1e-3 * a, fmt, scaling)
    assert up3 > up and np.all(np.isfinite(oracle.fp8_table(fmt)[c3]))
