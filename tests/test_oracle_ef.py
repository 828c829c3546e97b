"""Pins of the oracle's error-feedback quantizer (O8; Alg. 1 l.11-15) against what the paper and the
arithmetic fix: a hand-worked example, the reduction to the plain quantizer, the telescoping identity of error feedback,
the bound on the residual, and the 1/T decay of the time-averaged error."""
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(__file__)


def test_worked_example_from_the_golden_file():
    u = np.array([[448.0, 1.03125, -0.296875, 0.0]], np.float32)
    r = np.zeros_like(u)
    rows = [l for l in open(os.path.join(HERE, "golden", "ef_worked_example.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 4
    for line in rows:
        step, codes_hex, resid, sinv = [f.strip() for f in line.split("|")]
        codes, s, r = oracle.ef_quantize(u, r, oracle.E4M3, oracle.SCALE_TENSOR)
        assert [int(c, 16) for c in codes_hex.split()] == codes.ravel().tolist(), step
        assert np.array_equal(r.ravel(), np.array([float(x) for x in resid.split()], np.float32)), step
        assert s[0] == np.float32(float(sinv))


@pytest.mark.parametrize("fmt", [oracle.E4M3, oracle.E5M2])
@pytest.mark.parametrize("scaling", [oracle.SCALE_TENSOR, oracle.SCALE_BLOCK128])
def test_zero_residual_is_the_plain_quantizer_and_the_residual_is_its_error(fmt, scaling):
    rng = np.random.default_rng(5 + fmt + 2 * scaling)
    u = (rng.normal(0, 1, (150, 300)) * np.exp(rng.normal(0, 2, (150, 300)))).astype(np.float32)
    c0, s0 = oracle.quantize(u, fmt, scaling)
    c1, s1, r1 = oracle.ef_quantize(u, np.zeros_like(u), fmt, scaling)
    assert np.array_equal(c0, c1) and np.array_equal(s0, s1)
    tab = oracle.fp8_table(fmt)
    bn = (300 + 127) // 128
    sidx = (np.arange(150)[:, None] // 128) * bn + np.arange(300)[None, :] // 128 if scaling else np.zeros((150, 300), int)
    deq = (tab[c1].astype(np.float32) * s1[sidx]).astype(np.float32)
    assert np.array_equal(r1, (u - deq).astype(np.float32))
    # |residual| <= half the widest gap between neighbouring codes, in units of scale_inv (E4M3: 448 - 416 = 32; E5M2: 8192)
    half_gap = 16.0 if fmt == oracle.E4M3 else 4096.0
    assert np.all(np.abs(r1) <= half_gap * s1[sidx] * (1 + 1e-6))


@pytest.mark.parametrize("fmt", [oracle.E4M3, oracle.E5M2])
def test_telescoping_identity_and_time_averaged_error(fmt):
    """sum_t deq_t = sum_t u_t + R_0 - R_T (each step: deq = u~ - R_new, u~ = u + R_old), so the error of the running mean
    of what was sent is (R_0 - R_T) / T: it decays like 1 / T, while without feedback it does not decay at all."""
    rng = np.random.default_rng(11 + fmt)
    m, n, T = 64, 96, 40
    base = rng.normal(0, 1, (m, n)).astype(np.float32)
    tab = oracle.fp8_table(fmt)
    r = rng.normal(0, 1e-3, (m, n)).astype(np.float32)
    r0 = r.copy()
    sum_u = np.zeros((m, n)); sum_deq = np.zeros((m, n)); sum_plain = np.zeros((m, n))
    for t in range(T):
        u = (base + 0.05 * rng.normal(0, 1, (m, n))).astype(np.float32)
        codes, s, r = oracle.ef_quantize(u, r, fmt)
        sum_u += u
        sum_deq += (tab[codes].astype(np.float32) * s[0]).astype(np.float64)
        pc, ps = oracle.quantize(u, fmt)
        sum_plain += (tab[pc].astype(np.float32) * ps[0]).astype(np.float64)
    # FP32 rounding of the three operations per step: a few ulp of max|u| per step
    tol = T * 4 * np.finfo(np.float32).eps * float(np.abs(base).max() + 1)
    assert np.abs(sum_deq - (sum_u + r0 - r)).max() <= tol
    err_ef = np.linalg.norm(sum_deq - sum_u) / np.linalg.norm(sum_u)
    err_plain = np.linalg.norm(sum_plain - sum_u) / np.linalg.norm(sum_u)
    assert err_ef < 0.2 * err_plain           # (measured: ~ 1 / T of the per-step error against ~ 1 / sqrt(T))
    assert np.linalg.norm(sum_deq - sum_u) <= np.linalg.norm(r0 - r) + tol * np.sqrt(m * n)


def test_encode_ef_composes_whitening_and_feedback():
    """encode_ef = O3 then O8: with R = 0 it is encode(); its residual lives in the transformed coordinates (it is the
    quantization error of the WHITENED tensor)."""
    rng = np.random.default_rng(3)
    d, k = 48, 6
    X = rng.normal(0, 1, (400, d)) * np.linspace(2, 0.2, d)
    A = oracle.factor_accumulate(X)
    bas = oracle.refresh_basis(A, rng.normal(0, 1, (d, k)), 3, 1e-3)
    W = rng.normal(0, 1, (40, d))
    c0, s0, wt0 = oracle.encode(W, None, bas)
    c1, s1, r1, wt1 = oracle.encode_ef(W, np.zeros((40, d), np.float32), None, bas)
    assert np.array_equal(c0, c1) and np.array_equal(s0, s1) and np.array_equal(wt0, wt1)
    tab = oracle.fp8_table(oracle.E4M3)
    assert np.array_equal(r1, (wt1 - (tab[c1].astype(np.float32) * s1[0]).astype(np.float32)).astype(np.float32))
