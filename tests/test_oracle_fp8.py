"""Pins for the oracle's FP8 codecs, quantizer and reduce (O4, O5).  CPU only.

Each pin compares the oracle with something that is NOT the oracle: the format constants printed
in ref [24] (tests/golden/fp8_formats.txt), torch's own float8 dtypes (an independent library
implementation; in range only -- torch does not saturate), order/rounding properties that follow
from the definition of round-to-nearest-even, and numpy arithmetic for the reduce."""
import os

import numpy as np
import pytest
import torch

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden", "fp8_formats.txt")
FMTS = [(oracle.E4M3, "E4M3", torch.float8_e4m3fn), (oracle.E5M2, "E5M2", torch.float8_e5m2)]


def _golden():
    g = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if not line:
            continue
        f, key, *vals = line.split()
        g[(f, key)] = vals
    return g


@pytest.mark.parametrize("fmt,name,tdt", FMTS)
def test_printed_format_constants(fmt, name, tdt):
    g = _golden()
    tab = oracle.fp8_table(fmt)
    pos = tab[:128]
    finite = pos[np.isfinite(pos)]
    p = 3 if fmt == oracle.E4M3 else 2
    assert finite.max() == float(g[(name, "max_normal")][0]) == oracle.fp8_max(fmt)
    assert tab[1 << p] == float(g[(name, "min_normal")][0])
    assert tab[(1 << p) - 1] == float(g[(name, "max_subnormal")][0])
    assert tab[1] == float(g[(name, "min_subnormal")][0])
    if name == "E4M3":
        assert np.isnan(tab[int(g[(name, "nan_code")][0], 16)]) and np.isnan(tab[0xFF])
        assert not np.isinf(tab).any() and np.isnan(tab).sum() == 2
    else:
        assert np.isposinf(tab[int(g[(name, "inf_code")][0], 16)]) and np.isneginf(tab[0xFC])
        for c in g[(name, "nan_codes")]:
            assert np.isnan(tab[int(c, 16)])
        assert np.isnan(tab).sum() == 6


@pytest.mark.parametrize("fmt,name,tdt", FMTS)
def test_decode_table_matches_torch_float8(fmt, name, tdt):
    tab = oracle.fp8_table(fmt)
    ref = torch.arange(256, dtype=torch.uint8).view(tdt).to(torch.float64).numpy()
    assert np.array_equal(np.isnan(tab), np.isnan(ref))
    ok = ~np.isnan(tab)
    assert np.array_equal(tab[ok], ref[ok])
    assert np.array_equal(np.signbit(tab[ok]), np.signbit(ref[ok]))      # -0 keeps its sign


@pytest.mark.parametrize("fmt,name,tdt", FMTS)
def test_encode_roundtrip_monotone_midpoints_saturation(fmt, name, tdt):
    tab = oracle.fp8_table(fmt)
    # encode(decode(c)) == c for every finite code (including -0)
    for c in range(256):
        if np.isfinite(tab[c]):
            assert oracle.fp8_from_float(fmt, tab[c]) == c
    pos_codes = [c for c in range(128) if np.isfinite(tab[c])]
    vals = tab[pos_codes]
    assert np.all(np.diff(vals) > 0)                                    # codes ordered like values
    # every midpoint between neighbours goes to the even mantissa; just inside goes to the nearer
    for a, b in zip(pos_codes[:-1], pos_codes[1:]):
        mid = 0.5 * (tab[a] + tab[b])
        assert np.float32(mid) == mid
        even = a if a % 2 == 0 else b
        assert oracle.fp8_from_float(fmt, mid) == even
        assert oracle.fp8_from_float(fmt, -mid) == (even | 0x80)
        lo = np.nextafter(np.float32(mid), np.float32(0))
        hi = np.nextafter(np.float32(mid), np.float32(np.inf))
        assert oracle.fp8_from_float(fmt, lo) == a
        assert oracle.fp8_from_float(fmt, hi) == b
    # saturation: anything above max finite, the half step above it, and infinity -> +-max finite
    cmax = pos_codes[-1]
    step = tab[cmax] - tab[cmax - 1]
    for y in [tab[cmax] + step / 2, tab[cmax] + step, np.nextafter(np.float32(tab[cmax]), np.float32(np.inf)),
              1e30, np.inf]:
        assert oracle.fp8_from_float(fmt, y) == cmax
        assert oracle.fp8_from_float(fmt, -y) == (cmax | 0x80)
    assert np.isnan(tab[oracle.fp8_from_float(fmt, np.nan)])
    assert oracle.fp8_from_float(fmt, 0.0) == 0 and oracle.fp8_from_float(fmt, -0.0) == 0x80
    # below half the smallest subnormal -> zero; exactly half -> zero (tie to even)
    assert oracle.fp8_from_float(fmt, tab[1] / 2) == 0
    assert oracle.fp8_from_float(fmt, np.nextafter(np.float32(tab[1] / 2), np.float32(1))) == 1


@pytest.mark.parametrize("fmt,name,tdt", FMTS)
def test_encode_matches_torch_in_range(fmt, name, tdt):
    rng = np.random.default_rng(5)
    fmax = oracle.fp8_max(fmt)
    y = np.concatenate([rng.uniform(-fmax, fmax, 20000), rng.normal(0, 1, 20000),
                        rng.normal(0, 1e-3, 20000), rng.normal(0, 1e-6, 5000)]).astype(np.float32)
    y = y[np.abs(y) <= fmax]
    want = torch.from_numpy(y).to(tdt).view(torch.uint8).numpy()
    got = np.array([oracle.fp8_from_float(fmt, v) for v in y], dtype=np.uint8)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("fmt,name,tdt", FMTS)
@pytest.mark.parametrize("scaling", [oracle.SCALE_TENSOR, oracle.SCALE_BLOCK128])
def test_quantizer_properties(fmt, name, tdt, scaling):
    rng = np.random.default_rng(11)
    m, n = 200, 300                                                  # ragged against 128 x 128 blocks
    x = (rng.normal(0, 1, (m, n)) * np.exp(rng.normal(0, 2, (m, n)))).astype(np.float32)
    codes, sinv = oracle.quantize(x, fmt, scaling)
    tab = oracle.fp8_table(fmt)
    fmax = oracle.fp8_max(fmt)
    assert sinv.shape == (oracle.n_scales(scaling, m, n),)
    bn = (n + 127) // 128
    for bi in range((m + 127) // 128 if scaling else 1):
        for bj in range(bn if scaling else 1):
            sl = (slice(bi * 128, bi * 128 + 128), slice(bj * 128, bj * 128 + 128)) if scaling else (slice(None),) * 2
            xb, cb = x[sl], codes[sl]
            s_inv = sinv[bi * bn + bj if scaling else 0]
            amax = np.abs(xb).max()
            assert s_inv == np.float32(amax) / np.float32(fmax)
            # the largest element lands on +-fmax
            i = np.unravel_index(np.abs(xb).argmax(), xb.shape)
            assert abs(tab[cb[i]]) == fmax
            # per element: the code is a nearest representable value of y = x * scale
            y = (xb * (np.float32(fmax) / np.float32(amax))).astype(np.float32).astype(np.float64)
            v = tab[cb]
            assert np.all(np.isfinite(v)) and np.all(np.sign(v) * np.sign(y) >= 0)
            pos = np.sort(tab[:128][np.isfinite(tab[:128])])
            ay = np.minimum(np.abs(y), fmax)
            idx = np.clip(np.searchsorted(pos, ay), 1, len(pos) - 1)
            half_step = 0.5 * (pos[idx] - pos[idx - 1])
            assert np.all(np.abs(np.abs(v) - ay) <= half_step * (1 + 1e-12))


def test_quantizer_degenerate_inputs():
    z = np.zeros((5, 7), np.float32)
    for fmt in (oracle.E4M3, oracle.E5M2):
        codes, sinv = oracle.quantize(z, fmt)
        assert not codes.any() and sinv[0] == 1.0
        x = np.array([[1e-44, -1e-45]], np.float32)                  # scale = fmax/amax overflows
        codes, sinv = oracle.quantize(x, fmt)
        assert sinv[0] == 1.0 and not (codes & 0x7F).any()
        x = np.array([[1.0, np.nan, -np.inf, 3.0]], np.float32)     # non-finite => scale 1, NaN code
        codes, sinv = oracle.quantize(x, fmt)
        tab = oracle.fp8_table(fmt)
        assert sinv[0] == 1.0 and tab[codes[0, 0]] == 1.0 and np.isnan(tab[codes[0, 1]])
        assert tab[codes[0, 2]] == -oracle.fp8_max(fmt) and tab[codes[0, 3]] == 3.0


@pytest.mark.parametrize("scaling", [oracle.SCALE_TENSOR, oracle.SCALE_BLOCK128])
def test_reduce_is_mean_of_dequantised_payloads(scaling):
    rng = np.random.default_rng(3)
    m, n, R = 130, 260, 4
    payloads = [oracle.quantize(rng.normal(0, 1 + r, (m, n)).astype(np.float32), oracle.E4M3, scaling)
                for r in range(R)]
    cs, ss = [p[0] for p in payloads], [p[1] for p in payloads]
    out = oracle.reduce(cs, ss, oracle.E4M3, scaling, average=True)
    tab = oracle.fp8_table(oracle.E4M3)
    bn = (n + 127) // 128

    def expand(s):
        if scaling == oracle.SCALE_TENSOR:
            return np.full((m, n), s[0], np.float64)
        g = s.reshape((m + 127) // 128, bn).astype(np.float64)
        return np.kron(g, np.ones((128, 128)))[:m, :n]

    exact = sum(tab[c] * expand(s) for c, s in zip(cs, ss)) / R           # float64 mean
    assert np.abs(out - exact).max() <= 4 * np.finfo(np.float32).eps * np.abs(exact).max()
    # R = 1, no averaging == plain dequantisation, exactly (one FP32 product)
    one = oracle.reduce(cs[:1], ss[:1], oracle.E4M3, scaling, average=False)
    assert np.array_equal(one, (tab[cs[0]].astype(np.float32) * expand(ss[0]).astype(np.float32)))
    # rank order is part of the definition: it is what a left-to-right FP32 fma chain gives
    acc = np.zeros((m, n), np.float64)
    for c, s in zip(cs, ss):                                             # emulate fmaf: exact product+sum, one rounding
        acc = (tab[c] * expand(s) + acc).astype(np.float32).astype(np.float64)
    assert np.array_equal(out, (acc.astype(np.float32) * np.float32(1.0 / R)))


def test_bf16_conversion_matches_torch():
    rng = np.random.default_rng(9)
    x = np.concatenate([rng.normal(0, 1, 50000), rng.normal(0, 1e-30, 1000), [0.0, -0.0, 1.0, 3.3895314e38,
                       1.00390625, 1.01171875]]).astype(np.float32)
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = oracle.to_bf16_bits(x.astype(np.float64))
    assert np.array_equal(got, want)
    back = oracle.from_bf16_bits(got)
    assert np.array_equal(back, torch.from_numpy(x).to(torch.bfloat16).double().numpy())
