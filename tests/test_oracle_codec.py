"""Pins for the oracle's E4M3 codec and quantiser (O1, O2) -- CPU only."""
import os

import numpy as np
import torch

from oracle import spense_oracle as o


def _read_golden(golden_dir):
    vals, rounds = [], []
    with open(os.path.join(golden_dir, "e4m3_fixed_points.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            t = line.split()
            if t[0] == "R":
                rounds.append((float(t[1]), int(t[2], 16)))
            else:
                vals.append((int(t[0], 16), float(t[1])))
    return vals, rounds


def test_decode_golden_fixed_points(golden_dir):
    vals, _ = _read_golden(golden_dir)
    for b, v in vals:
        d = o.e4m3_decode(np.array([b], dtype=np.uint8))[0]
        assert d == v and np.signbit(d) == np.signbit(v), (hex(b), d, v)


def test_encode_golden_midpoints(golden_dir):
    _, rounds = _read_golden(golden_dir)
    for x, b in rounds:
        assert o.e4m3_encode(np.array([x], dtype=np.float32))[0] == b, (x, hex(b))


def test_decode_all_256_vs_torch_and_ml_dtypes():
    import ml_dtypes
    b = np.arange(256, dtype=np.uint8)
    d = o.e4m3_decode(b)
    t = torch.from_numpy(b.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    m = b.view(ml_dtypes.float8_e4m3fn).astype(np.float64)
    for ref in (t, m):
        assert np.array_equal(np.isnan(d), np.isnan(ref))
        ok = ~np.isnan(d)
        assert np.array_equal(d[ok], ref[ok])
        assert np.array_equal(np.signbit(d[ok]), np.signbit(ref[ok]))
    assert np.isnan(d[0x7F]) and np.isnan(d[0xFF]) and np.isnan(d).sum() == 2


def test_encode_roundtrip_all_finite_bytes():
    b = np.array([v for v in range(256) if (v & 0x7F) != 0x7F], dtype=np.uint8)
    assert np.array_equal(o.e4m3_encode(o.e4m3_decode(b).astype(np.float32)), b)


def test_encode_every_midpoint_ties_to_even():
    # brute force over the grid: midpoint between adjacent non-negative grid values
    pos = np.array(sorted(set(o.e4m3_decode(np.arange(0, 0x7F, dtype=np.uint8)).tolist())))
    for lo, hi in zip(pos[:-1], pos[1:]):
        mid = np.float32((lo + hi) / 2)
        assert float(mid) == (lo + hi) / 2     # midpoints are exact in fp32
        blo = o.e4m3_encode(np.array([lo], np.float32))[0]
        bhi = o.e4m3_encode(np.array([hi], np.float32))[0]
        want = blo if (blo & 1) == 0 else bhi
        assert o.e4m3_encode(np.array([mid]))[0] == want
        assert o.e4m3_encode(np.array([-mid]))[0] == (want | 0x80)
        # just off the midpoint goes to the nearer neighbour
        assert o.e4m3_encode(np.array([np.nextafter(mid, np.float32(0))]))[0] == blo
        assert o.e4m3_encode(np.array([np.nextafter(mid, np.float32(1e9))]))[0] == bhi


def test_encode_dense_sweep_vs_torch_clamped_cast():
    rng = np.random.default_rng(1)
    # 4M random fp32 bit patterns (all exponents incl. subnormal/inf) + 4M in the E4M3 range
    bits = rng.integers(0, 2**32, size=4_000_000, dtype=np.uint64).astype(np.uint32)
    x1 = bits.view(np.float32)
    x1 = x1[~np.isnan(x1)]
    x2 = (rng.standard_normal(4_000_000) * np.exp(rng.uniform(-8, 7, 4_000_000))).astype(np.float32)
    for x in (x1, x2):
        ref = torch.clamp(torch.from_numpy(x.copy()), -448, 448).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
        got = o.e4m3_encode(x)
        assert np.array_equal(got, ref)


def test_encode_nan_and_saturation():
    x = np.array([np.nan, np.inf, -np.inf, 448.0, 449.0, 1e30], dtype=np.float32)
    got = o.e4m3_encode(x)
    assert (got[0] & 0x7F) == 0x7F
    assert list(got[1:]) == [0x7E, 0xFE, 0x7E, 0x7E, 0x7E]


def test_quantize_closed_forms():
    # powers of two: amax = 448 -> scale exactly 1 -> bytes are the exact codes
    x = np.array([[448.0, 1.0, -2.0, 0.5], [0.0, 0.0, 0.0, 0.0]], dtype=np.float32)
    q, s = o.quantize_per_tensor(x)
    assert s == np.float32(1.0)
    assert list(q[0]) == [0x7E, 0x38, 0xC0, 0x30] and list(q[1]) == [0, 0, 0, 0]
    q, s = o.quantize_per_row(x)
    assert s[0] == np.float32(1.0) and s[1] == np.float32(1.0)     # all-zero row -> scale 1
    # amax element always maps to +-0x7E; scaling the input by 2^k scales s by 2^k, same bytes
    rng = np.random.default_rng(0)
    y = rng.standard_normal((5, 64)).astype(np.float32)
    q1, s1 = o.quantize_per_row(y)
    q2, s2 = o.quantize_per_row(y * np.float32(8))
    assert np.array_equal(q1, q2) and np.array_equal(s2, s1 * np.float32(8))
    am = np.argmax(np.abs(y), axis=1)
    assert all((q1[r, am[r]] & 0x7F) == 0x7E for r in range(5))
    qt, st = o.quantize_per_tensor(y)
    assert st == np.float32(np.abs(y).max() / np.float32(448))
    assert np.array_equal(qt, o.e4m3_encode(y / st))
