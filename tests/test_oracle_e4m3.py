"""Pin P1: the oracle's E4M3 codec against what the format definition fixes."""
import os

import numpy as np
import pytest

from oracle import e4m3

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_all_codes_roundtrip():
    t = e4m3.decode_table()
    for c in range(256):
        if c in (0x7F, 0xFF):
            assert np.isnan(t[c])
            assert e4m3.encode(np.float32(t[c]))[()] & 0x7F == 0x7F
        else:
            assert int(e4m3.encode(np.float32(t[c]))) == c, hex(c)


def test_value_table_closed_forms():
    t = e4m3.decode_table()
    pos = t[:0x7F]
    assert len(set(t[~np.isnan(t)].tolist())) == 253          # +-0 compare equal
    assert pos.max() == 448.0 and pos[1] == 2.0 ** -9 and pos[8] == 2.0 ** -6
    # sum of the 126 positive finite values: 11.5*sum_{e=1..15} 2^(e-7) - 480 + 28*2^-9
    closed = 11.5 * sum(2.0 ** (e - 7) for e in range(1, 16)) - 480 + 28 * 2.0 ** -9
    assert closed == 5407.875 and float(np.sum(pos)) == closed
    assert np.all(np.diff(pos) > 0)                            # codes order like magnitudes
    assert np.array_equal(t[0x80:0xFF], -t[0x00:0x7F])


def test_value_pins_from_golden():
    for line in open(os.path.join(GOLD, "e4m3_value_pins.txt")):
        if line.startswith("#") or not line.strip():
            continue
        expr, code = line.split()
        x = np.float32(eval(expr, {"inf": np.inf}))
        assert int(e4m3.encode(x)) == int(code, 16), (expr, hex(int(e4m3.encode(x))))


def test_midpoints_tie_to_even_and_neighbours():
    t = e4m3.decode_table()
    for c in range(0x7E):
        lo, hi = t[c], t[c + 1]
        mid = np.float32((lo + hi) / 2)          # exactly representable in fp32
        assert float(mid) == (lo + hi) / 2
        even = c if (c & 1) == 0 else c + 1
        assert int(e4m3.encode(mid)) == even
        assert int(e4m3.encode(np.nextafter(mid, np.float32(0)))) == c
        assert int(e4m3.encode(np.nextafter(mid, np.float32(1e9)))) == c + 1
        assert int(e4m3.encode(-mid)) == (even | 0x80)


def test_brute_force_nearest_value():
    """encode == argmin |x - v| over the finite values, ties to even code, saturating."""
    t = e4m3.decode_table()
    vals = t[:0x7F]
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.standard_normal(3000) * np.exp(rng.standard_normal(3000) * 4),
                        rng.uniform(-2.0 ** -5, 2.0 ** -5, 2000), rng.uniform(-600, 600, 2000)]).astype(np.float32)
    got = e4m3.encode(x)
    for xi, gi in zip(x, got):
        a = abs(float(xi))
        dist = np.abs(vals - a)
        best = np.flatnonzero(dist == dist.min())
        c = int(best[0]) if len(best) == 1 else int([b for b in best if b % 2 == 0][0])
        if np.signbit(xi):
            c |= 0x80
        assert int(gi) == c, (xi, hex(int(gi)), hex(c))


def test_matches_torch_cast_in_range():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(1_000_000) * np.exp(rng.standard_normal(1_000_000) * 3)).astype(np.float32)
    x = x[np.abs(x) <= 464]
    ours = e4m3.encode(x)
    theirs = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(ours, theirs)


def test_saturation_and_specials():
    x = np.array([464, 465, 1e9, np.inf, -464, -1e30, -np.inf], dtype=np.float32)
    assert e4m3.encode(x).tolist() == [0x7E, 0x7E, 0x7E, 0x7E, 0xFE, 0xFE, 0xFE]
    assert int(e4m3.encode(np.float32(np.nan))) & 0x7F == 0x7F
    assert int(e4m3.encode(np.float32(463.99))) == 0x7E
