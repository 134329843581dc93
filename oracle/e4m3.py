"""ORACLE (test infrastructure, not product code): the OCP FP8 E4M3 ("E4M3FN") codec.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2606_18502_b200/.

What the paper fixes: "FP8 (E4M3) weight-and-activation quantization (W8A8)" (PAPER.md:98,
section 3.2).  BASELINE.json:north_star adds "round-to-nearest-even with saturation".
The format itself is the OCP 8-bit floating point E4M3 definition restated here:
  1 sign bit, 4 exponent bits (bias 7), 3 mantissa bits; no infinities;
  NaN = S.1111.111 (0x7F / 0xFF); largest finite 448 = 0x7E;
  e == 0: value = (-1)^s * m * 2^-9  (subnormals, m = 0..7);
  e  > 0: value = (-1)^s * (1 + m/8) * 2^(e-7).
encode() is the definition "nearest representable value, ties to the even mantissa,
magnitudes beyond the largest finite saturate to +-448" (reading R-codec), which is
also what the hardware conversion cvt.rn.satfinite.e4m3x2.f32 does.

Pins (tests/test_oracle_e4m3.py): all 256 codes round-trip; value table checksum 5407.875
(closed form); every midpoint between adjacent values goes to the even mantissa; saturation;
agreement with torch's float8_e4m3fn CPU cast for |x| <= 464; a brute-force nearest-value
search over the 253 finite values.
"""
import numpy as np

E4M3_MAX = 448.0


def decode_table():
    """fp64 value of each of the 256 codes (NaN for 0x7F and 0xFF)."""
    t = np.empty(256, dtype=np.float64)
    for c in range(256):
        s = -1.0 if c & 0x80 else 1.0
        e = (c >> 3) & 0xF
        m = c & 0x7
        if e == 0xF and m == 0x7:
            t[c] = np.nan
        elif e == 0:
            t[c] = s * m * 2.0 ** -9
        else:
            t[c] = s * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return t


_TABLE = decode_table()


def decode(codes):
    """uint8 codes -> fp64 values (exact)."""
    return _TABLE[np.asarray(codes, dtype=np.uint8)]


def encode(x):
    """fp32 (or anything castable) -> uint8 E4M3 codes, RNE, saturate-to-finite.

    Step by step, per element, on the exact value of the fp32 input held in fp64:
      1. a = |x|;  binade exponent E = floor(log2 a) clamped below at -6 (the subnormal
         spacing equals the spacing of the first normal binade);
      2. spacing q = 2^(E-3); n = rint(a / q)  (a/q is exact; rint rounds half to even, and
         an even n is an even mantissa because q divides the binade into 8 steps);
      3. v = n*q, saturated to 448;  4. re-derive (e, m) from v (n == 16 carries into the next
         binade).
    """
    xf = np.asarray(x, dtype=np.float32)
    sign = np.signbit(xf)
    a = np.abs(xf).astype(np.float64)
    isnan = np.isnan(a)
    a = np.where(isnan, 0.0, np.minimum(a, 1.0e6))       # +-inf and huge -> saturate below
    _, ex = np.frexp(a)                                   # a = f * 2^ex, f in [0.5, 1)
    E = np.maximum(ex - 1, -6)
    q = np.ldexp(1.0, E - 3)
    v = np.minimum(np.rint(a / q) * q, E4M3_MAX)
    _, ev = np.frexp(v)
    Ev = ev - 1
    normal = v >= 2.0 ** -6
    m_norm = np.rint((v / np.ldexp(1.0, np.where(normal, Ev, 0)) - 1.0) * 8.0)
    code_norm = ((Ev + 7) << 3) + m_norm.astype(np.int64)
    code_sub = np.rint(v * 2.0 ** 9).astype(np.int64)
    code = np.where(normal, code_norm, code_sub)
    code = np.where(isnan, 0x7F, code)
    code = code | np.where(sign, 0x80, 0)
    return code.astype(np.uint8)
