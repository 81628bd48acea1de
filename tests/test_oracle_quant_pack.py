"""Pins P5, S2, S14: integer-only quantisation (Appendix A.3) and the correctly-rounded
pack (Appendix A.6) against exact rational arithmetic (fractions.Fraction / Python int->float RNE)."""
import math
import random
import struct
from fractions import Fraction


def bits_of(x):
    return struct.unpack("<Q", struct.pack("<d", x))[0]


def float_of(b):
    return struct.unpack("<d", struct.pack("<Q", b))[0]


def rne_fraction(fr):
    """Round a Fraction to the nearest integer, ties to even."""
    fl = math.floor(fr)
    rem = fr - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2):
        return fl + 1
    return fl


def exact_round_to_double(num, g):
    """RNE_fp64(num * 2^-g) by rational arithmetic, returns the bit pattern."""
    if num == 0:
        return 0
    sgn = (1 << 63) if num < 0 else 0
    a = abs(num)
    v = Fraction(a, 1) / Fraction(2) ** g if g >= 0 else Fraction(a * 2 ** (-g), 1)
    e = a.bit_length() - 1 - g                     # floor(log2 v)
    if e < -1022:
        q = rne_fraction(v * Fraction(2) ** 1074)
        return sgn | q
    q = rne_fraction(v / Fraction(2) ** (e - 52))
    if q == 2 ** 53:
        q, e = 2 ** 52, e + 1
    if e > 1023:
        return sgn | 0x7FF0000000000000
    return sgn | ((e + 1023) << 52) | (q - 2 ** 52)


def test_pack_matches_python_float_in_normal_range(O):
    rng = random.Random(5)
    for _ in range(20000):
        nb = rng.randrange(1, 118)
        R = rng.randrange(-(2 ** nb), 2 ** nb)
        g = rng.randrange(60, 180)
        want = bits_of(math.ldexp(float(R), -g)) if R else 0   # int->float is RNE; ldexp exact here
        assert O.pack(R, g) == want


def test_pack_ties_and_carry(O):
    for L in (54, 60, 100, 117):
        base = 1 << (L - 1)
        for q_low in (0, 1):                     # even / odd kept significand
            top = base | (q_low << (L - 53))
            half = 1 << (L - 54)
            for delta in (-1, 0, 1):
                R = top + half + delta
                for sg in (1, -1):
                    assert O.pack(sg * R, 70) == exact_round_to_double(sg * R, 70)
        allones = (1 << L) - 1                   # rounds up into the next binade
        assert O.pack(allones, 64) == exact_round_to_double(allones, 64)
        assert float_of(O.pack(allones, 64)) == math.ldexp(1.0, L - 64)
    assert O.pack(0, 100) == 0                   # +0.0 (reading S14)


def test_pack_subnormal_overflow(O):
    rng = random.Random(6)
    for _ in range(5000):
        nb = rng.randrange(1, 118)
        R = rng.randrange(-(2 ** nb), 2 ** nb)
        g = rng.randrange(1000, 1250)            # results straddle 2^-1022 and 2^-1074
        assert O.pack(R, g) == exact_round_to_double(R, g)
    # single rounding into the subnormal grid (never round to 53 bits first)
    R = (1 << 60) + (1 << 7) + 1                 # 53-bit rounding would land on a tie of the coarser grid
    for g in range(1074 + 1, 1074 + 70):
        assert O.pack(R, g) == exact_round_to_double(R, g)
    assert O.pack(1, 1075) == 0 and O.pack(3, 1075) == 2      # ties to even at the bottom
    assert O.pack(1 << 100, -930) == 0x7FF0000000000000       # overflow -> +inf
    assert O.pack(-(1 << 100), -930) == 0xFFF0000000000000


def test_quantise_vs_rational(O):
    rng = random.Random(8)
    for _ in range(20000):
        x = rng.choice([1.0, -1.0]) * rng.random() * 2.0 ** rng.randrange(-40, 40)
        tmax = math.frexp(x)[1] - 1 + rng.choice([0, 0, 1, 2, 10, 30, 52, 53, 54, 55, 60, 70])
        want = rne_fraction(Fraction(x) * Fraction(2) ** (52 - tmax)) if tmax <= 52 else \
            rne_fraction(Fraction(x) / Fraction(2) ** (tmax - 52))
        assert O.quantise(bits_of(x), tmax) == want
        assert abs(want) <= 2 ** 53 - 1 or abs(want) == 2 ** 53 - 0 and False


def test_quantise_shift_edge_cases(O):
    m = (1 << 53) - 1                             # all-ones significand, value m * 2^-52 in [1,2)
    x = math.ldexp(float(m), -52)
    assert O.quantise(bits_of(x), 0) == m         # sh = 0
    for sh in (1, 2, 52, 53, 54, 55, 63, 64, 100):
        want = rne_fraction(Fraction(m, 2 ** sh))
        assert O.quantise(bits_of(x), sh) == want
        assert O.quantise(bits_of(-x), sh) == -want
    assert O.quantise(bits_of(1.0), 53) == 0      # exactly 1/2 -> 0 (ties to even)
    assert O.quantise(bits_of(1.5), 53) == 1
    assert O.quantise(bits_of(1.0), 52) == 1      # 1/2 ... sh=52: 2^52 >> 52 = 1
    assert O.quantise(bits_of(3.0), 53) == 2      # 1.5 -> 2
    assert O.quantise(bits_of(0.0), 5) == 0 and O.quantise(bits_of(-0.0), 5) == 0


def test_quantise_subnormals_and_column_top(O):
    tiny = 5e-324                                  # 2^-1074
    sub = 12345 * tiny
    st, t = O.column_top([bits_of(sub), bits_of(tiny), bits_of(0.0)])
    assert st == 1 and t == -1074 + (12345).bit_length() - 1
    assert O.quantise(bits_of(sub), t) == 12345 << (52 - ((12345).bit_length() - 1))   # exact left shift
    assert O.quantise(bits_of(tiny), t) == 1 << (52 - ((12345).bit_length() - 1))
    st, t = O.column_top([bits_of(3.0), bits_of(-1e-300), bits_of(0.75)])
    assert (st, t) == (1, 1)
    assert O.column_top([0, 1 << 63])[0] == 0                                             # all zero
    assert O.column_top([bits_of(1.0), bits_of(float("inf"))])[0] == 2                     # non-finite
    assert O.column_top([bits_of(float("nan"))])[0] == 2
    # a normal next to a subnormal: generic shift rule
    st, t = O.column_top([bits_of(2.0 ** -1020), bits_of(sub)])
    assert t == -1020
    want = rne_fraction(Fraction(12345, 2 ** 1074) * Fraction(2) ** (52 + 1020))
    assert O.quantise(bits_of(sub), t) == want
