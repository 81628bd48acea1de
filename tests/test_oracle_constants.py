"""Pins P1: the oracle's constants against what the paper prints
(tests/golden/paper_constants.txt) and against Python big-integer re-derivations."""
import math
import os
from fractions import Fraction

import mpmath

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    g = {}
    for line in open(os.path.join(HERE, "golden", "paper_constants.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            g[k.strip()] = v.split()
    return g


def test_moduli_and_M(O):
    g = golden()
    mods = [int(x) for x in g["moduli"]]
    assert O.moduli() == mods
    M = math.prod(mods)
    assert O.M() == M
    assert M.bit_length() == int(g["bitlen_M"][0])
    assert round(math.log2(M), 2) == float(g["log2_M"][0])
    assert math.log2(M) > int(g["capacity_bits_required"][0])       # Eq. (2)
    assert 1 + math.log2(32) + 2 * (53 + 1) == int(g["capacity_bits_required"][0])
    for i, a in enumerate(mods):                                     # pairwise coprime
        for b in mods[i + 1:]:
            assert math.gcd(a, b) == 1
    assert M % 2 == 0                                                # M/2 is an integer (reading S11)


def test_rev33_set(O):
    g = golden()
    O.select_modset(1)
    try:
        mods = O.moduli()
        assert mods[:3] == [int(x) for x in g["moduli_rev33_replaced"]]
        assert round(math.log2(math.prod(mods)), 2) == float(g["log2_M_rev33"][0])
        assert math.log2(math.prod(mods)) < int(g["capacity_bits_required"][0])
    finally:
        O.select_modset(0)


def test_idempotents_and_slices(O):
    g = golden()
    mods, M = O.moduli(), O.M()
    S = O.num_slices()
    assert S == int(g["num_slices_S"][0]) == -(-M.bit_length() // 8)
    for k, m in enumerate(mods):
        u = O.u(k)
        assert 0 < u < M
        assert O.t_inv(k) == pow(M // m, -1, m)
        assert u == (M // m) * pow(M // m, -1, m)                     # Eq. (17)
        for j, mj in enumerate(mods):                                # u_k = delta_kj mod m_j
            assert u % mj == (1 if j == k else 0)
        assert sum(O.uslice(k, s) << (8 * s) for s in range(S)) == u  # Eq. (19)
        assert all(0 <= O.uslice(k, s) < 256 for s in range(S))


def test_lift_fractions(O):
    g = golden()
    f = int(g["frac_bits_f"][0])
    M = O.M()
    for k in range(12):
        w = O.w(k)
        assert w == math.floor(Fraction(2 ** f * O.u(k), M) + Fraction(1, 2))   # reading S10
        assert w < 2 ** f
        assert sum(O.wslice(k, s) << (8 * s) for s in range(int(g["num_frac_slices"][0]))) == w


def test_positional_bounds(O):
    g = golden()
    mods, M = O.moduli(), O.M()
    assert sum((m - 1) * O.u(k) for k, m in enumerate(mods)) == int(g["sum_canonical_bound_over_M"][0]) * M - 1
    tot = sum((2 * m - 1) * O.u(k) for k, m in enumerate(mods))
    assert tot == int(g["sum_signed_bound_over_M"][0]) * M - 1
    assert tot.bit_length() == int(g["raw_sum_magnitude_bits"][0])
    assert max(mods) - 1 == 2038 and 2038 * 255 == int(g["max_product"][0])
    assert 12 * 2038 * 255 == int(g["max_column_sum_fp16"][0]) < 2 ** 23
    # worst Phase-A column the oracle can actually produce
    vmax = [m - 1 for m in mods]
    P, Z = O.phaseA(vmax)
    assert max(P) <= int(g["max_column_sum_fp16"][0]) and max(Z) <= int(g["max_column_sum_fp16"][0])
    # two-limb shifted-column bound: v0 in [-128,128), v1 in [0,8]
    assert 12 * (128 * 255 + 8 * 255) == int(g["two_limb_column_sum"][0])


def test_twiddle_table(O):
    """Reading S5: RN(2^53 cos/sin) with exact symmetries; checked against mpmath at 200 digits."""
    mpmath.mp.dps = 60
    two53 = mpmath.mpf(2) ** 53
    mind = 1.0
    for t in range(1024):
        c, s = O.twiddle(t)
        th = 2 * mpmath.pi * t / 1024
        ec, es = two53 * mpmath.cos(th), two53 * mpmath.sin(th)
        assert c == int(mpmath.nint(ec)) and s == int(mpmath.nint(es)), t
        for e in (ec, es):
            fr = abs(e - mpmath.floor(e) - mpmath.mpf(0.5))
            mind = min(mind, float(fr))
        c2, s2 = O.twiddle((t + 512) % 1024)
        assert (c2, s2) == (-c, -s)
        c3, s3 = O.twiddle((1024 - t) % 1024)
        assert (c3, s3) == (c, -s)
    assert O.twiddle(0) == (2 ** 53, 0) and O.twiddle(256) == (0, 2 ** 53)
    assert mind > 2.0 ** -11          # no near-tie: generators with < 2^-11 abs error agree
