"""Pins P2, P3, S10: CRT reconstruction, Kulisch deposits, lift."""
import random

import pytest


def centred(x, M):
    x %= M
    return x - M if x >= M // 2 else x


def test_crt_identity_random_and_boundary(O):
    M = O.M()
    mods = O.moduli()
    rng = random.Random(1234)
    cases = [0, 1, -1, M // 2 - 1, -(M // 2 - 1), -(M // 2), 2 ** 111, -(2 ** 111), 12345678901234567890123]
    cases += [rng.randrange(-(M // 2), M // 2) for _ in range(20000)]
    for Cv in cases:
        v = O.residues(Cv)
        assert v == [Cv % m for m in mods]                  # canonical residues (Appendix A.4)
        assert O.crt(v, 0) == Cv                            # Algorithm 2, two-sided
        assert O.crt(v, 1) == Cv                            # plain sum v_k u_k mod M
        assert O.crt(v, 2) == Cv                            # Garner mixed radix
    assert O.capacity_violations() == 0


def test_crt_arbitrary_residues_vs_bigint(O):
    """Random residue vectors (not derived from a C): compare with Python big-int CRT."""
    M, mods = O.M(), O.moduli()
    rng = random.Random(99)
    for _ in range(5000):
        v = [rng.randrange(m) for m in mods]
        E = sum(vk * O.u(k) for k, vk in enumerate(v))
        want = centred(E, M)
        assert O.crt(v, 0) == want and O.crt(v, 2) == want
        P, Z = O.phaseA(v)
        assert sum(p << (8 * s) for s, p in enumerate(P)) == E          # Eq. (19)
        assert sum(z << (8 * t) for t, z in enumerate(Z)) == sum(vk * O.w(k) for k, vk in enumerate(v))
        assert max(P) < 2 ** 23


def test_one_sided_lift_fails_somewhere_two_sided_never(O):
    """The failure class of PAPER.md:370 (T4): near |C| = M/2 the estimate zhat is off by one and a
    one-sided correction is wrong by exactly M; the two-sided correction is exact on the whole sweep.
    Canonical residues tip zhat one too small near -M/2 (lower-only test fails); centred residues, which
    the biased deposits admit (reading S12), tip it one too large at C = M/2 - 1 (upper-only test fails).
    The paper's own "10 units above a rounding boundary" figure is not reproducible (parity unpinned)."""
    M, mods = O.M(), O.moduli()
    rng = random.Random(4)
    offs = list(range(64)) + [rng.randrange(2 ** 70) for _ in range(300)]
    fails = {3: 0, 4: 0}
    for d in offs:
        for Cv in (-(M // 2) + d, M // 2 - 1 - d):
            canon = O.residues(Cv)
            cent = [r - m if r > m // 2 else r for r, m in zip(canon, mods)]
            for v in (canon, cent):
                assert O.crt(v, 0) == Cv
                for route in (3, 4):
                    got = O.crt(v, route)
                    if got != Cv:
                        assert abs(got - Cv) == M
                        fails[route] += 1
    assert fails[3] > 0 and fails[4] > 0
    assert O.capacity_violations() == 0


def test_kulisch_deposit_counterexample_and_random(O):
    """T3: P_0 = -1 must give E = -1; random signed slice sums vs big ints."""
    B_tot = sum(2 ** 23 << (8 * s) for s in range(15))

    def value(W):
        assert all(0 <= w < 2 ** 28 for w in W[:5])
        return sum(w << (28 * i) for i, w in enumerate(W)) - B_tot

    assert value(O.kulisch_deposit([-1] + [0] * 14)) == -1
    assert value(O.kulisch_deposit([0] * 15)) == 0
    rng = random.Random(7)
    for _ in range(5000):
        P = [rng.randrange(-(2 ** 23), 2 ** 23) for _ in range(15)]
        assert value(O.kulisch_deposit(P)) == sum(p << (8 * s) for s, p in enumerate(P))
    worst = [2 ** 23 - 1] * 15
    assert value(O.kulisch_deposit(worst)) == sum(p << (8 * s) for s, p in enumerate(worst))


def test_zhat_bounds(O):
    """Reading S9: canonical z <= 4359, so E = C + zM with the exact bounds of PAPER.md:74."""
    M, mods = O.M(), O.moduli()
    v = [m - 1 for m in mods]
    E = sum(vk * O.u(k) for k, vk in enumerate(v))
    assert E == 4360 * M - 1 and O.crt(v, 0) == -1


def test_rev33_dc_regression(O):
    """with the Rev-33 set a DC column (K=32 terms of 2^53 * (2^53-1)) exceeds M/2 and
    reconstructs wrong by exactly M; with Rev-34 it is exact."""
    R = 32 * (2 ** 53) * (2 ** 53 - 1)
    assert O.crt(O.residues(R), 0) == R
    O.select_modset(1)
    try:
        M33 = O.M()
        assert R > M33 // 2
        got = O.crt(O.residues(R), 0)
        assert got == R - M33
    finally:
        O.select_modset(0)
