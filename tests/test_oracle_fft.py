"""Pins P4, P6-P12: the stage and the 1-D / 3-D transforms of the oracle."""
import mpmath
import numpy as np
import pytest

from paper_2606_23698_b200 import inputs


def bits(a):
    return np.ascontiguousarray(a).view(np.uint64)


def test_stage_matches_python_bigint_definition(O):
    """The stage definition re-derived with Python big ints and Fraction-free integer rounding:
    a dropped term, wrong sign or transposed index in oz_stage fails here."""
    rng = np.random.default_rng(3)
    for K in (2, 4, 16, 32):
        x = (rng.standard_normal(K) + 1j * rng.standard_normal(K)) * 2.0 ** rng.integers(-8, 8, K)
        tidx = np.array([[(1024 // K) * j * k % 1024 for j in range(K)] for k in range(K)], dtype=np.int32)
        for sign in (-1, 1):
            y, bad = O.stage(x, tidx.reshape(-1), sign, K, K, route=2)
            assert bad == 0
            st, tmax = O.column_top([int(b) for b in bits(x)])
            xr = [O.quantise(int(b), tmax) for b in bits(x)[0::2]]
            xi = [O.quantise(int(b), tmax) for b in bits(x)[1::2]]
            g = 53 + 52 - tmax
            for k in range(K):
                R = I = 0
                for j in range(K):
                    c, s = O.twiddle(int(tidx[k, j]))
                    ar, ai = c, sign * s
                    R += ar * xr[j] - ai * xi[j]
                    I += ar * xi[j] + ai * xr[j]
                assert int(bits(y)[2 * k]) == O.pack(R, g)
                assert int(bits(y)[2 * k + 1]) == O.pack(I, g)
                assert np.float64(y[k].real) == np.float64(np.ldexp(float(R), -g))


def test_capacity_worst_case_below_half_M(O):
    """P4: all-ones significands against the k=0 row and against a 45-degree row stay below M/2."""
    O.reset_capacity_violations()
    K = 32
    big = np.ldexp(float(2 ** 53 - 1), -52)
    x = np.full(K, big + 1j * big)
    x[1::2] *= 1                                   # DC
    tidx0 = np.zeros((K, K), dtype=np.int32)
    y, bad = O.stage(x, tidx0.reshape(-1), -1, K, K, route=2)
    assert bad == 0
    x45 = np.full(K, big - 1j * big)               # re - im: aligns with the (c, -s) of a 45-degree twiddle
    tidx45 = np.full((K, K), 128, dtype=np.int32)
    y, bad = O.stage(x45, tidx45.reshape(-1), -1, K, K, route=2)
    assert bad == 0
    assert O.capacity_violations() == 0
    c, s = O.twiddle(128)
    worst = K * (c + s) * (2 ** 53 - 1)
    assert 2 ** 111 < worst < O.M() // 2           # 2^111.5, 5.4 bits under M/2 (reading S4)


@pytest.mark.parametrize("n", [2, 8, 32, 64, 128, 512, 1024])
def test_fft1d_residue_route_equals_direct_and_f128(O, n):
    """P6 + P9: residue/CRT/Kulisch route == __int128 definition bit-for-bit; <= 5e-15 vs __float128 DFT."""
    batch = 4 if n >= 512 else 16
    x = inputs.uniform_pm1((batch, n), seed=10 + n)
    O.reset_capacity_violations()
    y, bad = O.fft1d(x, -1, route=2)
    assert bad == 0 and O.capacity_violations() == 0
    assert O.relerr_1d_f128(x, y, -1) <= 5e-15
    ref = np.fft.fft(x, axis=-1)                   # P12 sanity vs a library FFT
    assert np.linalg.norm(y - ref) / np.linalg.norm(ref) < 1e-14
    yi, bad = O.fft1d(y, +1, route=2)
    assert bad == 0
    assert np.linalg.norm(yi / n - x) / np.linalg.norm(x) < 5e-15       # P10 round trip


def test_f128_reference_against_mpmath(O):
    """The __float128 DFT used as accuracy reference is itself pinned to mpmath (50 digits)."""
    mpmath.mp.dps = 50
    n = 16
    x = inputs.uniform_pm1((1, n), seed=77)
    Y = []
    for k in range(n):
        acc = mpmath.mpc(0)
        for j in range(n):
            acc += mpmath.mpc(float(x[0, j].real), float(x[0, j].imag)) * mpmath.expj(-2 * mpmath.pi * j * k / n)
        Y.append(complex(acc))
    Y = np.array(Y).reshape(1, n)
    assert O.relerr_1d_f128(x, Y, -1) < 3e-16      # Y is the exact DFT rounded to double
    assert O.relerr_1d_f128(x, Y * (1 + 1e-12), -1) == pytest.approx(1e-12, rel=1e-3)
    assert O.relerr_1d_f128(x, np.conj(Y), -1) > 0.1


@pytest.mark.parametrize("n", [32, 64, 1024])
def test_closed_forms_bit_exact(O, n):
    """P7: impulse -> all ones; constant -> n at k=0 and exactly 0 elsewhere, bit for bit."""
    imp = np.zeros((1, n), dtype=np.complex128); imp[0, 0] = 1.0
    y, _ = O.fft1d(imp, -1)
    assert np.array_equal(bits(y), bits(np.ones((1, n), dtype=np.complex128)))
    dc = np.ones((1, n), dtype=np.complex128)
    y, _ = O.fft1d(dc, -1)
    want = np.zeros((1, n), dtype=np.complex128); want[0, 0] = n
    assert np.array_equal(bits(y), bits(want))
    # shifted impulse: |Y_k| = 1 to within an ulp or two, phase -2 pi j k / n
    sh = np.zeros((1, n), dtype=np.complex128); sh[0, 3] = 1.0
    y, _ = O.fft1d(sh, -1)
    ph = np.array([O.twiddle((1024 // n) * ((3 * k) % n)) for k in range(n)], dtype=np.float64) / 2.0 ** 53
    assert np.abs(y[0] - (ph[:, 0] - 1j * ph[:, 1])).max() < 4e-16
    if n <= 32:                                    # single stage: exactly the rounded table entry
        assert np.array_equal(y[0].real, ph[:, 0]) and np.array_equal(y[0].imag, -ph[:, 1])


@pytest.mark.parametrize("n", [32, 256, 1024])
def test_exact_symmetries(O, n):
    """P8: power-of-two scaling, negation, conjugation and Hermitian symmetry hold exactly
    (value equality: an exact zero is always +0.0, reading S14)."""
    x = inputs.normal((3, n), seed=5)
    y, _ = O.fft1d(x, -1)
    y2, _ = O.fft1d(x * 2.0 ** 17, -1)
    assert np.array_equal(y2, y * 2.0 ** 17)
    yn, _ = O.fft1d(-x, -1)
    assert np.array_equal(yn, -y)
    yc, _ = O.fft1d(np.conj(x), +1)
    assert np.array_equal(yc, np.conj(y))
    xr = np.ascontiguousarray(x.real).astype(np.complex128)
    yr, _ = O.fft1d(xr, -1)
    k = np.arange(n)
    assert np.array_equal(yr[:, (-k) % n], np.conj(yr))


def test_single_frequency_and_parseval(O):
    """P10, P11."""
    n = 1024
    j = np.arange(n)
    x = np.exp(2j * np.pi * 37 * j / n).reshape(1, n)
    y, _ = O.fft1d(x, -1)
    want = np.zeros(n, dtype=np.complex128); want[37] = n
    assert np.abs(y[0] - want).max() < 64 * n * 2.2e-16
    x = inputs.normal((8, n), seed=21)
    y, _ = O.fft1d(x, -1)
    lhs = np.sum(np.abs(y).astype(np.longdouble) ** 2)
    rhs = n * np.sum(np.abs(x).astype(np.longdouble) ** 2)
    assert abs(lhs - rhs) / rhs < 1e-14
    # wide dynamic range, cancellation-heavy: alternating +-1 plus tiny noise
    x = (np.where(j % 2 == 0, 1.0, -1.0) + 2.0 ** -40 * inputs.uniform_pm1((1, n), seed=3).real).astype(np.complex128).reshape(1, n)
    y, bad = O.fft1d(x, -1, route=2)
    assert bad == 0 and O.relerr_1d_f128(x, y, -1) < 5e-15


def test_fft3d_small_full_checks(O):
    """3-D: routes agree; closed forms; <= 5e-15 vs the __float128 DFT on every output of 8x16x4 and on
    sampled outputs of config 1 (32^3, uniform, seed 0)."""
    x = inputs.uniform_pm1((8, 16, 4), seed=1)
    O.reset_capacity_violations()
    y, bad = O.fft3d(x, -1, route=2)
    assert bad == 0 and O.capacity_violations() == 0
    idx = np.arange(x.size, dtype=np.int64)
    assert O.relerr_3d_f128(x, idx, y.reshape(-1), -1) <= 5e-15
    ref = np.fft.fftn(x)
    assert np.linalg.norm(y - ref) / np.linalg.norm(ref) < 1e-14
    # axis order/layout: a transposed index would break the separable closed form below
    imp = np.zeros((8, 16, 4), dtype=np.complex128); imp[1, 2, 3] = 1.0
    yi, _ = O.fft3d(imp, -1)
    kx, ky, kz = np.meshgrid(np.arange(8), np.arange(16), np.arange(4), indexing="ij")
    want = np.exp(-2j * np.pi * (((2 * kx + 2 * ky + 12 * kz) % 16) / 16))
    assert np.abs(yi - want).max() < 1e-15
    dc = np.ones((32, 32, 32), dtype=np.complex128)
    yd, _ = O.fft3d(dc, -1)
    want = np.zeros_like(dc); want[0, 0, 0] = 32 ** 3
    assert np.array_equal(bits(yd), bits(want))
    x1 = inputs.uniform_pm1((32, 32, 32), seed=0)          # config 1
    y1, _ = O.fft3d(x1, -1)
    rng = np.random.default_rng(0)
    idx = rng.choice(x1.size, 64, replace=False).astype(np.int64)
    assert O.relerr_3d_f128(x1, idx, y1.reshape(-1)[idx], -1) <= 5e-15
    back, _ = O.fft3d(y1, +1)
    assert np.linalg.norm(back / x1.size - x1) / np.linalg.norm(x1) < 5e-15


def test_fft3d_two_stage_axes_pinned(O):
    """3-D with two-stage axes (n > 32: q = 32 first stage, p = n/32 twiddle-fused second stage, PAPER.md:115-124,
    210-214) on 64 x 32 x 64, residue route (route 2): (i) bit-identical to composing the 1-D transform (itself pinned
    to the __float128 DFT above) along z, y, x with the array rounded to fp64 between passes (reading
    S6) -- a wrong stride, axis order or stage index in the 3-D driver fails here; (ii) <= 5e-15 against the
    __float128 3-D DFT on 512 sampled outputs; (iii) closed forms: off-origin impulse, DC."""
    shape = (64, 32, 64)
    x = inputs.uniform_pm1(shape, seed=5)
    O.reset_capacity_violations()
    y, bad = O.fft3d(x, -1, route=2)
    assert bad == 0 and O.capacity_violations() == 0
    comp = x
    for axis in (2, 1, 0):
        moved = np.ascontiguousarray(np.moveaxis(comp, axis, -1))
        t, bad1 = O.fft1d(moved.reshape(-1, shape[axis]), -1, route=0)
        assert bad1 == 0
        comp = np.ascontiguousarray(np.moveaxis(t.reshape(moved.shape), -1, axis))
    assert np.array_equal(bits(y), bits(comp))
    rng = np.random.default_rng(1)
    idx = np.sort(rng.choice(x.size, 512, replace=False)).astype(np.int64)
    assert O.relerr_3d_f128(x, idx, y.reshape(-1)[idx], -1) <= 5e-15
    yi, _ = O.fft3d(y, +1, route=0)
    assert np.linalg.norm(yi / x.size - x) / np.linalg.norm(x) < 5e-15
    imp = np.zeros(shape, dtype=np.complex128); imp[5, 3, 41] = 1.0
    yimp, _ = O.fft3d(imp, -1)
    kx, ky, kz = np.meshgrid(np.arange(64), np.arange(32), np.arange(64), indexing="ij")
    want = np.exp(-2j * np.pi * (((5 * kx + 6 * ky + 41 * kz) % 64) / 64))
    assert np.abs(yimp - want).max() < 1e-15
    yd, _ = O.fft3d(np.ones(shape, dtype=np.complex128), -1)
    want = np.zeros(shape, dtype=np.complex128); want[0, 0, 0] = x.size
    assert np.array_equal(bits(yd), bits(want))


def test_lograng_dynamic_range_config2_slice(O):
    """Config 2's distribution (|x| log-uniform in 2^+-30) on a 1-D batch: capacity never trips,
    residue route == direct, accuracy bound holds."""
    x = inputs.loguniform((8, 128), seed=1)
    O.reset_capacity_violations()
    y, bad = O.fft1d(x, -1, route=2)
    assert bad == 0 and O.capacity_violations() == 0
    assert O.relerr_1d_f128(x, y, -1) <= 5e-15


def test_nonfinite_and_zero_columns(O):
    x = np.zeros((1, 64), dtype=np.complex128)
    y, _ = O.fft1d(x, -1)
    assert np.array_equal(bits(y), np.zeros((1, 128), dtype=np.uint64))
    x[0, 5] = np.inf
    y, _ = O.fft1d(x, -1)
    assert np.isnan(y).any()
