"""Host tables of the byte-fed stage kernel (csrc/stage_bf.cuh), checked WITHOUT a GPU: this test replays the
kernel's integer dataflow in numpy / Python integers on the library's own tables -- data bytes of x~ + 2^53,
u8 x u8 stage products per modulus and digit (even-j and odd-j sums apart), Phase A on the little-endian bytes of
the accumulators (sum and difference outputs), deposits, centred lift, minus the offset constant, pack -- and
compares every output bit with the oracle's stage (Alg. 1 + 399-416 Alg. 2).  It pins the table
layouts the kernel indexes; the kernel itself is checked on the GPU (tests/test_gpu_parity.py)."""
import numpy as np
import pytest

from paper_2606_23698_b200 import inputs, ozfft

MODS = [2039, 2029, 2027, 1089, 1024, 961, 841, 625, 529, 511, 491, 487]


def _geom(K):
    H = K // 2
    PB = (7 * H + 15) // 16 * 16
    return H, PB, (H + 1) // 2


def _planes(B, K, mid, ch, par):
    """-> int64 [48, 2*PB] logical matrix rows of one (matrix, chunk, parity)"""
    H, PB, NCH = _geom(K)
    SB = 48 * 2 * PB
    blob = B[(mid * NCH * 2 + ch * 2 + par) * SB:][:SB].reshape(2 * PB // 16, 48, 16)
    return blob.transpose(1, 0, 2).reshape(48, 2 * PB).astype(np.int64)


def _pa(PA):
    return PA.reshape(12, 32, 16).transpose(1, 0, 2).reshape(32, 192).astype(np.int64)


def _bytes7(v):
    assert 0 <= v < 1 << 56
    return [(v >> (8 * b)) & 255 for b in range(7)]


def emulate_stage(O, x, K, fusedN, sign, mid, tabs):
    B, Cc, PA = tabs
    H, PB, NCH = _geom(K)
    M = O.M()
    bits = np.ascontiguousarray(x).view(np.uint64)
    st, Tmax = O.column_top([int(b) for b in bits])
    assert st == 1
    q = [O.quantise(int(b), Tmax) for b in bits]
    xr, xi = q[0::2], q[1::2]
    off = 1 << 53
    XR = [_bytes7(v + off) for v in xr]
    XI = [_bytes7(v + off) for v in xi]
    NXI = [_bytes7(-v + off) for v in xi]
    out = np.zeros(K, dtype=np.complex128)
    ob = out.view(np.uint64)
    pam = _pa(PA)
    for part, (p0, p1) in enumerate([(XR, NXI), (XI, XR)]):
        A = np.zeros((2, 2 * PB), dtype=np.int64)
        for par in range(2):
            for h, pl in enumerate((p0, p1)):
                for jj in range(H):
                    A[par, h * PB + jj * 7: h * PB + jj * 7 + 7] = pl[2 * jj + par]
        for ch in range(NCH):
            acc = [_planes(B, K, mid, ch, par) @ A[par] for par in range(2)]  # [48] each: even-j sums, odd-j sums
            assert max(a.max() for a in acc) < 1 << 24
            for g in range(2):
                kp = 2 * ch + g
                if kp >= H:
                    continue
                kb = np.concatenate([np.ascontiguousarray(a[g * 24:(g + 1) * 24].astype(np.uint32)).view(np.uint8) for a in acc]).astype(np.int64)
                P = pam @ kb  # [32]: o*16 + s
                assert P.max() < 1 << 23
                for o in range(2):
                    k = kp + o * H
                    E = sum(int(P[o * 16 + s]) << (8 * s) for s in range(16))
                    assert E < 1 << 134
                    Rp = E % M
                    if Rp >= M // 2:
                        Rp -= M
                    c = sum(int(Cc[mid * K + k, l]) << (32 * l) for l in range(4))
                    if c >> 127:
                        c -= 1 << 128
                    ob[2 * k + part] = O.pack(Rp - c, 53 + 52 - Tmax)
    return out


@pytest.mark.parametrize("K,fused", [(32, False), (32, True), (16, True), (8, False), (4, True), (2, True), (2, False), (16, False)])
@pytest.mark.parametrize("sign", [-1, 1])
def test_bf_tables_reproduce_the_oracle_stage(O, K, fused, sign):
    fusedN = 32 * K if fused else 0
    tabs = ozfft.debug_bf_tables(K, fusedN, sign)
    rng = np.random.default_rng(K * 3 + fused)
    for trial, mid in enumerate([0, 31, 7] if fused else [0]):
        if trial == 0:
            x = inputs.uniform_pm1((1, K), seed=K + 40).reshape(-1)
        elif trial == 1:
            x = inputs.loguniform((1, K), seed=K + 41).reshape(-1)
        else:  # worst-case magnitudes: all-ones significands, alternating signs
            x = (np.full(K, 2.0 - 2.0 ** -52) * rng.choice([-1, 1], K) + 1j * np.full(K, 2.0 - 2.0 ** -52) * rng.choice([-1, 1], K))
        tidx = np.array([[((1024 // fusedN) * j * (mid + 32 * k)) % 1024 if fused else ((1024 // K) * j * k) % 1024
                          for j in range(K)] for k in range(K)], dtype=np.int32)
        want, bad = O.stage(x, tidx.reshape(-1), sign, K, K, route=2)
        assert bad == 0
        got = emulate_stage(O, x, K, fusedN, sign, mid, tabs)
        assert np.array_equal(got.view(np.uint64), want.view(np.uint64)), (K, fused, sign, mid)
