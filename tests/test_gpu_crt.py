"""The device reconstruction on caller residues: Phase-A MMA, deposits, lift and the
two-sided centring (Alg. 2 lines 9-13 at PAPER.md:408-413; the paper's T4), compared bit for bit
with the oracle's Algorithm 2 (O.crt(v, 0)).  An FFT never reaches |R| near M/2 (|R| <= 2^111.5), so only this
probe executes the correction branch of the device code."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _device_crt(vs, variant):
    import torch
    from paper_2606_23698_b200 import ozfft
    res = torch.from_numpy(np.asarray(vs, dtype=np.uint16)).cuda()
    out = ozfft.probe_crt(res, variant).cpu().numpy().astype(np.uint32)
    vals = []
    for row in out:
        v = int(row[0]) | int(row[1]) << 32 | int(row[2]) << 64 | int(row[3]) << 96
        vals.append(v - (1 << 128) if v >> 127 else v)
    return vals


def _sweep(O):
    M, mods = O.M(), O.moduli()
    rng = random.Random(4)
    offs = list(range(64)) + [rng.randrange(2 ** 70) for _ in range(300)]
    cases = [0, 1, -1, M // 2 - 1, -(M // 2 - 1), -(M // 2), 2 ** 111, -(2 ** 111)]
    for d in offs:
        cases += [-(M // 2) + d, M // 2 - 1 - d]
    cases += [rng.randrange(-(M // 2), M // 2) for _ in range(3000)]
    return M, mods, rng, cases


@pytest.mark.parametrize("variant", [1, 0])
def test_two_sided_lift_boundary_sweep_canonical(O, variant):
    M, mods, rng, cases = _sweep(O)
    vs = [O.residues(c) for c in cases]
    got = _device_crt(vs, variant)
    assert got == cases
    assert got == [O.crt(v, 0) for v in vs]


def test_two_sided_lift_noncanonical_representatives(O):
    """Tensor-core form: any representative in [0, 2m) serves (m_k u_k == 0 mod M); upper representatives push
    the quotient estimate to its other side, so both correction directions run."""
    M, mods, rng, cases = _sweep(O)
    vs, want = [], []
    for c in cases:
        canon = O.residues(c)
        for mode in (1, 2):
            v = [r + m if (mode == 1 or rng.random() < 0.5) and r + m < 2 * m else r for r, m in zip(canon, mods)]
            vs.append(v)
            want.append(c)
    assert _device_crt(vs, 1) == want


@pytest.mark.parametrize("variant", [1, 0])
def test_random_residue_vectors(O, variant):
    M, mods = O.M(), O.moduli()
    rng = random.Random(99)
    vs = [[rng.randrange(m) for m in mods] for _ in range(4000)]
    vs += [[m - 1 for m in mods], [0] * 12, [1] * 12]
    assert _device_crt(vs, variant) == [O.crt(v, 0) for v in vs]
