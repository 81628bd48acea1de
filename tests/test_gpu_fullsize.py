"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.
configs[2] (1-D 1024 x 65536) and configs[3] (512^3): every output against the full oracle.
configs[4] (1024^3, 16 GiB per buffer): each axis pass separately (ozfft_exec_axis), sampled pencils of the
GPU's own pass input against the oracle's 1-D transform, bit for bit (pencils are independent, so this pins
every pass); then the one-call transform must equal the composition of the three passes."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint64)


@pytest.mark.parametrize("sign", [-1, +1])
def test_config3_batched_1d_full(O, sign):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.normal((65536, 1024), 2)
    plan = ozfft.Plan.batched_1d(1024, 65536, sign=sign)
    got = plan.exec(torch.from_numpy(x).cuda()).cpu().numpy()
    plan.destroy()
    want, bad = O.fft1d(x, sign, route=0)
    assert np.array_equal(_bits(got), _bits(want))
    assert O.relerr_1d_f128(x[:16], got[:16], sign) <= 5e-15


def test_config4_512cubed_full(O):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.uniform_pm1((512, 512, 512), 3)
    plan = ozfft.Plan(512, 512, 512)
    got = plan.exec(torch.from_numpy(x).cuda()).cpu().numpy()
    plan.destroy()
    torch.cuda.empty_cache()
    O.reset_capacity_violations()
    want, _ = O.fft3d(x, -1, route=0)
    assert O.capacity_violations() == 0
    assert np.array_equal(_bits(got), _bits(want))
    idx = np.sort(np.random.default_rng(7).choice(512 ** 3, 16, replace=False)).astype(np.int64)
    assert O.relerr_3d_f128(x, idx, got.reshape(-1)[idx]) <= 5e-15


def test_config5_1024cubed_sampled_passes_and_roundtrip(O):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    n = 1024
    h = torch.empty((n, n, n), dtype=torch.complex128)
    inputs.uniform_pm1((n, n, n), 4, out=h.numpy())
    x = h.cuda()
    plan = ozfft.Plan(n, n, n, sign=-1)
    rng = np.random.default_rng(11)
    cur = x
    for axis in range(3):  # 0 = z, 1 = y, 2 = x
        nxt = plan.exec_axis(axis, cur)
        torch.cuda.synchronize()
        for _ in range(64):
            a, b = (int(v) for v in rng.integers(0, n, 2))
            sl = (a, b, slice(None)) if axis == 0 else ((a, slice(None), b) if axis == 1 else (slice(None), a, b))
            pin = cur[sl].cpu().numpy()
            pout = nxt[sl].cpu().numpy()
            assert np.array_equal(_bits(pout), _bits(O.fft1d_pencil(pin, -1))), (axis, a, b)
        if axis:
            del cur
        cur = nxt
    full = plan.exec(x)
    torch.cuda.synchronize()
    assert torch.equal(full.view(torch.float64), cur.view(torch.float64))
    del cur
    # sampled outputs against the __float128 DFT of the input (north_star: <= 5e-15 normwise)
    idx = np.sort(rng.choice(n ** 3, 3, replace=False)).astype(np.int64)
    ys = full.view(-1)[torch.from_numpy(idx).cuda()].cpu().numpy()
    assert O.relerr_3d_f128(h.numpy(), idx, ys) <= 5e-15
    # forward then inverse (configs[4]): the inverse passes are bit-checked the same way (sampled pencils of each
    # pass against the oracle's sign=+1 transform), then the round-trip error
    inv = ozfft.Plan(n, n, n, sign=+1)
    cur = full
    for axis in range(3):
        nxt = inv.exec_axis(axis, cur)
        torch.cuda.synchronize()
        for _ in range(32):
            a, b = (int(v) for v in rng.integers(0, n, 2))
            sl = (a, b, slice(None)) if axis == 0 else ((a, slice(None), b) if axis == 1 else (slice(None), a, b))
            assert np.array_equal(_bits(nxt[sl].cpu().numpy()), _bits(O.fft1d_pencil(cur[sl].cpu().numpy(), +1))), (axis, a, b)
        if axis:
            del cur
        cur = nxt
    back = inv.exec(full)
    torch.cuda.synchronize()
    assert torch.equal(back.view(torch.float64), cur.view(torch.float64))
    del cur
    num = den = 0.0
    for i in range(0, n, 64):
        d = back[i:i + 64] / float(n ** 3) - x[i:i + 64]
        num += float((d.abs() ** 2).sum())
        den += float((x[i:i + 64].abs() ** 2).sum())
    assert (num / den) ** 0.5 < 5e-15
    plan.destroy()
    inv.destroy()
