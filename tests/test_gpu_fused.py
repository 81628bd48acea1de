"""GPU parity of the two schedules of the byte-fed kernel (Alg. 1 lines 7-8 at 220-241):
fused -- both stages of an axis of length 1024 in one launch, Y' in an L2-resident ring -- and unfused (two launches per
axis, OZFFT_SCHEDULE=unfused).  Both must equal the oracle bit for bit.  The shapes cover: the contiguous axis fused
(ring [k2][pencil][j1]), a strided axis fused (ring [k2][j1][lane]), the strided axis that also takes the z permutation
out (8 x 16 patch), more groups than ring slots (slot reuse, both hand-shakes), a fused axis next to an
unfusable one (inner length 2), and the batched 1-D plan."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SHAPES = [((8, 64, 1024), 5, 4),     # z fused (4 groups, output permuted along z), y two unfused stages, the first with the patch
          ((1024, 4, 128), 6, 4),    # x fused (strided, 4 groups)
          ((2, 1024, 256), 7, 4),    # y fused (2 groups); z of length 256 keeps the natural order
          ((2, 1024, 1024), 11, 3),  # z fused and permuted, y fused AND un-permuting (patch)
          ((16, 256, 1024), 8, 4),    # z fused with 32 groups > 16 ring slots
          ((1024, 1024, 2), 9, 4)]   # x fused, y cannot be (inner length 2)


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint64)


@pytest.fixture(params=["fused", "unfused"])
def schedule(request, monkeypatch):
    monkeypatch.setenv("OZFFT_VARIANT", "bf")
    monkeypatch.setenv("OZFFT_SCHEDULE", request.param)
    return request.param


@pytest.mark.parametrize("shape,seed,fused_launches", SHAPES)
@pytest.mark.parametrize("sign", [-1, +1])
def test_schedules_bit_exact_3d(O, schedule, shape, seed, fused_launches, sign):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.uniform_pm1(shape, seed)
    plan = ozfft.Plan(*shape, sign=sign)
    if schedule == "fused":
        assert plan.num_launches == fused_launches
    y = plan.exec(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    got = y.cpu().numpy()
    # a second execution of the same plan reuses the ring and the counters
    y2 = plan.exec(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    plan.destroy()
    want, _ = O.fft3d(x, sign, route=0)
    assert np.array_equal(_bits(got), _bits(want))
    assert np.array_equal(_bits(y2.cpu().numpy()), _bits(want))


def test_schedules_bit_exact_batched_1d(O, schedule):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.normal((2048, 1024), 2)
    plan = ozfft.Plan.batched_1d(1024, 2048)
    assert plan.num_launches == (1 if schedule == "fused" else 2)
    got = plan.exec(torch.from_numpy(x).cuda()).cpu().numpy()
    plan.destroy()
    want, _ = O.fft1d(x, -1, route=0)
    assert np.array_equal(_bits(got), _bits(want))


def test_axis_hook_matches_fused_transform(schedule):
    """ozfft_exec_axis runs every pass with natural-order intermediates; the one-call transform (fused axes, permuted z
    between the z and y passes) must equal the composition of the three passes."""
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    shape = (4, 1024, 1024)
    x = torch.from_numpy(inputs.uniform_pm1(shape, 10)).cuda()
    plan = ozfft.Plan(*shape)
    cur = x
    for axis in range(3):
        cur = plan.exec_axis(axis, cur)
    full = plan.exec(x)
    torch.cuda.synchronize()
    plan.destroy()
    assert torch.equal(full.view(torch.float64), cur.view(torch.float64))


def test_edge_columns_through_the_fused_axis(O, schedule):
    """all-zero, subnormal, huge, DC, impulse, wide-exponent and non-finite pencils in a batch that takes the fused schedule
    (256 pencils = 2 groups): exact zeros and tiny results go through the generic pack, zero / non-finite columns through the
    flag path of both stages, and every group counter still reaches its target."""
    import torch
    from paper_2606_23698_b200 import ozfft
    rng = np.random.default_rng(3)
    x = (rng.standard_normal((256, 1024)) + 1j * rng.standard_normal((256, 1024)))
    x[0] = 0
    x[1] *= 5e-324 * 1e3
    x[2] *= 1e300
    x[3, ::2] = 0
    x[4] = 1.0
    x[5] = 0; x[5, 0] = 1.0
    x[6].real = np.ldexp(1.0, -rng.integers(0, 60, 1024)) * (1 + 2.0 ** -52)
    e7 = rng.integers(-500, 500, 1024)
    x[7] = np.ldexp(x[7].real, e7) + 1j * np.ldexp(x[7].imag, e7)
    x[130, 77] = np.inf
    x[200] = 0
    plan = ozfft.Plan.batched_1d(1024, 256)
    assert plan.num_launches == (1 if schedule == "fused" else 2)
    got = plan.exec(torch.from_numpy(x).cuda()).cpu().numpy()
    plan.destroy()
    want = O.fft1d(x, -1, route=0)[0]
    assert np.array_equal(_bits(got), _bits(want))
    assert got[4, 0] == 1024 and np.all(got[4, 1:] == 0)
    assert np.all(got[5] == 1.0)
    assert np.isnan(got[130]).all() and not np.isnan(got[129]).any()
