"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit (north_star: "the GPU
result must be bit-exact against the oracle, because the only rounding is the final conversion")."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_F128 = 5e-15  # north_star: normwise relative error vs the __float128 naive DFT


@pytest.fixture(autouse=True, params=["bf", "tc", "simt", "fp8"])
def variant(request, monkeypatch):
    """every parity case runs on the byte-fed tensor-core kernel (the default), on the residue-digit tensor-core
    kernel, on the all-SIMT cross-check kernel and on the FP8 (kind::f8f6f4 + Karatsuba) rung"""
    monkeypatch.setenv("OZFFT_VARIANT", request.param)
    return request.param


def _torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _run3d(x, sign=-1):
    torch = _torch()
    from paper_2606_23698_b200 import ozfft
    plan = ozfft.Plan(*x.shape, sign=sign)
    d = torch.from_numpy(x).cuda()
    y = plan.exec(d)
    torch.cuda.synchronize()
    out = y.cpu().numpy()
    plan.destroy()
    return out


def _run1d(x, sign=-1):
    torch = _torch()
    from paper_2606_23698_b200 import ozfft
    batch, n = x.shape
    plan = ozfft.Plan.batched_1d(n, batch, sign=sign)
    y = plan.exec(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    out = y.cpu().numpy()
    plan.destroy()
    return out


def _bits(a):
    return np.ascontiguousarray(a).view(np.uint64)


def _assert_bit_exact(got, want):
    gb, wb = _bits(got), _bits(want)
    bad = np.flatnonzero(gb != wb)
    assert bad.size == 0, f"{bad.size} of {gb.size} words differ; first at {bad[:5]}: got {gb.flat[bad[0]]:#x} want {wb.flat[bad[0]]:#x}"


def test_config1_32cubed_bit_exact_and_accurate(O):
    from paper_2606_23698_b200 import inputs
    x = inputs.uniform_pm1((32, 32, 32), 0)
    got = _run3d(x)
    want, bad = O.fft3d(x, -1, route=0)
    assert bad == 0
    _assert_bit_exact(got, want)
    idx = np.arange(0, 32 ** 3, 37, dtype=np.int64)
    assert O.relerr_3d_f128(x, idx, got.reshape(-1)[idx]) <= TOL_F128


def test_config2_128cubed_lograng_bit_exact(O):
    from paper_2606_23698_b200 import inputs
    x = inputs.loguniform((128, 128, 128), 1)
    got = _run3d(x)
    O.reset_capacity_violations()
    want, _ = O.fft3d(x, -1, route=0)
    assert O.capacity_violations() == 0
    _assert_bit_exact(got, want)
    rng = np.random.default_rng(5)
    idx = np.sort(rng.choice(128 ** 3, 256, replace=False)).astype(np.int64)
    assert O.relerr_3d_f128(x, idx, got.reshape(-1)[idx]) <= TOL_F128


@pytest.mark.parametrize("shape", [(32, 64, 128), (64, 32, 32), (32, 32, 256), (2, 16, 32), (32, 4, 64)])
def test_mixed_shapes_bit_exact(O, shape):
    from paper_2606_23698_b200 import inputs
    x = inputs.uniform_pm1(shape, 11)
    _assert_bit_exact(_run3d(x), O.fft3d(x, -1, route=0)[0])


def test_inverse_and_roundtrip(O):
    from paper_2606_23698_b200 import inputs
    x = inputs.uniform_pm1((32, 64, 64), 12)
    y = _run3d(x, -1)
    z = _run3d(y, +1)
    _assert_bit_exact(z, O.fft3d(y, +1, route=0)[0])
    assert np.linalg.norm(z / x.size - x) / np.linalg.norm(x) < 5e-15


@pytest.mark.parametrize("sign", [-1, +1])
@pytest.mark.parametrize("n", [1024, 512, 64, 32, 8])
def test_batched_1d_bit_exact(O, n, sign):
    """both directions at every fused-stage width (second-stage K = 32, 16, 2, -, -)"""
    from paper_2606_23698_b200 import inputs
    x = inputs.normal((96, n), 2)
    got = _run1d(x, sign)
    _assert_bit_exact(got, O.fft1d(x, sign, route=0)[0])
    assert O.relerr_1d_f128(x[:8], got[:8], sign) <= TOL_F128


def test_edge_columns_zero_subnormal_huge(O):
    """all-zero columns, subnormal inputs, values near overflow, exact ties in the quantiser."""
    rng = np.random.default_rng(3)
    x = (rng.standard_normal((64, 1024)) + 1j * rng.standard_normal((64, 1024)))
    x[0] = 0
    x[1] *= 5e-324 * 1e3           # subnormal pencil
    x[2] *= 1e300                  # outputs overflow-free but large
    x[3, ::2] = 0
    x[4] = 1.0                     # DC: exact closed form
    x[5] = 0; x[5, 0] = 1.0        # impulse
    x[6].real = np.ldexp(1.0, -rng.integers(0, 60, 1024)) * (1 + 2.0 ** -52)
    e7 = rng.integers(-500, 500, 1024)
    x[7] = np.ldexp(x[7].real, e7) + 1j * np.ldexp(x[7].imag, e7)
    got = _run1d(x)
    want = O.fft1d(x, -1, route=0)[0]
    _assert_bit_exact(got, want)
    assert got[4, 0] == 1024 and np.all(got[4, 1:] == 0)
    assert np.all(got[5] == 1.0)


def test_nonfinite_column_gives_nan(O):
    x = np.ones((32, 64), dtype=np.complex128)
    x[3, 5] = np.inf
    got = _run1d(x)
    assert np.isnan(got[3]).any()
    _assert_bit_exact(got, O.fft1d(x, -1, route=0)[0])


def test_exec_host_and_axis(O):
    torch = _torch()
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.uniform_pm1((32, 64, 32), 13)
    plan = ozfft.Plan(32, 64, 32)
    xin = torch.from_numpy(x).pin_memory()
    out = torch.empty_like(xin).pin_memory()
    plan.exec_host(xin, out)
    _assert_bit_exact(out.numpy(), O.fft3d(x, -1, route=0)[0])
    # one axis pass (y): every y-pencil equals the oracle's 1-D transform
    ya = plan.exec_axis(1, torch.from_numpy(x).cuda()).cpu().numpy()
    for (ix, iz) in [(0, 0), (7, 31), (31, 5)]:
        _assert_bit_exact(ya[ix, :, iz], O.fft1d_pencil(x[ix, :, iz]))
    assert plan.num_launches == 4 and plan.device_bytes > x.nbytes
    plan.destroy()


def test_bad_arguments():
    torch = _torch()
    from paper_2606_23698_b200 import ozfft
    with pytest.raises(RuntimeError):
        ozfft.Plan(32, 32, 48)
    with pytest.raises(RuntimeError):
        ozfft.Plan(32, 32, 2048)  # beyond the K <= 32 capacity budget
    plan = ozfft.Plan(32, 32, 32)
    x = torch.zeros(32 ** 3, dtype=torch.complex128, device="cuda")
    assert ozfft.lib().ozfft_exec(plan.h, x.data_ptr(), x.data_ptr(), None) == 1  # in == out
    assert ozfft.lib().ozfft_exec(plan.h, x.data_ptr() + 8, x.data_ptr(), None) == 1  # misaligned
    plan.destroy()


@pytest.mark.parametrize("shape", [(16, 16, 16), (8, 8, 32), (2, 2, 2), (4, 64, 8), (2, 1024, 4)])
def test_small_shapes_masked_tail_tiles(O, shape):
    """every power-of-two size in [2, 1024] per axis is accepted: blocks with fewer than 32 columns and
    tiles with missing blocks are masked, not rejected"""
    from paper_2606_23698_b200 import inputs
    x = inputs.uniform_pm1(shape, 17)
    _assert_bit_exact(_run3d(x), O.fft3d(x, -1, route=0)[0])
    _assert_bit_exact(_run3d(x, +1), O.fft3d(x, +1, route=0)[0])


@pytest.mark.parametrize("n,batch", [(1024, 1), (64, 5), (8, 33), (512, 100), (2, 7)])
def test_batched_1d_any_batch(O, n, batch):
    from paper_2606_23698_b200 import inputs
    x = inputs.normal((batch, n), 19)
    _assert_bit_exact(_run1d(x), O.fft1d(x, -1, route=0)[0])


def test_plan_lifetime_and_threads(O, variant):
    """a destroyed handle is refused without touching freed memory; destroying twice is a no-op; two plans created and
    executed from two host threads (each on its own stream) give the oracle's bits"""
    if variant == "simt":
        pytest.skip("host-side logic; run on the tensor-core kernels")
    import threading
    torch = _torch()
    from paper_2606_23698_b200 import inputs, ozfft
    plan = ozfft.Plan(32, 32, 32)
    h = plan.h
    x = torch.zeros(32 ** 3, dtype=torch.complex128, device="cuda")
    y = torch.empty_like(x)
    assert ozfft.lib().ozfft_exec(h, x.data_ptr(), y.data_ptr(), None) == 0
    torch.cuda.synchronize()
    ozfft.lib().ozfft_plan_destroy(h)
    ozfft.lib().ozfft_plan_destroy(h)  # second destroy: no-op
    assert ozfft.lib().ozfft_exec(h, x.data_ptr(), y.data_ptr(), None) == 1  # OZFFT_EINVAL
    assert ozfft.lib().ozfft_plan_num_launches(h) == -1
    plan.h = None
    res = {}

    def work(i, shape, sign):
        xx = inputs.uniform_pm1(shape, 30 + i)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            p = ozfft.Plan(*shape, sign=sign)
            d = torch.from_numpy(xx).cuda()
            out = p.exec(d, stream=st.cuda_stream)
            st.synchronize()
            res[i] = (xx, sign, out.cpu().numpy())
            p.destroy()

    ts = [threading.Thread(target=work, args=(0, (32, 64, 32), -1)), threading.Thread(target=work, args=(1, (64, 32, 128), +1))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    for i in (0, 1):
        xx, sign, got = res[i]
        _assert_bit_exact(got, O.fft3d(xx, sign, route=0)[0])


def test_exec_host_pipelined_path(O, variant):
    """sizes >= 2^24 elements take the slab pipeline in ozfft_exec_host (copies overlapped with the passes):
    same bits as the device-resident call and as the oracle"""
    if variant != "bf":
        pytest.skip("pipeline logic is kernel-independent; run once")
    torch = _torch()
    from paper_2606_23698_b200 import inputs, ozfft
    shape = (256, 256, 256)
    x = inputs.uniform_pm1(shape, 21)
    plan = ozfft.Plan(*shape)
    xin = torch.from_numpy(x).pin_memory()
    out = torch.empty_like(xin).pin_memory()
    plan.exec_host(xin, out)
    dev = plan.exec(torch.from_numpy(x).cuda()).cpu()
    assert torch.equal(out.view(torch.float64), dev.view(torch.float64))
    _assert_bit_exact(out.numpy(), O.fft3d(x, -1, route=0)[0])
    plan.exec_host(xin, out)  # a second call reuses streams and events
    assert torch.equal(out.view(torch.float64), dev.view(torch.float64))
    plan.destroy()
