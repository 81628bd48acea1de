"""The entry point that allocates nothing (include/ozfft.h: ozfft_fft1d_1024_static): the batched 1-D transform of length 1024
with the fused-axis kernel's scratch (ring + group counters) in a file-scope static __device__ array of the library, for
callers that cannot call cudaMalloc.  Its output must equal the plan path's (ozfft_plan_create_1d + ozfft_exec) bit for bit
-- the tolerance every parity test of this repository uses -- on two calls in a row (the second call finds the first call's
contents in the shared scratch), for both directions, with more groups than ring slots, and it must refuse sizes beyond
its stated maximum.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after
the other tests (it depends on no environment variable and on no state but the library's own static arrays)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _default_kernel(monkeypatch):
    monkeypatch.delenv("OZFFT_VARIANT", raising=False)
    monkeypatch.delenv("OZFFT_SCHEDULE", raising=False)


def _plan_path(x, sign):
    import torch
    from paper_2606_23698_b200 import ozfft
    plan = ozfft.Plan.batched_1d(1024, x.shape[0], sign=sign)
    y = plan.exec(x)
    torch.cuda.synchronize()
    plan.destroy()
    return y


@pytest.mark.parametrize("batch,sign", [(256, -1), (2048, -1), (1152, +1), (65536, -1)])  # 2, 16, 9 groups and the stated maximum (512)
def test_static_entry_matches_the_plan_path_twice_in_a_row(batch, sign):
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    ozfft.static_setup()  # once per device: symbol addresses + table upload; allocates nothing
    xa = torch.from_numpy(inputs.normal((batch, 1024), 31)).cuda()
    xb = torch.from_numpy(inputs.loguniform((batch, 1024), 32)).cuda()
    want_a, want_b = _plan_path(xa, sign), _plan_path(xb, sign)
    out_a, out_b = torch.empty_like(xa), torch.empty_like(xb)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    ozfft.fft1d_1024_static(xa, out_a, sign)   # two calls in a row on one stream, different data: the second one starts
    ozfft.fft1d_1024_static(xb, out_b, sign)   # from the first one's ring contents and counters
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert torch.equal(out_a.view(torch.float64), want_a.view(torch.float64))
    assert torch.equal(out_b.view(torch.float64), want_b.view(torch.float64))
    assert free_after >= free_before, "the entry point must not take device memory"
    # and again into the same buffers, after the scratch has seen other data
    ozfft.fft1d_1024_static(xa, out_b, sign)
    torch.cuda.synchronize()
    assert torch.equal(out_b.view(torch.float64), want_a.view(torch.float64))


def test_static_entry_against_the_oracle(O):
    """not only equal to the plan path: equal to the CPU oracle"""
    import torch
    from paper_2606_23698_b200 import inputs, ozfft
    x = inputs.uniform_pm1((128, 1024), 33)
    d = torch.from_numpy(x).cuda()
    out = torch.empty_like(d)
    ozfft.fft1d_1024_static(d, out, -1)
    torch.cuda.synchronize()
    want = O.fft1d(x, -1, route=0)[0]
    assert np.array_equal(out.cpu().numpy().view(np.uint64), want.view(np.uint64))


def test_static_entry_refuses_sizes_beyond_its_maximum():
    import torch
    from paper_2606_23698_b200 import ozfft
    L = ozfft.lib()
    buf = torch.zeros(256 * 1024, dtype=torch.complex128, device="cuda")
    out = torch.zeros_like(buf)
    st = torch.cuda.current_stream().cuda_stream
    for batch in (0, 100, 129, ozfft.STATIC_MAX_BATCH + 128, -128):
        assert L.ozfft_fft1d_1024_static(batch, -1, buf.data_ptr(), out.data_ptr(), st) == 1  # OZFFT_EINVAL, nothing launched
        assert "multiple of 128" in ozfft.last_error()
    assert L.ozfft_fft1d_1024_static(256, 0, buf.data_ptr(), out.data_ptr(), st) == 1       # bad sign
    assert L.ozfft_fft1d_1024_static(256, -1, None, out.data_ptr(), st) == 1                # null input
    assert L.ozfft_fft1d_1024_static(256, -1, buf.data_ptr(), buf.data_ptr(), st) == 1      # in == out
    torch.cuda.synchronize()
