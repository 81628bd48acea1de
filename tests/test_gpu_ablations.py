"""Ablation rungs (PAPER.md:872 protocol item 2) on the SIMT kernel, selected with OZFFT_VARIANT:
  garner  -- recursive Garner mixed-radix reconstruction (Eq. 9-11) instead of the direct CRT:
             the integer is unique, so the result must still be bit-exact against the oracle;
  fp64sum -- direct-CRT slice sums followed by the naive fp64 Phase B (Eq. 21): rounds at every step,
             NOT exact by design (PAPER.md:1131-1143 expects bits to be lost); its error against the __float128 DFT is
             measured and must sit far above the exact path's and far below garbage."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _run(x, variant, monkeypatch, sign=-1):
    import torch
    from paper_2606_23698_b200 import ozfft
    monkeypatch.setenv("OZFFT_VARIANT", variant)
    if x.ndim == 3:
        plan = ozfft.Plan(*x.shape, sign=sign)
    else:
        plan = ozfft.Plan.batched_1d(x.shape[1], x.shape[0], sign=sign)
    y = plan.exec(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    out = y.cpu().numpy()
    plan.destroy()
    return out


@pytest.mark.parametrize("shape", [(32, 32, 32), (32, 64, 128), (96, 1024), (40, 512)])
def test_garner_reconstruction_is_bit_exact(O, shape, monkeypatch):
    from paper_2606_23698_b200 import inputs
    x = inputs.uniform_pm1(shape, 23) if len(shape) == 3 else inputs.normal(shape, 23)
    got = _run(x, "garner", monkeypatch)
    want = O.fft3d(x, -1, route=0)[0] if len(shape) == 3 else O.fft1d(x, -1, route=0)[0]
    assert np.array_equal(np.ascontiguousarray(got).view(np.uint64), want.view(np.uint64))


def test_garner_on_wide_dynamic_range(O, monkeypatch):
    from paper_2606_23698_b200 import inputs
    x = inputs.loguniform((64, 1024), 24)
    got = _run(x, "garner", monkeypatch)
    assert np.array_equal(np.ascontiguousarray(got).view(np.uint64), O.fft1d(x, -1, route=0)[0].view(np.uint64))


def test_fp64sum_loses_bits_but_not_the_answer(O, monkeypatch):
    from paper_2606_23698_b200 import inputs
    x = inputs.normal((64, 1024), 25)
    exact = _run(x, "bf", monkeypatch)
    naive = _run(x, "fp64sum", monkeypatch)
    e_exact = O.relerr_1d_f128(x[:16], exact[:16])
    e_naive = O.relerr_1d_f128(x[:16], naive[:16])
    print(f"normwise error vs __float128 DFT: exact path {e_exact:.3e}, naive fp64 Phase B {e_naive:.3e}")
    assert e_exact <= 5e-15
    assert 1e-14 < e_naive < 1e-6  # the cancellation E - zM in fp64 costs tens of bits, not the answer
