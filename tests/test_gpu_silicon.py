"""Silicon contracts the design leans on (PAPER.md:338, 890 flags them as unmeasured): tcgen05 MMAs on
integer-valued operands accumulate exactly.  kind::i8 (s8 x s8 -> s32) is exact by construction; kind::f8f6f4
(E4M3 -> f32) and kind::f16 (-> f32) are exact as long as every partial sum stays below 2^24."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _probe(kind, A, B):
    import torch
    from paper_2606_23698_b200 import ozfft
    return ozfft.probe_mma(kind, torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()).cpu().numpy()


def _e4m3(ints):
    import torch
    return torch.tensor(ints, dtype=torch.float32).to(torch.float8_e4m3fn).view(torch.uint8).numpy()


@pytest.mark.parametrize("n,kb", [(16, 32), (64, 128), (192, 64), (256, 256)])
def test_i8_exact(n, kb):
    rng = np.random.default_rng(n + kb)
    A = rng.integers(-128, 128, (128, kb), dtype=np.int8)
    B = rng.integers(-128, 128, (n, kb), dtype=np.int8)
    D = _probe(2, A.view(np.uint8), B.view(np.uint8))
    assert np.array_equal(D, A.astype(np.int64) @ B.astype(np.int64).T)


@pytest.mark.parametrize("n,kb", [(16, 32), (128, 128), (256, 96)])
def test_e4m3_integer_digits_exact(n, kb):
    rng = np.random.default_rng(n * 7 + kb)
    Ai = rng.integers(-16, 17, (128, kb))
    Bi = rng.integers(-16, 17, (n, kb))
    D = _probe(0, _e4m3(Ai), _e4m3(Bi)).view(np.float32)
    assert np.array_equal(D.astype(np.int64), Ai @ Bi.T) and np.all(D == np.round(D))


def test_e4m3_mixed_magnitude_addends_exact():
    """large and small addends in one accumulation chain: sums reach 2^19 with unit-sized terms mixed in"""
    rng = np.random.default_rng(9)
    Ai = 2 ** rng.integers(0, 9, (128, 128)) * rng.choice([-1, 1], (128, 128))
    Bi = rng.integers(-16, 17, (64, 128))
    D = _probe(0, _e4m3(Ai), _e4m3(Bi)).view(np.float32)
    assert np.array_equal(D.astype(np.int64), Ai @ Bi.T)


@pytest.mark.parametrize("kind", [1, 3])
def test_f16_phase_a_contract(kind):
    """Phase A carrier: 12 canonical residues (< 2048) x byte slices (< 256), sums < 2^23."""
    rng = np.random.default_rng(kind)
    V = np.zeros((128, 16), dtype=np.float16)
    V[:, :12] = rng.integers(0, 2039, (128, 12))
    V[0, :12] = 2038
    U = np.zeros((32, 16), dtype=np.float16)
    U[:21, :12] = rng.integers(0, 256, (21, 12))
    U[0, :12] = 255
    D = _probe(kind, V.view(np.uint8).reshape(128, 32), U.view(np.uint8).reshape(32, 32)).view(np.float32)
    want = V.astype(np.int64) @ U.astype(np.int64).T
    assert want.max() == 12 * 2038 * 255
    assert np.array_equal(D.astype(np.int64), want)


def test_u8_phase_a_two_limb_contract():
    """Phase A in the two-limb shifted-column form: u8 residue limbs x u8 slices -> s32."""
    rng = np.random.default_rng(4)
    A = rng.integers(0, 256, (128, 32), dtype=np.uint8)
    B = rng.integers(0, 256, (16, 32), dtype=np.uint8)
    A[0] = 255
    B[0] = 255
    D = _probe(4, A, B)
    assert np.array_equal(D, A.astype(np.int64) @ B.astype(np.int64).T) and D.max() == 32 * 255 * 255


@pytest.mark.parametrize("n1,kb,n2", [(16, 32, 16), (48, 224, 32), (96, 448, 32)])
def test_i8_mma_reads_s32_accumulators_from_tmem_as_bytes(n1, kb, n2):
    """The byte-fed stage kernel runs Phase A with its A operand read straight from the stage
    accumulators in TMEM: a 32-bit cell must act as four unsigned K bytes, little endian, K byte = 4*column + b."""
    import torch
    from paper_2606_23698_b200 import ozfft
    rng = np.random.default_rng(n1 + kb + n2)
    A = rng.integers(0, 256, (128, kb), dtype=np.uint8)
    B1 = rng.integers(0, 256, (n1, kb), dtype=np.uint8)
    A[0] = 255
    B1[0] = 255
    B2 = rng.integers(0, 256, (n2, 4 * n1), dtype=np.uint8)
    D1, D2 = ozfft.probe_chain(torch.from_numpy(A).cuda(), torch.from_numpy(B1).cuda(), torch.from_numpy(B2).cuda())
    D1, D2 = D1.cpu().numpy(), D2.cpu().numpy()
    want1 = A.astype(np.int64) @ B1.astype(np.int64).T
    assert np.array_equal(D1, want1)
    by = np.ascontiguousarray(want1.astype(np.uint32)).view(np.uint8).reshape(128, 4 * n1)  # little-endian bytes
    assert np.array_equal(D2, by.astype(np.int64) @ B2.astype(np.int64).T)


@pytest.mark.parametrize("kb", [16, 112, 672])
def test_tcgen05_cp_moves_operand_chunks_into_tmem(kb):
    """shared memory -> TMEM copy (tcgen05.cp 128x128b) of the byte-fed kernel's data operand: bytes unchanged"""
    import torch
    from paper_2606_23698_b200 import ozfft
    A = np.random.default_rng(kb).integers(0, 256, (128, kb), dtype=np.uint8)
    got = ozfft.probe_cp(torch.from_numpy(A).cuda()).cpu().numpy()
    assert np.array_equal(got, A)
