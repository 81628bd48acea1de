"""Thin ctypes binding of libozfft.so (include/ozfft.h). Argument marshalling only.

PyTorch supplies device memory and streams; every step of the transform runs in the CUDA kernels behind
the C ABI. There is no CPU fallback: if the library is missing or fails, this raises.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libozfft.so")
_lib = None

SYMBOLS = ["ozfft_plan_create", "ozfft_plan_create_1d", "ozfft_exec", "ozfft_exec_host", "ozfft_plan_destroy",
           "ozfft_last_error", "ozfft_twiddle_checksum", "ozfft_plan_num_launches", "ozfft_plan_device_bytes",
           "ozfft_exec_axis", "ozfft_probe_mma", "ozfft_probe_chain", "ozfft_probe_crt", "ozfft_debug_bf_tables", "ozfft_probe_cp", "ozfft_debug_timers", "ozfft_debug_fuse_sequence",
           "ozfft_static_setup", "ozfft_fft1d_1024_static"]


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} not built: run `python paper_2606_23698_b200/build.py` (no fallback path exists)")
        L = C.CDLL(_SO)
        vp = C.c_void_p
        L.ozfft_plan_create.restype = vp
        L.ozfft_plan_create.argtypes = [C.c_int] * 4
        L.ozfft_plan_create_1d.restype = vp
        L.ozfft_plan_create_1d.argtypes = [C.c_int] * 3
        L.ozfft_exec.argtypes = [vp, vp, vp, vp]
        L.ozfft_exec_host.argtypes = [vp, vp, vp, vp]
        L.ozfft_exec_axis.argtypes = [vp, C.c_int, vp, vp, vp]
        L.ozfft_plan_destroy.argtypes = [vp]
        L.ozfft_plan_destroy.restype = None
        L.ozfft_last_error.restype = C.c_char_p
        L.ozfft_twiddle_checksum.restype = C.c_uint64
        L.ozfft_plan_num_launches.argtypes = [vp]
        L.ozfft_plan_device_bytes.argtypes = [vp]
        L.ozfft_plan_device_bytes.restype = C.c_size_t
        L.ozfft_probe_mma.argtypes = [C.c_int, C.c_int, C.c_int, vp, vp, vp, vp]
        L.ozfft_probe_chain.argtypes = [C.c_int, C.c_int, C.c_int, vp, vp, vp, vp, vp, vp]
        L.ozfft_probe_crt.argtypes = [C.c_int, vp, vp, C.c_int, vp]
        L.ozfft_probe_cp.argtypes = [C.c_int, vp, vp, vp]
        L.ozfft_debug_timers.argtypes = [vp]
        L.ozfft_fft1d_1024_static.argtypes = [C.c_int, C.c_int, vp, vp, vp]
        L.ozfft_debug_fuse_sequence.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.ozfft_debug_bf_tables.restype = C.c_size_t
        L.ozfft_debug_bf_tables.argtypes = [C.c_int, C.c_int, C.c_int, vp, vp, vp]
        _lib = L
    return _lib


def last_error():
    return lib().ozfft_last_error().decode()


def _stream(stream):
    if stream is not None:
        return stream
    import torch
    return torch.cuda.current_stream().cuda_stream


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed (code {rc}): {last_error()}")


class Plan:
    """ozfft plan. Plan(nx, ny, nz, sign=-1) for 3-D; Plan.batched_1d(n, batch, sign=-1) for contiguous pencils."""

    def __init__(self, nx, ny, nz, sign=-1, _handle=None, _count=None):
        self.h = _handle if _handle is not None else lib().ozfft_plan_create(nx, ny, nz, sign)
        self.count = _count if _count is not None else nx * ny * nz
        if not self.h:
            raise RuntimeError("ozfft_plan_create failed: " + last_error())

    @classmethod
    def batched_1d(cls, n, batch, sign=-1):
        h = lib().ozfft_plan_create_1d(n, batch, sign)
        if not h:
            raise RuntimeError("ozfft_plan_create_1d failed: " + last_error())
        return cls(0, 0, 0, sign, _handle=h, _count=n * batch)

    def _args(self, x, out):
        import torch
        assert x.is_cuda and x.dtype == torch.complex128 and x.is_contiguous() and x.numel() == self.count
        if out is None:
            out = torch.empty_like(x)
        assert out.is_cuda and out.dtype == torch.complex128 and out.is_contiguous() and out.numel() == self.count
        return x, out

    def exec(self, x, out=None, stream=None):
        """x, out: CUDA complex128 tensors (contiguous). Asynchronous on the stream."""
        x, out = self._args(x, out)
        _check(lib().ozfft_exec(self.h, x.data_ptr(), out.data_ptr(), _stream(stream)), "ozfft_exec")
        return out

    def exec_axis(self, axis, x, out=None, stream=None):
        x, out = self._args(x, out)
        _check(lib().ozfft_exec_axis(self.h, axis, x.data_ptr(), out.data_ptr(), _stream(stream)), "ozfft_exec_axis")
        return out

    def exec_host(self, x_host, out_host, stream=None):
        """x_host, out_host: CPU complex128 tensors (pinned for speed). Synchronous."""
        _check(lib().ozfft_exec_host(self.h, x_host.data_ptr(), out_host.data_ptr(), _stream(stream)), "ozfft_exec_host")
        return out_host

    @property
    def num_launches(self):
        return lib().ozfft_plan_num_launches(self.h)

    @property
    def device_bytes(self):
        return lib().ozfft_plan_device_bytes(self.h)

    def destroy(self):
        if self.h:
            lib().ozfft_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


STATIC_MAX_BATCH = 65536


def static_setup():
    """once per device: addresses of the library's static scratch / tables, table upload (no allocation)"""
    _check(lib().ozfft_static_setup(), "ozfft_static_setup")


def fft1d_1024_static(x, out, sign=-1, stream=None):
    """x, out: CUDA complex128 [batch, 1024], contiguous, batch a multiple of 128 up to STATIC_MAX_BATCH.  Allocates nothing:
    the caller passes the output; the scratch is a static device array of the library (calls that overlap on the GPU race)."""
    import torch
    assert x.is_cuda and out.is_cuda and x.dtype == out.dtype == torch.complex128 and x.is_contiguous() and out.is_contiguous()
    assert x.dim() == 2 and x.shape[1] == 1024 and out.shape == x.shape
    _check(lib().ozfft_fft1d_1024_static(x.shape[0], sign, x.data_ptr(), out.data_ptr(), _stream(stream)), "ozfft_fft1d_1024_static")
    return out


def twiddle_checksum():
    return int(lib().ozfft_twiddle_checksum())


def probe_mma(kind, A, B):
    """A: uint8 CUDA tensor [128, kbytes]; B: uint8 CUDA [n, kbytes] -> int32 CUDA [128, n] raw accumulators."""
    import torch
    n, kb = B.shape
    D = torch.zeros((128, n), dtype=torch.int32, device=A.device)
    _check(lib().ozfft_probe_mma(kind, n, kb, A.data_ptr(), B.data_ptr(), D.data_ptr(), _stream(None)), "ozfft_probe_mma")
    torch.cuda.synchronize()
    return D


def probe_chain(A, B1, B2):
    """A: uint8 CUDA [128, kb]; B1: uint8 [n1, kb]; B2: uint8 [n2, 4*n1] -> (D1 int32 [128, n1], D2 int32 [128, n2]):
    D2 = bytes(D1) @ B2^T with the second MMA's A operand read from the TMEM accumulator of the first."""
    import torch
    n1, kb = B1.shape
    n2 = B2.shape[0]
    assert B2.shape[1] == 4 * n1
    D1 = torch.zeros((128, n1), dtype=torch.int32, device=A.device)
    D2 = torch.zeros((128, n2), dtype=torch.int32, device=A.device)
    _check(lib().ozfft_probe_chain(n1, kb, n2, A.data_ptr(), B1.data_ptr(), B2.data_ptr(), D1.data_ptr(), D2.data_ptr(),
                                   _stream(None)), "ozfft_probe_chain")
    torch.cuda.synchronize()
    return D1, D2


def probe_crt(residues, variant):
    """residues: uint16 CUDA tensor [n, 12] -> int32 CUDA [n, 4]: two's-complement limbs of the centred CRT result."""
    import torch
    n = residues.shape[0]
    assert residues.dtype == torch.uint16 and residues.shape[1] == 12 and residues.is_contiguous()
    out = torch.zeros((n, 4), dtype=torch.int32, device=residues.device)
    _check(lib().ozfft_probe_crt(n, residues.data_ptr(), out.data_ptr(), variant, _stream(None)), "ozfft_probe_crt")
    return out


def debug_bf_tables(K, fusedN, sign):
    """Host tables of the byte-fed stage kernel as numpy arrays (B planes uint8, C limbs uint32 [nmat*K, 4], PA uint8)."""
    import numpy as np
    size = lib().ozfft_debug_bf_tables(K, fusedN, sign, None, None, None)
    if not size:
        raise ValueError("bad (K, fusedN, sign)")
    nmat = 32 if fusedN else 1
    B = np.zeros(size, dtype=np.uint8)
    Cc = np.zeros((nmat * K, 4), dtype=np.uint32)
    PA = np.zeros(6144, dtype=np.uint8)
    lib().ozfft_debug_bf_tables(K, fusedN, sign, B.ctypes.data, Cc.ctypes.data, PA.ctypes.data)
    return B, Cc, PA


def probe_cp(A):
    """A: uint8 CUDA [128, kb] -> uint8 CUDA [128, kb] read back from TMEM after a tcgen05.cp of every 16-byte chunk."""
    import torch
    kb = A.shape[1]
    D = torch.zeros((128, kb // 4), dtype=torch.int32, device=A.device)
    _check(lib().ozfft_probe_cp(kb, A.data_ptr(), D.data_ptr(), _stream(None)), "ozfft_probe_cp")
    torch.cuda.synchronize()
    return D.view(torch.uint8).reshape(128, kb)
