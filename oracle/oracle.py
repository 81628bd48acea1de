"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE, not product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module. It shares nothing with paper_2606_23698_b200/csrc.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboz_oracle.so")
_SRC = os.path.join(_HERE, "ozfft_oracle.c")


def build(force=False):
    """Compile oracle/ozfft_oracle.c -> oracle/liboz_oracle.so (gcc, OpenMP, libquadmath)."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_SRC[:-1] + "h"))):
        return _SO
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lquadmath", "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u64p, i32p, ip, dp = C.POINTER(C.c_uint64), C.POINTER(C.c_int32), C.POINTER(C.c_int), C.POINTER(C.c_double)
        L.oz_get_w.restype = C.c_uint64
        L.oz_twiddle_checksum.restype = C.c_uint64
        L.oz_capacity_violations.restype = C.c_long
        L.oz_quantise.restype = C.c_int64
        L.oz_quantise.argtypes = [C.c_uint64, C.c_int]
        L.oz_pack.restype = C.c_uint64
        L.oz_pack.argtypes = [C.c_uint64, C.c_uint64, C.c_int]
        L.oz_residues.argtypes = [C.c_uint64, C.c_uint64, ip]
        L.oz_crt.argtypes = [ip, C.c_int, u64p]
        L.oz_phaseA.argtypes = [ip, i32p, i32p]
        L.oz_kulisch_deposit.argtypes = [i32p, C.c_int, C.POINTER(C.c_uint32)]
        L.oz_column_top.argtypes = [u64p, C.c_int, ip]
        L.oz_stage.argtypes = [C.c_int, C.c_int, u64p, ip, C.c_int, u64p, C.c_int]
        L.oz_fft1d.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp, C.c_int]
        L.oz_fft3d.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, dp, dp, C.c_int]
        L.oz_fft1d_strided.argtypes = [C.c_int, C.c_int, dp, C.c_long, dp, C.c_long, C.c_int]
        L.oz_relerr_1d_f128.restype = C.c_double
        L.oz_relerr_1d_f128.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp]
        L.oz_relerr_3d_f128.restype = C.c_double
        L.oz_relerr_3d_f128.argtypes = [C.c_int] * 4 + [dp, C.POINTER(C.c_long), C.c_int, dp]
        L.oz_twiddle.argtypes = [C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.oz_init()
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _to128(lo, hi):
    v = (hi << 64) | lo
    return v - (1 << 128) if v >> 127 else v


def _from128(x):
    x &= (1 << 128) - 1
    return x & ((1 << 64) - 1), x >> 64


def select_modset(which):
    lib().oz_select_modset(which)


def moduli():
    return [lib().oz_modulus(k) for k in range(lib().oz_num_moduli())]


def M():
    o = (C.c_uint64 * 2)()
    lib().oz_get_M(o)
    return (o[1] << 64) | o[0]


def u(k):
    o = (C.c_uint64 * 2)()
    lib().oz_get_u(k, o)
    return (o[1] << 64) | o[0]


def t_inv(k):
    return lib().oz_get_t(k)


def w(k):
    return int(lib().oz_get_w(k))


def num_slices():
    return lib().oz_num_slices()


def uslice(k, s):
    return lib().oz_get_uslice(k, s)


def wslice(k, s):
    return lib().oz_get_wslice(k, s)


def twiddle(t):
    c, s = C.c_int64(), C.c_int64()
    lib().oz_twiddle(t, C.byref(c), C.byref(s))
    return c.value, s.value


def twiddle_checksum():
    return int(lib().oz_twiddle_checksum())


def capacity_violations():
    return lib().oz_capacity_violations()


def reset_capacity_violations():
    lib().oz_reset_capacity_violations()


def quantise(bits, tmax):
    return int(lib().oz_quantise(bits, tmax))


def column_top(bits_list):
    arr = (C.c_uint64 * len(bits_list))(*bits_list)
    t = C.c_int()
    st = lib().oz_column_top(arr, len(bits_list), C.byref(t))
    return st, t.value


def pack(R, g):
    lo, hi = _from128(R)
    return int(lib().oz_pack(lo, hi, g))


def residues(Cval):
    lo, hi = _from128(Cval)
    v = (C.c_int * 12)()
    lib().oz_residues(lo, hi, v)
    return list(v)


def crt(v, route=0):
    arr = (C.c_int * 12)(*v)
    o = (C.c_uint64 * 2)()
    lib().oz_crt(arr, route, o)
    return _to128(o[0], o[1])


def phaseA(v):
    arr = (C.c_int * 12)(*v)
    P, Z = (C.c_int32 * 16)(), (C.c_int32 * 6)()
    lib().oz_phaseA(arr, P, Z)
    return list(P)[: num_slices()], list(Z)


def kulisch_deposit(P):
    arr = (C.c_int32 * len(P))(*P)
    W = (C.c_uint32 * 6)()
    lib().oz_kulisch_deposit(arr, len(P), W)
    return list(W)


def stage(x, tidx, sign, K, R, route=2):
    """x: complex128[K]; tidx: int[R*K] -> (complex128[R], mismatches)."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    ti = np.ascontiguousarray(tidx, dtype=np.int32)
    y = np.empty(R, dtype=np.complex128)
    bad = lib().oz_stage(K, R, x.ctypes.data_as(C.POINTER(C.c_uint64)), ti.ctypes.data_as(C.POINTER(C.c_int)),
                         sign, y.ctypes.data_as(C.POINTER(C.c_uint64)), route)
    return y, bad


def fft1d(x, sign=-1, route=0):
    """x: complex128[batch, n] (or [n]); returns (y, mismatches)."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    n = x.shape[-1]
    batch = x.size // n
    y = np.empty_like(x)
    bad = lib().oz_fft1d(n, batch, sign, _dp(x), _dp(y), route)
    return y, bad


def fft3d(x, sign=-1, route=0):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    nx, ny, nz = x.shape
    y = np.empty_like(x)
    bad = lib().oz_fft3d(nx, ny, nz, sign, _dp(x), _dp(y), route)
    return y, bad


def fft1d_pencil(xpencil, sign=-1, route=0):
    """1-D transform of one gathered pencil (complex128[n])."""
    return fft1d(np.ascontiguousarray(xpencil).reshape(1, -1), sign, route)[0].reshape(-1)


def relerr_1d_f128(x, y, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    y = np.ascontiguousarray(y, dtype=np.complex128)
    n = x.shape[-1]
    return lib().oz_relerr_1d_f128(n, x.size // n, sign, _dp(x), _dp(y))


def relerr_3d_f128(x, idx, ysamp, sign=-1):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    ysamp = np.ascontiguousarray(ysamp, dtype=np.complex128)
    nx, ny, nz = x.shape
    return lib().oz_relerr_3d_f128(nx, ny, nz, sign, _dp(x), idx.ctypes.data_as(C.POINTER(C.c_long)), len(idx), _dp(ysamp))


def num_threads():
    return lib().oz_num_threads()
