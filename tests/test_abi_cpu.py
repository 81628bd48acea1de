"""CPU-only checks of the C-ABI library: it builds, loads, exports every symbol include/ozfft.h declares,
and its independent (double-double) twiddle generator reproduces the oracle's (libquadmath) table
checksum (reading S5). No compute call is made."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2606_23698_b200 import build
    return ctypes.CDLL(build.build())


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "ozfft.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(ozfft_[a-z0-9_]+)\s*\(", hdr))
    assert {"ozfft_plan_create", "ozfft_exec", "ozfft_plan_destroy"} <= names
    L = _lib()
    for n in sorted(names):
        assert hasattr(L, n), n
    from paper_2606_23698_b200 import ozfft
    assert set(ozfft.SYMBOLS) == names


def test_twiddle_checksum_matches_oracle(O):
    L = _lib()
    L.ozfft_twiddle_checksum.restype = ctypes.c_uint64
    assert int(L.ozfft_twiddle_checksum()) == O.twiddle_checksum()


def test_bad_arguments_fail_without_gpu():
    L = _lib()
    L.ozfft_plan_create.restype = ctypes.c_void_p
    L.ozfft_last_error.restype = ctypes.c_char_p
    assert not L.ozfft_plan_create(48, 32, 32, -1)  # not a power of two
    assert b"power" in L.ozfft_last_error()
    assert not L.ozfft_plan_create(32, 32, 32, 0)  # bad sign (or no device): NULL either way
    L.ozfft_exec.argtypes = [ctypes.c_void_p] * 4
    assert L.ozfft_exec(None, None, None, None) != 0
    L.ozfft_plan_destroy.argtypes = [ctypes.c_void_p]
    L.ozfft_plan_destroy(None)  # no-op


def test_product_does_not_touch_oracle():
    """The product package must not import or link anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2606_23698_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ozfft_oracle" not in src, f
