"""Static checks on the compiled kernels (cuobjdump, no GPU): the hot kernels contain NO fp64 arithmetic
(north_star: "kernels contain no fp64 arithmetic") and the tensor-core kernel really is
Blackwell-native: tcgen05.mma -> UTCIMMA, tcgen05.ld -> LDTM, TMA bulk copy -> UBLKCP."""
import re
import shutil
import subprocess

import pytest

FP64 = re.compile(r"\b(DADD|DMUL|DFMA|DSETP|DMNMX|F2F\.F64|F2F\.F32\.F64|I2F\.F64|F2I\.[A-Z0-9.]*F64|MUFU\.[A-Z0-9]*64)\b")


def _kernels():
    from paper_2606_23698_b200 import build
    so = build.build()
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    txt = subprocess.run(["cuobjdump", "-sass", so], capture_output=True, text=True, check=True).stdout
    out, name = {}, None
    for line in txt.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            out[name] = []
        elif name:
            out[name].append(line)
    return {k: "\n".join(v) for k, v in out.items()}


def test_no_fp64_arithmetic_in_hot_kernels():
    ks = {k: v for k, v in _kernels().items() if "stage_tc_kernel" in k or "stage_simt_kernel" in k}
    assert len(ks) >= 4
    for k, v in ks.items():
        hit = FP64.search(v)
        assert hit is None, (k, hit.group(0))


def test_tensor_core_kernel_is_blackwell_native():
    ks = {k: v for k, v in _kernels().items() if "stage_tc_kernel" in k}
    assert len(ks) == 3
    for k, v in ks.items():
        for op in ("UTCIMMA", "LDTM", "UBLKCP", "SYNCS"):
            assert op in v, (k, op)
        assert "HMMA" not in v and "IMMA." not in v.replace("UTCIMMA", "")
