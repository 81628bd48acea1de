"""Static checks on the compiled kernels (cuobjdump, no GPU): NO function of the library contains fp64 arithmetic
(north_star: "kernels contain no fp64 arithmetic") -- except the ablation kernel that is allowed to by
name (fp64sum: Eq. 21, the rung the paper measures against) -- and the tensor-core kernels really are
Blackwell-native: tcgen05.mma -> UTCIMMA, tcgen05.ld -> LDTM, tcgen05.cp -> UTCCP, TMA bulk copy -> UBLKCP."""
import re
import shutil
import subprocess

import pytest

# any fp64 pipe opcode (DADD, DMUL, DFMA, DSETP, DMNMX, DMMA, ...), any conversion or op with an F64 type suffix,
# and the 64-bit MUFU seeds of double division / rsqrt.  DEPBAR is a dependency barrier, not arithmetic.
FP64 = re.compile(r"\b(D(?:ADD|MUL|FMA|SETP|MNMX|MMA|SEL)\b|[A-Z0-9_.]+\.F64\b|MUFU\.\w*64\w*)")
ALLOWED_FP64 = ("fp64sum",)


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


def test_fp64_pattern_self_test():
    for bad in ("DADD R0, R2, R4 ;", "DFMA R0, R2, R4, R6 ;", "MUFU.RCP64H R3, R5 ;", "MUFU.RSQ64H R3, R5 ;", "DMMA.8x8x4 R0 ;",
                "F2F.F64.F32 R2, R0 ;", "I2F.F64.S32 R2, R0 ;", "F2I.S64.F64.TRUNC R2, R4 ;", "FRND.F64.FLOOR R2, R4 ;", "DSETP.GT.AND P0 ;"):
        assert FP64.search(bad), bad
    for ok in ("DEPBAR.LE SB0, 0x0 ;", "IMAD.WIDE.U32 R2, R3, R4, R6 ;", "LDG.E.64.CONSTANT R2, desc[UR4][R2.64] ;", "MUFU.RCP R3, R5 ;",
               "STG.E.128 desc[UR4][R2.64], R8 ;", "UTCIMMA gdesc[UR8], gdesc[UR6], tmem[UR26] ;"):
        assert not FP64.search(ok), ok


def test_no_fp64_arithmetic_anywhere_in_the_library():
    ks = _kernels()
    assert sum("stage_bf_kernel" in k for k in ks) == 6 and sum("stage_tc_kernel" in k for k in ks) == 3
    assert any("stage_simt_kernel" in k for k in ks)
    for k, v in ks.items():
        if any(a in k for a in ALLOWED_FP64):
            continue
        hit = FP64.search(v)
        assert hit is None, (k, hit.group(0))


def test_tensor_core_kernels_are_blackwell_native():
    ks = _kernels()
    for k, v in ks.items():
        if "stage_tc_kernel" in k:
            ops = ("UTCIMMA", "LDTM", "UBLKCP", "SYNCS")
        elif "stage_f8_kernel" in k:
            ops = ("UTCQMMA", "LDTM", "UBLKCP", "SYNCS")  # kind::f8f6f4 -> UTCQMMA
        elif "stage_bf_kernel" in k:
            ops = ("UTCIMMA", "UTCCP", "LDTM", "UBLKCP", "SYNCS", "ELECT", "STG.E.128") + (("CCTL",) if "ELb1" in k else ("LDG.E.128",))  # fused axis: discard.global.L2
        else:
            continue
        for op in ops:
            assert op in v, (k, op)
        assert "HMMA" not in v and "IMMA." not in v.replace("UTCIMMA", "")
    assert any("stage_f8_kernel" in k for k in ks)
