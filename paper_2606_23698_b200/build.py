"""Builds paper_2606_23698_b200/libozfft.so (sm_100a) in-tree with nvcc. No JIT cache, no torch extension."""
import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
SO = os.path.join(_HERE, "libozfft.so")
CSRC = os.path.join(_HERE, "csrc")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(_ROOT, "include", "*.h"))


SO_TIMERS = os.path.join(_HERE, "libozfft_timers.so")


def build(force=False, verbose=False, timers=False):
    """timers=True builds libozfft_timers.so: the same library with -DOZFFT_PIPE_TIMERS (clock64 stamps around every
    mbarrier wait of the byte-fed kernel's issuer and of one epilogue warp, read back by ozfft_debug_timers; a measuring
    build for `bench.py --pipe-timers`, never the one that is timed)."""
    so = SO_TIMERS if timers else SO
    if not force and os.path.exists(so) and os.path.getmtime(so) >= max(os.path.getmtime(f) for f in _deps()):
        return so
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(_ROOT, "include"), "-I", CSRC,
           "-o", so] + sources() + ["-lcudart"]
    if timers:
        cmd.insert(1, "-DOZFFT_PIPE_TIMERS")
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return so


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv, timers="--timers" in sys.argv))
