"""Host logic of the fused-axis schedule (csrc/stage_bf.cuh BfFuse), no GPU: the tile sequence the
persistent CTAs walk must (i) visit every (stage, group) block exactly once, (ii) put the second stage of a group after
its first stage, at the distance the design states (2 lag + 1 blocks in the steady state), and (iii) make every wait of
the ring hand-shake point at EARLIER blocks -- a second-stage block waits for the first stage of its own group, a
first-stage block that overwrites ring slot g mod R waits for the second stage of group g - R -- which, with all CTAs
resident and each walking the sequence in order, rules out a cycle."""
import ctypes as C

import pytest

LAG, RING = 8, 16  # the plan's constants (ozfft.cu make_plan)


def _seq(groups, lag):
    from paper_2606_23698_b200 import build, ozfft
    build.build()
    L = ozfft.lib()
    st, grp = C.c_int(), C.c_int()
    out = []
    for q in range(2 * groups):
        assert L.ozfft_debug_fuse_sequence(q, lag, groups, C.byref(st), C.byref(grp)) == 0
        out.append((st.value, grp.value))
    return out


@pytest.mark.parametrize("groups", [1, 2, 4, 7, 8, 9, 16, 17, 64, 512, 8192])
def test_sequence_is_a_bijection_with_ordered_dependencies(groups):
    lag = min(LAG, groups)
    seq = _seq(groups, lag)
    assert sorted(seq) == sorted((s, g) for s in (0, 1) for g in range(groups))
    pos = {sg: q for q, sg in enumerate(seq)}
    for g in range(groups):
        assert pos[(1, g)] > pos[(0, g)]                       # data before its reader
        if g >= RING:
            assert pos[(1, g - RING)] < pos[(0, g)]            # the slot's previous tenant is read before it is overwritten
        if lag <= g < groups:
            assert pos[(1, g - lag)] == pos[(0, g)] + 1        # steady state: first stage of g, then second stage of g - lag
    if groups > 2 * lag:
        g = groups // 2
        assert pos[(1, g)] - pos[(0, g)] == 2 * lag + 1
    # ring slots alive at once never exceed the ring: between a group's first-stage block and its second-stage block at
    # most RING - 1 other groups start their first stage
    for g in range(groups):
        started = sum(1 for h in range(groups) if pos[(0, g)] < pos[(0, h)] < pos[(1, g)])
        assert started < RING


def test_sequence_rejects_bad_arguments():
    from paper_2606_23698_b200 import build, ozfft
    build.build()
    L = ozfft.lib()
    st, grp = C.c_int(), C.c_int()
    assert L.ozfft_debug_fuse_sequence(-1, 8, 16, C.byref(st), C.byref(grp)) != 0
    assert L.ozfft_debug_fuse_sequence(32, 8, 16, C.byref(st), C.byref(grp)) != 0
    assert L.ozfft_debug_fuse_sequence(0, 9, 8, C.byref(st), C.byref(grp)) != 0
    assert L.ozfft_debug_fuse_sequence(0, 8, 16, None, None) != 0
