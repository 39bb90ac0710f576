"""Host-side tests of the post-link operand-reuse pass (paper_1811_05903_b200/sass_reuse.py)."""
import shutil

import pytest

from paper_1811_05903_b200 import build, sass_reuse

A, B, C = (1 << 58), (1 << 59), (1 << 60)
NY = 1 << sass_reuse.NO_YIELD_BIT


def _ins(texts):
    return [(16 * i, t, 0, 0) for i, t in enumerate(texts)]


def test_adjacent_pair_sharing_a_slot_gets_the_hint():
    p = sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "DFMA R12, R4, R20, R12", "DFMA R14, R6, R20, R14"]))
    assert p == {0: B | NY, 1: B | NY}


def test_same_register_in_a_different_slot_is_not_reuse():
    assert sass_reuse.plan(_ins(["DFMA R10, R20, R2, R10", "DFMA R12, R4, R20, R12"])) == {}


def test_overwritten_operand_is_not_reused():
    # the first instruction overwrites R20 itself; an integer instruction in between overwrites R21 (upper half)
    assert sass_reuse.plan(_ins(["DFMA R20, R2, R20, R10", "DFMA R12, R4, R20, R12"])) == {}
    assert sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "IMAD.MOV.U32 R21, RZ, RZ, RZ", "DFMA R12, R4, R20, R12"])) == {}


def test_neutral_instruction_in_between_keeps_the_pair_and_others_break_it():
    assert sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "ISETP.NE.AND P0, PT, R40, 0x100, PT",
                                 "DFMA R12, R4, R20, R12"])) == {0: B | NY}
    assert sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "LDS.128 R40, [R60]", "DFMA R12, R4, R20, R12"])) == {}
    assert sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "BRA.U UP0, 0x1000", "DFMA R12, R4, R20, R12"])) == {}


def test_branch_target_and_predication_reset_the_pair():
    # 0x10 is a branch target: another path may reach the second instruction
    assert sass_reuse.plan(_ins(["DFMA R10, R2, R20, R10", "DFMA R12, R4, R20, R12", "@P0 BRA 0x10"])) == {}
    assert sass_reuse.plan(_ins(["@P1 DFMA R10, R2, R20, R10", "DFMA R12, R4, R20, R12"])) == {}


def test_packed_pair_and_broadcast_scalar_of_the_same_number_differ():
    t = ["FFMA2 R10, R2.F32x2.HI_LO, R20.F32, R30.F32", "FFMA2 R12, R4.F32x2.HI_LO, R20.F32x2.HI_LO, R30.F32"]
    assert sass_reuse.plan(_ins(t)) == {0: C | NY}


def test_already_flagged_instruction_is_left_alone():
    ins = [(0, "DFMA R10, R2, R20.reuse, R10", 0, B | NY), (16, "DFMA R12, R4, R20, R12", 0, 0)]
    assert sass_reuse.plan(ins) == {}


@pytest.mark.skipif(shutil.which("cuobjdump") is None and shutil.which("/usr/local/cuda/bin/cuobjdump") is None,
                    reason="cuobjdump not available")
def test_built_library_is_calibrated_and_fully_patched():
    lib = build.build()
    funcs = sass_reuse.disassemble(lib)
    sass_reuse._calibrate(funcs)                      # bit assignment agrees with every flag in the library
    names = [n for n in funcs if any(p in n for p in sass_reuse.KERNEL_PATTERNS)]
    assert len(names) >= 4
    for n in names:
        assert sass_reuse.plan(funcs[n]) == {}, n     # the build step left nothing to patch (idempotent)
    # the fp64 far loop: every accumulate triple shares s through the reuse cache
    text = [t for _, t, _, _ in funcs[[n for n in names if "persistent" in n and "Fp64" in n and "Li4ELi0E" in n][0]]]
    assert sum(".reuse" in t and t.startswith("DFMA") for t in text) >= 20
