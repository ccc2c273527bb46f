"""Pin T9: the instruction count of the inner loop, read from the SASS of the built library.

PAPER.md Table I: the per-pixel exponent goes from 3 SUB + 8 MUL + 1 ADD to "5 FMA"; the blend goes
from 7 MUL + 3 ADD + 2 SUB + 2 branches to "4 FMA".  The B200 kernel evaluates TWO horizontally adjacent pixels per thread
and walks TWO list entries per loop iteration.  The two pixels share their row, so V_hoisted . B_local (Eq. 9-10) is
evaluated in the separable form (A x' + H) x' + G with H = B y' + D and G = C y'^2 + E y' + F common to both pixels: per
iteration the hot path must hold exactly
    exponent: 2 entries x (3 scalar FFMA [H, G] + 2 FFMA2 [two pixels])      -- 3.5 issue slots per pixel, Table I has 5
    blend:    2 entries x (1 FMUL2 [w = alpha T] + 4 FFMA2 [T -= w; C_rgb += f w])
    alpha:    2 entries x 2 pixels x 1 MUFU.EX2
and no other scalar FFMA / FMUL / FADD.  CPU-only: needs cuobjdump and the object file build() produced.
"""
import os
import re
import shutil
import subprocess

import pytest

from paper_2606_16566_b200 import build as gs_build

INSTR = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)\s*(.*?);")


def _sass(function_substr):
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    gs_build.build()
    obj = os.path.join(gs_build.OBJ, "render_b200.o")
    out = subprocess.run([exe, "-sass", obj], check=True, capture_output=True, text=True).stdout
    ins, on = [], False
    for line in out.splitlines():
        if "Function :" in line:
            on = function_substr in line
            continue
        if on:
            m = INSTR.match(line)
            if m:
                ins.append((int(m.group(1), 16), m.group(2), m.group(3)))
    assert ins, "kernel %s not found in %s" % (function_substr, obj)
    return ins


def _blend_loops(ins):
    """Innermost loops (backward branch target .. branch) that contain MUFU.EX2; the region a forward branch inside the
    loop jumps over when its predicate is false (the rare repair block behind the warp vote) is not on the hot path."""
    loops = []
    for k, (addr, op, args) in enumerate(ins):
        if op == "BRA":
            m = re.search(r"0x([0-9a-f]+)", args)
            if m and int(m.group(1), 16) <= addr:
                loops.append((int(m.group(1), 16), addr))
    inner = [l for l in loops if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in loops)]
    res = []
    for lo, hi in inner:
        body = [i for i in ins if lo <= i[0] <= hi]
        if not any(op == "MUFU.EX2" for _, op, _ in body):
            continue
        skip = []
        for addr, op, args in body:
            if op == "BRA":
                m = re.search(r"0x([0-9a-f]+)", args)
                t = int(m.group(1), 16)
                if addr < t <= hi:
                    skip.append((addr, t))
        hot = [i for i in body if not any(a < i[0] < t for a, t in skip)]
        res.append(hot)
    return res


def _count(hot, prefix):
    return sum(1 for _, op, _ in hot if op.startswith(prefix))


@pytest.mark.parametrize("kernel,slots", [("render_b200_kernelILb0ELb0E", 23), ("render_b200_kernelILb1ELb0E", 32)])   # without / with per-pixel counts
def test_blend_loop_is_7_fma_slots_exponent_and_4_fma_blend_per_entry(kernel, slots):
    loops = _blend_loops(_sass(kernel))
    assert len(loops) >= 1
    hot = min(loops, key=len)                        # the GUARD = false instance (the common path): no guard selects
    n_ex2 = _count(hot, "MUFU.EX2")
    assert n_ex2 % 2 == 0 and n_ex2 >= 2
    entries = n_ex2 // 2                             # two pixels per thread
    assert _count(hot, "FFMA2") == entries * (2 + 4), (_count(hot, "FFMA2"), entries)
    assert _count(hot, "FMUL2") == entries * 1
    for scalar, want in (("FFMA", 3 * entries), ("FMUL", 0), ("FADD", 0)):   # exact mnemonic or with modifiers, not the packed forms
        n = sum(1 for _, op, _ in hot if re.fullmatch(scalar + r"(\.[A-Z0-9.]+)?", op))
        assert n == want, "%d scalar %s in the blend loop, expected %d" % (n, scalar, want)
    # one warp vote (the R1 termination test), no other branch than the loop's own and the vote's
    assert _count(hot, "VOTE") == 1
    assert _count(hot, "BRA") <= 2
    # the whole iteration stays small (Table I counts 9 arithmetic instructions per pixel and entry; here 12 for two pixels)
    assert len(hot) <= slots * entries, len(hot)
