"""The roofline numerator is tied to the binary: the FP64 instruction count of the innermost (radial, 4 nodes per
trip) loop of every shipped no3n_kernel variant, read from `cuobjdump -sass libno3n.so`, must equal what
bench.py:flops_per_eval puts into `roofline.achieved`.  A kernel edit that changes the loop
body fails here instead of silently skewing `roofline.frac`.  Needs no GPU (cuobjdump reads the cross-compiled
library); the hot loop of the cfg5 variant is committed as profiles/r03a_hotloop_sass.txt, checked below too."""
import os
import re
import shutil
import subprocess

import pytest

import bench
from paper_2603_24532_b200 import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NODES_PER_TRIP = 4          # no_core.h: nodes<> handles four radial nodes per trip of the innermost loop
INS = re.compile(r"^\s*/\*([0-9a-f]{4,})\*/\s+(.*?);", re.M)


def _cuobjdump():
    for cand in (shutil.which("cuobjdump"), "/usr/local/cuda/bin/cuobjdump"):
        if cand and os.path.exists(cand):
            return cand
    pytest.skip("cuobjdump not found")


@pytest.fixture(scope="module")
def functions():
    """{mangled name: [(address, instruction text)]} of every no3n_kernel variant in the built library."""
    lib = build.build()
    text = subprocess.run([_cuobjdump(), "-sass", lib], check=True, capture_output=True, text=True).stdout
    out = {}
    for chunk in re.split(r"\n\s*Function : ", text)[1:]:
        name = chunk.split("\n", 1)[0].strip()
        if "no3n_kernel" in name:
            out[name] = [(int(a, 16), t) for a, t in INS.findall(chunk)]
    return out


def innermost_loops(ins):
    """[(first address, last address)] of the loops (backward branches) that contain no other loop."""
    loops = []
    for addr, text in ins:
        m = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", text)
        if m and int(m.group(1), 16) <= addr:
            loops.append((int(m.group(1), 16), addr))
    return [l for l in loops if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in loops)]


def fp64_counts(ins, lo, hi):
    body = [t for a, t in ins if lo <= a <= hi]
    return tuple(sum(1 for t in body if re.search(r"\b%s\b" % op, t)) for op in ("DFMA", "DMUL", "DADD"))


def hot_loop_counts(ins):
    """(DFMA, DMUL, DADD) of the innermost loop with the most FP64 work, and how many innermost loops share it
    (the guarded and the unguarded copy of the radial loop hold the same arithmetic)."""
    counts = [fp64_counts(ins, lo, hi) for lo, hi in innermost_loops(ins)]
    best = max(counts, key=sum)
    return best, counts.count(best)


def variant(name):
    """template arguments <NREG, C4, WARPS, MINB, SPLIT, FWD> from the mangled name"""
    m = re.search(r"no3n_kernelILi(n?\d+)ELb([01])ELi(\d+)ELi(\d+)ELi(\d+)ELb([01])EEE", name)
    assert m, name
    nreg = -int(m.group(1)[1:]) if m.group(1).startswith("n") else int(m.group(1))
    return nreg, bool(int(m.group(2))), int(m.group(3)), int(m.group(4)), int(m.group(5)), bool(int(m.group(6)))


def test_every_variant_the_launcher_can_pick_is_in_the_library(functions):
    got = {variant(n) for n in functions}
    for nreg in (-1, 0, 1, 2, 3, 4):
        for c4 in (False, True):
            assert {(nreg, c4, 2, 6, 1, False), (nreg, c4, 4, 3, 4, False), (nreg, c4, 2, 6, 1, True)} <= got


def test_hot_loop_fp64_instructions_match_the_bench_flop_table(functions):
    checked = 0
    for name, ins in functions.items():
        nreg, c4, warps, minb, split, fwd = variant(name)
        if nreg == 0:
            continue          # generic exponent (n_reg > 4): not a bench variant, its loop calls a power routine
        (fma, mul, add), copies = hot_loop_counts(ins)
        assert fma % NODES_PER_TRIP == mul % NODES_PER_TRIP == add % NODES_PER_TRIP == 0, (name, fma, mul, add)
        flops = (2 * fma + mul + add) / NODES_PER_TRIP
        regulated = nreg > 0
        want = bench.flops_per_eval(nreg if regulated else 4, regulated, forward=fwd)
        assert flops == want, f"{name}: SASS {fma}/{mul}/{add} per {NODES_PER_TRIP} nodes = {flops} flop per node, bench.py says {want}"
        if regulated:
            assert copies == 2, name       # guarded + unguarded copy of the radial loop
        checked += 1
    assert checked == 5 * 2 * 3


def test_headline_variants_have_the_documented_counts(functions):
    """cfg5 / cfg2-4 run <4, no c4>: 25 DFMA + 16 DMUL + 10 DADD = 51 FP64 instructions = 76 flop per node; the forward
    fast path (Hartree-Fock) 20 + 12 + 7 = 39 instructions = 59 flop; unregulated 15 + 14 + 9 = 53 flop."""
    by = {variant(n): hot_loop_counts(i)[0] for n, i in functions.items()}
    assert by[(4, False, 2, 6, 1, False)] == (100, 64, 40)
    assert by[(4, False, 4, 3, 4, False)] == (100, 64, 40)
    assert by[(4, False, 2, 6, 1, True)] == (80, 48, 28)
    assert by[(-1, False, 2, 6, 1, False)] == (60, 56, 36)
    assert bench.flops_per_eval(4, True) == 76.0 and bench.flops_per_eval(4, True, forward=True) == 59.0
    assert bench.flops_per_eval(4, False) == 53.0


def test_committed_hot_loop_listing_matches_the_library(functions):
    """profiles/r03a_hotloop_sass.txt is the second copy of the radial loop of no3n_kernel<4,0,2,6,1,0> as built from this tree:
    same opcode sequence (register allocation and addresses may move with the compiler, the opcodes may not)."""
    path = os.path.join(ROOT, "profiles", "r03a_hotloop_sass.txt")
    stored = [l.split(";")[0] for l in open(path) if l.lstrip().startswith("/*")]
    stored_ops = [INS.match(l + ";").group(2).split()[0] if not INS.match(l + ";").group(2).startswith("@")
                  else INS.match(l + ";").group(2).split()[1] for l in stored]
    name = next(n for n in functions if variant(n) == (4, False, 2, 6, 1, False))
    ins = functions[name]
    loops = [l for l in innermost_loops(ins) if fp64_counts(ins, *l) == (100, 64, 40)]
    lo, hi = loops[-1]
    ops = [(t.split()[1] if t.startswith("@") else t.split()[0]) for a, t in ins if lo <= a <= hi]
    assert sum(1 for o in stored_ops if o.startswith(("DFMA", "DMUL", "DADD"))) == 204
    assert ops == stored_ops
