"""Static checks on the compiled kernels (cuobjdump, no GPU): the properties DESIGN.md sec. 7 relies on.

1. The lens records are read through the uniform datapath (LDCU c[0x0][UR..]) in every fast
   kernel variant -- never through vector-indexed LDC, which would put the constants in vector
   registers and make the lens algebra's FMAs three-register (3-cycle) ones.
2. No local-memory spills, no libdevice slow paths (calls) in the fast variants.
"""
import re
import shutil
import subprocess

import pytest

import paper_2004_06352_b200 as lh

CUOBJDUMP = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"


@pytest.fixture(scope="module")
def sass():
    try:
        out = subprocess.run([CUOBJDUMP, "-sass", lh.library_path()], capture_output=True, text=True, check=True).stdout
    except (OSError, subprocess.CalledProcessError) as e:  # pragma: no cover
        pytest.skip(f"cuobjdump unavailable: {e}")
    funcs, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
        elif name:
            funcs[name].append(line)
    return funcs


FAST = ["ILb1ELb1ELb0ELb0E", "ILb1ELb0ELb0ELb0E", "ILb0ELb1ELb0ELb0E"]  # <GRAD, HESS, EXTREME = false, POINTS = false>


@pytest.mark.parametrize("variant", FAST)
def test_lens_records_come_through_uniform_registers(sass, variant):
    name = next(n for n in sass if "superpose_kernel" in n and variant in n)
    body = "\n".join(sass[name])
    vector_indexed = re.findall(r"LDC(?:\.\d+)? R\d+, c\[0x0\]\[R\d+", body)
    uniform_indexed = re.findall(r"LDCU(?:\.\d+)? UR\d+, c\[0x0\]\[UR\d+", body)
    assert not vector_indexed, f"{name}: {len(vector_indexed)} vector-indexed parameter loads (lens fields in vector registers)"
    assert len(uniform_indexed) >= 10
    assert re.search(r"D(FMA|MUL|ADD) R\d+, [^;]*UR\d+", body), "no FP64 instruction takes a uniform operand"


@pytest.mark.parametrize("variant", FAST)
def test_no_spills_and_no_calls_in_fast_variants(sass, variant):
    name = next(n for n in sass if "superpose_kernel" in n and variant in n)
    body = "\n".join(sass[name])
    assert not re.search(r"\b(STL|LDL)\b", body), "local-memory traffic (register spill)"
    # the only calls allowed are the IEEE-division slow paths of the per-pixel epilogue (mu = 1/det): they may sit
    # inside a loop that holds other loops (a persistent loop over pixel tiles) but in no lens loop
    loops, calls = [], []
    for line in sass[name]:
        m = re.search(r"/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d\s+)?(BRA(?:\.U)?|CALL\S*)\s+(?:!?U?P\d,\s+)?0x([0-9a-f]+)", line)
        if not m:
            continue
        at, op, to = int(m.group(1), 16), m.group(2), int(m.group(3), 16)
        if op.startswith("BRA") and to < at:
            loops.append((to, at))
        if op.startswith("CALL"):
            calls.append(at)
    assert loops

    def is_outer(l):  # a loop that holds other loops (e.g. a persistent loop over pixel tiles) is not a lens loop
        return any(m != l and l[0] <= m[0] and m[1] <= l[1] for m in loops)

    for c in calls:
        inside = [l for l in loops if l[0] <= c <= l[1] and not is_outer(l)]
        assert not inside, "a slow-path call inside a lens loop of a fast variant"


def test_extreme_variants_exist_and_use_libdevice_paths(sass):
    names = [n for n in sass if "superpose_kernel" in n and re.search(r"ILb[01]ELb[01]ELb1ELb[01]E", n)]
    assert len(names) == 6  # grad / hess / both, grid and points


# ---------------------------------------------------------------------------------------------------------------
# bench.py's per-evaluation instruction counts are NOT typed in from a profile: they are recounted here from the
# lens loops of the built library, and the test fails when bench.py and the kernel drift apart.
def _lens_loops(lines):
    """Innermost backward-branch loops of a kernel, in address order, each as a dict opcode -> count."""
    ins = []
    for line in lines:
        m = re.search(r"/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)\s*([^;]*);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2), m.group(3)))
    loops = []
    for at, op, args in ins:
        if op.startswith("BRA"):
            m = re.search(r"0x([0-9a-f]+)", args)
            if m and int(m.group(1), 16) < at:
                loops.append((int(m.group(1), 16), at))
    inner = [l for l in loops if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in loops)]
    out = []
    for lo, hi in sorted(inner):
        ops = {}
        for at, op, _ in ins:
            if lo <= at <= hi:
                ops[op.split(".")[0]] = ops.get(op.split(".")[0], 0) + 1
        if ops.get("DFMA", 0) + ops.get("DMUL", 0) + ops.get("DADD", 0) > 20:  # a lens loop, not a staging loop
            out.append(ops)
    return out


# MUFU seeds per evaluation (lh_math.cuh): they tell how many evaluations one loop iteration holds
_MUFU_PER_EVAL = {"grad+hess": {"dpie": 5, "nsie": 5, "sis": 1}, "grad": {"dpie": 5, "nsie": 4, "sis": 1},
                  "hess": {"dpie": 3, "nsie": 2, "sis": 1}}
_VARIANT = {"ILb1ELb1ELb0ELb0E": "grad+hess", "ILb1ELb0ELb0ELb0E": "grad", "ILb0ELb1ELb0ELb0E": "hess"}


@pytest.mark.parametrize("variant", FAST)
def test_bench_instruction_counts_match_the_built_kernel(sass, variant):
    import bench

    mode = _VARIANT[variant]
    name = next(n for n in sass if "superpose_kernel" in n and variant in n)
    loops = _lens_loops(sass[name])
    assert len(loops) == 3, f"{name}: expected the dPIE, NSIE and SIS loops, found {len(loops)}"
    for cls, ops in zip(("dpie", "nsie", "sis"), loops):
        evals = ops.get("MUFU", 0) / _MUFU_PER_EVAL[mode][cls]
        assert evals == int(evals) and evals >= 1, (cls, ops)
        per_eval = (ops.get("DFMA", 0) / evals, ops.get("DMUL", 0) / evals, ops.get("DADD", 0) / evals)
        assert sum(per_eval) == bench.FP64_INSTR_PER_EVAL_CLASS[mode][cls], (mode, cls, per_eval)
        if cls == "dpie":
            assert per_eval == bench.FP64_OPS_PER_EVAL[mode], (mode, per_eval)
            assert bench.FLOPS_PER_EVAL[mode] == 2 * per_eval[0] + per_eval[1] + per_eval[2]
            assert bench.FP64_INSTR_PER_EVAL[mode] == sum(per_eval)
