"""A memcheck of our own for the superposition kernel (-m gpu): compute-sanitizer is closed on this GPU pool
(profiles/r02_sanitizer.md: "Find a bad access with bounds checks and asserts of your own, small cases, and a
comparison with the CPU reference").  The CHECKING build of the library (same sources, -DLH_BOUNDS_CHECK,
paper_2004_06352_b200/liblh_check.so) compares every global-memory access of superpose_kernel -- carry loads and
stores, statistics read-modify-writes, output stores, point-coordinate and table loads -- with the exact address
ranges each launch may touch, counts and skips anything outside.  tests/bounds_child.py drives it through the
cases that exercise the addressing (ragged grids, lens chunks, row slabs, batches on one and two launch chains,
statistics, shared lenses, points, the host entry points) and compares every result with the oracle."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_no_access_outside_the_buffers_of_a_launch():
    from paper_2004_06352_b200 import _build

    try:
        lib = _build.build_check()
    except (OSError, subprocess.CalledProcessError):  # no compiler on this box: use the library that travelled with the tree
        lib = _build.LIB_CHECK
    assert os.path.exists(lib), "liblh_check.so is missing: run __graft_entry__.build()"
    env = dict(os.environ, LH_LIBRARY=lib)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "bounds_child.py")], env=env, cwd=ROOT,
                       capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-3000:])
    line = next(l for l in r.stdout.splitlines() if l.startswith("BOUNDS_REPORT "))
    rep = json.loads(line[len("BOUNDS_REPORT "):])
    print(line)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "bounds_report.json"), "w") as f:
            json.dump(rep, f, indent=1)
    assert rep["library"] == "liblh_check.so"
    for name, c in rep["cases"].items():
        assert c["violations"] == 0, (name, c)
        assert c["worst_parity_ratio"] <= 1.0, (name, c)
    n = rep["negative_control"]
    assert n["violations"] >= 1 and n["last_element_untouched"] and n["all_others_written"], n
