"""bench.py's DRAM-traffic constants are typed in from Nsight Compute captures; unlike the instruction counts
(tests/test_sass_cpu.py recounts those from the SASS) nothing would notice when they and the profile notes they cite
drift apart.  This test reads the figures back out of profiles/*.md and compares (CPU only)."""
import os
import re

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _read(name):
    with open(os.path.join(ROOT, "profiles", name)) as f:
        return f.read()


def _close(a, b, rel=2e-3):
    """the notes print MB with two decimals: half a unit of the last digit (5 kB) on top of the relative slack"""
    return abs(a - b) <= max(rel * max(abs(a), abs(b)), 6e3)


def test_traffic_constants_match_the_profile_notes():
    allc = _read("r02_all_configs_ncu.md")
    # "cfg N, launch K: derived: ... DRAM traffic X MB in this launch."  (cfg 4: the launch with the larger figure)
    per_cfg = {}
    for cfg, mb in re.findall(r"cfg (\d), launch \d+: derived:.*?DRAM traffic ([0-9.]+) MB in this launch", allc):
        per_cfg[int(cfg)] = max(per_cfg.get(int(cfg), 0.0), float(mb) * 1e6)
    for cfg in (0, 1, 2, 4):
        assert cfg in per_cfg, f"no DRAM figure for cfg {cfg} in r02_all_configs_ncu.md"
        assert _close(bench.NCU_TRAFFIC_BYTES[cfg], per_cfg[cfg], 3e-2), (cfg, bench.NCU_TRAFFIC_BYTES[cfg], per_cfg[cfg])
    m = re.search(r"DRAM traffic ([0-9.]+) MB in this launch", _read("r02_cfg3_ncu.md"))
    assert m and _close(bench.NCU_TRAFFIC_BYTES[3], float(m.group(1)) * 1e6), (bench.NCU_TRAFFIC_BYTES[3], m and m.group(1))
    nxt = _read("r03_next_rows_ncu.md")
    sect = {k: nxt[nxt.index(h):] for k, h in (("delens", "## delens_kernel"), ("stats", "## superpose_kernel"))}
    for key, const in (("delens", bench.NCU_TRAFFIC_DELENS_BYTES), ("stats", bench.NCU_TRAFFIC_STATS_BYTES)):
        rd = float(re.search(r"dram__bytes_read.sum`\) \| ([0-9.]+) Mbyte", sect[key]).group(1))
        wr = float(re.search(r"dram__bytes_write.sum`\) \| ([0-9.]+) Mbyte", sect[key]).group(1))
        assert _close(const, (rd + wr) * 1e6), (key, const, rd + wr)
