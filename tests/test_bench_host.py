"""Host logic of bench.py: roofline arithmetic, the replicas aggregation under gloo (world size 2), the reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bytes_per_update():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.bytes_per_update(19, "f64", "2POP_SOA") == 304     # 2*19*8, Eq 16
    assert bench.bytes_per_update(19, "f32", "AA_SOA") == 152
    assert bench.bytes_per_update(19, "f64", "SWAP_SOA") == 592
    assert bench.bytes_per_update(27, "f64", "SWAP_AOS") == 848
    assert bench.bytes_per_update(27, "f64", "AA_AOS") == 432


def test_roofline_arithmetic_reproduces_the_papers_table3():
    """tests/golden/paper_table3_peak_fractions.txt: the paper's own MLUPS and "% of peak" for three GPUs
    (Table 3, Eq 16).  bench.py's bytes per update and MLUPS -> fraction arithmetic
    must give back the printed percentages (they are rounded to integers)."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2010_11751_b200 import sweep
    rows = [l.split("|") for l in open(os.path.join(ROOT, "tests", "golden", "paper_table3_peak_fractions.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 9
    for gpu, bw, code, mlups, pct in rows:
        scheme = "AA_SOA" if "AA" in code else "2POP_SOA"
        bpu = bench.bytes_per_update(19, "f64", scheme)
        assert bpu == sweep.bytes_per_update(19, "f64", scheme) == 2 * 19 * 8
        frac = float(mlups) * 1e6 * bpu / (float(bw) * 1e9)
        assert abs(100.0 * frac - float(pct)) <= 0.6, (gpu, code, 100.0 * frac, pct)


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group(backend="gloo")
r = dist.get_rank()
ms, units = bench.aggregate(dist, 10.0 + 5.0 * r, 1000 * (r + 1))
dist.barrier()
assert ms == 15.0 and units == 3000.0, (ms, units)
print("OK", r)
dist.destroy_process_group()
"""


def test_aggregate_gloo_world2(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29517", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("OK") == 2


def test_reference_arm_prints_one_json_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "1",
                        "--steps", "3", "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "MLUPS" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "1",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_cavity_profile_helpers():
    """host logic of paper_2010_11751_b200/cavity.py: centre lines and the comparison of two resolutions"""
    import numpy as np
    from paper_2010_11751_b200 import cavity
    n = 8
    x, y, z = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    f = 100.0 * x + 10.0 * y + z
    # even n: the centre lies between the nodes 3 and 4 of the two other axes
    assert np.allclose(cavity.centre_line(f, 2), 100 * 3.5 + 10 * 3.5 + np.arange(1, n - 1))
    assert np.allclose(cavity.centre_line(f, 0), 100 * np.arange(1, n - 1) + 10 * 3.5 + 3.5)
    g = f[:7, :7, :7]
    assert np.allclose(cavity.centre_line(g, 1), 100 * 3 + 10 * np.arange(1, 6) + 3)
    pos = cavity.node_positions(n)
    assert pos[0] == 0.5 / 6 and pos[-1] == 1 - 0.5 / 6 and len(pos) == n - 2
    # a profile that is linear between the wall values is reproduced exactly at any resolution
    coarse = {"pos": cavity.node_positions(10).tolist(), "ux_along_z": cavity.node_positions(10).tolist(),
              "uz_along_x": (0.0 * cavity.node_positions(10)).tolist()}
    fine = {"pos": cavity.node_positions(18).tolist(), "ux_along_z": cavity.node_positions(18).tolist(),
            "uz_along_x": (0.0 * cavity.node_positions(18)).tolist()}
    assert cavity.profile_difference(coarse, fine, "ux_along_z") < 1e-15
    assert cavity.profile_difference(coarse, fine, "uz_along_x") == 0.0
    fine["uz_along_x"][3] = 0.25
    assert abs(cavity.profile_difference(coarse, fine, "uz_along_x") - 0.25) < 1e-15
