"""Host-side logic of bench.py: the C2 stream generator, the reference arm's JSON contract and the N>1 reduction
(world_size-2 gloo run on CPU: max over ranks of the timed seconds, sum of the routed requests)."""
import json
import os
import subprocess
import sys

import numpy as np

from conftest import ROOT

sys.path.insert(0, ROOT)


def test_c2_stream_shape():
    import bench
    from paper_2606_17949_b200 import synth
    sizes, elapsed, weights = bench.c2_stream(synth.CONFIGS["C2"], 400)
    assert len(sizes) == len(elapsed) == len(weights) == 400
    assert 4 <= min(sizes) and max(sizes) <= 64
    assert np.mean(sizes[:200]) < np.mean(sizes[200:])          # 12 req/s windows are smaller than 30 req/s windows
    assert all(e >= 0 for e in elapsed)
    assert set(weights) == set(synth.PRESETS.values())


_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%d" %% int(sys.argv[2]), rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
t, u = bench.reduce_over_ranks(dist, "cpu", seconds=1.0 + rank, units=100 * (rank + 1), backend_is_gloo=True)
print(json.dumps({"rank": rank, "t": t, "u": u}))
dist.destroy_process_group()
"""


def test_reduce_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    port = 29500 + (os.getpid() % 2000)
    procs = [subprocess.Popen([sys.executable, str(script), str(r), str(port)], stdout=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=120)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for o in outs:
        j = json.loads(o.strip().splitlines()[-1])
        assert j["t"] == 2.0 and j["u"] == 300.0        # max over ranks, sum over ranks


def test_reference_arm_contract():
    """bench.py --impl reference times the oracle and prints the contract's JSON line (tiny K so it stays quick)."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    j = json.loads(out.stdout.strip().splitlines()[-1])
    assert j["impl"] == "reference" and j["unit"] == "requests/s" and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["d2h_bytes_per_step"] == 0
    assert j["gpu_launches"] == 0
