"""N > 1 path on CPU (gloo, world_size 2): the path shards as REPLICAS ONLY (the paper
is single-card; independent pseudo-fermion sources), so what the ranks
share is host logic only — which source each rank solves, and how the whole-job time (MAX over
ranks) and work (SUM) are formed.  Also: the reference arm under a 2-rank launch prints exactly one
line, from rank 0."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(nproc, script_args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_args
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_source_deal_and_reduction_world2(tmp_path):
    r = _torchrun(2, [os.path.join(ROOT, "tests", "gloo_worker.py"), str(tmp_path)])
    assert r.returncode == 0, r.stderr[-2000:]
    got = [json.load(open(tmp_path / ("rank%d.json" % k))) for k in range(2)]
    assert [g["world"] for g in got] == [2, 2]
    # 2 ranks x 3 steps over 4 sources, dealt round-robin on the global step index
    assert got[0]["sources"] == [0, 1, 2] and got[1]["sources"] == [3, 0, 1]
    for g in got:                                   # every rank sees the same whole-job numbers
        assert g["secs"] == 2.0                      # MAX(1, 2)
        assert g["work"] == [30.0, 14.0]             # SUM
    # N = 1 degenerates to the identity
    sys.path.insert(0, ROOT)
    import torch
    import bench
    assert bench.reduce_over_ranks(torch, None, 1, 0.5, [3, 4], "cpu") == (0.5, [3.0, 4.0])
    assert [bench.source_for(0, 8, k, 4) for k in range(8)] == [0, 1, 2, 3, 0, 1, 2, 3]


def test_reference_arm_two_ranks_prints_one_line():
    r = _torchrun(2, [os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c2",
                      "--steps", "1", "--warmup", "0", "--ref-seconds", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
