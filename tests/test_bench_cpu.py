"""Host-side logic of bench.py that needs no GPU: the reference arm under a 2-rank launch (rank 0 alone
works and prints ONE JSON line; the other rank exits 0), the JSON contract keys, the flop bookkeeping."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_two_ranks_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29617", os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "3", "--warmup", "0", "--ref-box", "40"]
    env = dict(os.environ, OMP_NUM_THREADS="4")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "Mcell-steps/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["higher_is_better"] is True
    assert d["n_gpus"] == 2 and d["dtype"] == "f64" and "workload" in d["config"]
    assert d["steps"] == 3 and d["config"]["steps_timed"] == 2          # bounded: min(K, 2) oracle steps are timed


def test_flop_bookkeeping_matches_design():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.FLOPS_PER_FACE[True] == 518 + 968 + 2824 + 416
    assert bench.FLOPS_PER_FACE[False] == 518 + 968 + 2824 + 344
    assert abs(bench.FLOPS_PER_CELL_STEP - 28200) < 100
