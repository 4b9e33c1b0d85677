"""N > 1 path on CPU: world size 2, gloo backend (tier rule 5: marker shards, no data-path collective)."""
import json
import os
import socket
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(args, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_two_rank_gloo_aggregation(tmp_path):
    """Units are summed, time is the max over ranks, shards tile the marker range, ranks draw different markers."""
    r = _torchrun([os.path.join(HERE, "dist_worker.py"), str(tmp_path)])
    assert r.returncode == 0, r.stderr[-2000:]
    out = [json.load(open(tmp_path / f"rank{k}.json")) for k in range(2)]
    assert [o["world"] for o in out] == [2, 2]
    assert (out[0]["lo"], out[0]["hi"], out[1]["lo"], out[1]["hi"]) == (0, 501, 501, 1001)
    for o in out:
        assert o["agg"]["units"] == 300.0 and o["agg"]["seconds"] == 2.0 and o["agg"]["value"] == 150.0
        assert o["agg"]["launches"] == 7.0 and o["max_all"] == 1.0 and o["sum_all"] == 1.0
    assert out[0]["checksum"] != out[1]["checksum"]
    # row f1: shards projected separately + one all-reduce of the right-hand side = projection of all markers
    assert all(o["scatter_err"] < 1e-13 for o in out)


def test_reference_arm_under_torchrun_prints_one_line():
    """bench.py --impl reference at N = 2: rank 0 alone runs the oracle and prints the line, rank 1 exits 0."""
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "cfg1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
