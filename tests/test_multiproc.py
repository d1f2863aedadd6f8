"""N > 1 path on CPU: world_size-2 gloo jobs launched the way the driver launches bench.py."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def torchrun(script_args, nproc=2, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port())] + script_args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def json_lines(text):
    out = []
    for ln in text.splitlines():
        ln = ln.strip()
        if ln.startswith("{") and ln.endswith("}"):
            out.append(json.loads(ln))
    return out


def test_reduce_over_ranks_world_size_2_gloo():
    res = torchrun([os.path.join("tests", "gloo_worker.py")])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = json_lines(res.stdout)
    assert len(lines) == 1
    r = lines[0]
    assert r["world"] == 2
    assert r["ms"] == 15.0 and r["ms_sweeps"] == 8.0 and r["dt"] == 1.0      # MAX over ranks
    assert r["launches"] == 201 and r["attempts"] == 3000 and r["none"] == []  # SUM over ranks
    assert r["seeds"] == [1, 2]                                              # independent replicas


def test_reduce_over_ranks_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([3.5, 1.0], [7], "cpu") == ([3.5, 1.0], [7])


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    res = torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1", "--workload", "c1"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = json_lines(res.stdout)
    assert len(lines) == 1
    r = lines[0]
    assert r["impl"] == "reference" and r["n_gpus"] == 2 and r["steps"] == 2
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["value"] == r["value"]
    assert r["e2e"]["h2d_bytes_per_step"] == 0 and r["e2e"]["d2h_bytes_per_step"] == 0
    assert r["value"] > 0 and r["unit"] == "Gupd/s"
