"""The N > 1 launch contract of bench.py, on CPU: the path is "replicas only", so
the only multi-rank host logic is who prints.  Under torch.distributed.run with two ranks the reference
arm must print exactly one JSON line (rank 0) and the other rank must exit 0 without working."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(cmd, env=None):
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def json_lines(text):
    out = []
    for line in text.splitlines():
        line = line.strip()
        if line.startswith("{") and line.endswith("}"):
            try:
                out.append(json.loads(line))
            except ValueError:
                pass
    return out


def test_reference_arm_single_process_line_has_the_contract_keys():
    r = run([sys.executable, "bench.py", "--impl", "reference", "--config", "0", "--steps", "3", "--warmup", "3"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["unit"] == "atom-steps/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["steps"] == 3 and d["n_gpus"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["config"]["workload"] == "cfg1_tersoff_512"


def test_reference_arm_under_torchrun_two_ranks_prints_once():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731", "bench.py", "--impl", "reference",
           "--gpus", "2", "--config", "0", "--steps", "3", "--warmup", "3"]
    r = run(cmd)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [d for d in json_lines(r.stdout) if d.get("impl") == "reference"]
    assert len(lines) == 1
    assert lines[0]["n_gpus"] == 2 and lines[0]["value"] > 0
