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


def _gloo_worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mine = [10.0 + rank, 5.0 - rank, 7.0, 100.0 * (rank + 1)]
    got = bench.max_over_ranks(mine, "cpu", world)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, got))


def test_max_over_ranks_and_aggregate_with_gloo_world_size_2():
    """The replicas' timing reduction (bench.py, N > 1): every rank ends up with the slowest rank's
    times, and the job value counts all replicas' atoms against that time."""
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    import bench
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_gloo_worker, args=(r, 2, 29733, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert res[0] == res[1] == [11.0, 5.0, 7.0, 200.0]
    assert bench.max_over_ranks([3.0, 4.0], "cpu", 1) == [3.0, 4.0]
    assert bench.aggregate_value(512000, 10, 2, 2.0) == 2 * 512000 * 10 / 2e-3
