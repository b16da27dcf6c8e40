"""Multi-GPU slab decomposition, host side: world-size-2 run with the gloo backend on CPU."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_exchange_world_size_2_gloo():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29741",
                        os.path.join(ROOT, "tests", "slab_worker.py")],
                       capture_output=True, text=True, timeout=240, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "rank 0 ok" in r.stdout and "rank 1 ok" in r.stdout


def test_slab_domain_geometry():
    import torch
    from paper_1610_03343_b200 import slab
    d = slab.SlabDomain((80.0, 20.0, 20.0), 4, 3, 3.5)
    x = torch.tensor([0.0, 6.9, 7.1, 59.9, 60.0, 79.9, 46.0, 53.1])
    assert d.owner_of(x).tolist() == [0, 0, 0, 2, 3, 3, 2, 2]
    xl = d.local_x(x)
    assert abs(float(xl[4]) - 7.0) < 1e-12 and abs(float(xl[0]) - 27.0) < 1e-12     # slab start -> halo; x = 0 -> right halo
    assert d.halo_mask(x, d.owner_of(x)).tolist() == [True, True, False, True, False, False, False, True]
    import pytest
    with pytest.raises(ValueError):
        slab.SlabDomain((40.0, 20.0, 20.0), 4, 0, 3.5)                              # 10 A slabs < 4 r_list
