"""The N>1 path of bench.py is 'replicas only' (the north_star fixes one GPU, no sharding, no
collective on the data path): every rank runs the same workload and the only exchange is the
max-over-ranks reduction of the timed region.  This covers that host logic with world_size 2 on gloo."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_max_over_ranks_aggregation_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import os, sys, json
        sys.path.insert(0, %r)
        import torch, torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
        val = bench.aggregate_value(dof=1000, ms_step=ms, world=world)
        if rank == 0:
            print(json.dumps({"ms": ms, "val": val}))
        dist.destroy_process_group()
    """ % ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29517")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", "29517", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json

    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["ms"] == 15.0  # the slower rank
    assert abs(d["val"] - 2 * 1000 / 15e-3 / 1e9) < 1e-12
