"""N > 1 is N independent replicas: the only cross-rank code is
bench.py's reduction of (device time, units) -> (max over ranks, sum).  World size 2 over gloo, on CPU."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo")
    r = dist.get_rank()
    ms, units = bench.reduce_over_ranks(10.0 + 5.0 * r, 1000 * (r + 1), dist)
    assert ms == 15.0 and units == 3000, (ms, units)
    cfg0, cfg = bench.replica_config(0), bench.replica_config(r)
    assert cfg["seed"] == cfg0["seed"] + r and {k: v for k, v in cfg.items() if k != "seed"} == \\
        {k: v for k, v in cfg0.items() if k != "seed"}
    dist.barrier()
    dist.destroy_process_group()
    print("rank", r, "ok")
""") % ROOT


def test_rank_reduction_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0, out
        assert "ok" in out


def test_single_process_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.5, 7) == (3.5, 7)
