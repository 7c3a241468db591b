"""world_size-2 gloo test (CPU) of the N>1 timing plumbing bench.py uses: replicas only,
no data-path collective; value = units of all ranks / max-over-ranks time."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["VIBE_ROOT"])
from paper_2606_00735_b200 import dist as D
g = D.init_from_env("gloo")
assert g.world == 2
g.barrier()
ms = 10.0 if g.rank == 0 else 25.0          # rank 1 is the straggler
tput, max_ms = D.aggregate_throughput(g, units_this_rank=4096.0, device_ms_this_rank=ms)
assert max_ms == 25.0, max_ms
assert abs(tput - 8192.0 / 0.025) < 1e-6, tput
assert g.max_over_ranks(g.rank) == 1.0 and g.sum_over_ranks(1.0) == 2.0
g.barrier()
if g.is_main:
    print(json.dumps({"ok": True, "tput": tput}))
g.close()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_rank_gloo_replica_aggregation(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), VIBE_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=120)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert '"ok": true' in outs[0]


def test_single_process_group_is_trivial():
    sys.path.insert(0, ROOT)
    from paper_2606_00735_b200 import dist as D
    env_backup = {k: os.environ.pop(k, None) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    try:
        g = D.init_from_env()
        assert g.world == 1 and g.is_main
        tput, ms = D.aggregate_throughput(g, 100.0, 50.0)
        assert tput == 2000.0 and ms == 50.0
    finally:
        for k, v in env_backup.items():
            if v is not None:
                os.environ[k] = v
