"""The N > 1 path of bench.py on CPU: two `gloo` ranks run the replica plumbing.
The data path has no collective; torch.distributed only brackets the timed region with a barrier and reduces the
per-rank device time to its maximum, and `value` = units of all ranks / that time."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    from paper_2203_02479_b200 import replicas
    rank, local_rank, world = replicas.env_world()
    assert world == 2 and local_rank == rank
    assert replicas.init("gloo") == 2
    replicas.barrier()
    # rank r "processed" 100 (r + 1) units in 0.5 (r + 1) s: whole job = 300 units / max time 1.0 s
    value, slowest = replicas.whole_job_throughput(100.0 * (rank + 1), 0.5 * (rank + 1))
    assert abs(slowest - 1.0) < 1e-12 and abs(value - 300.0) < 1e-9, (value, slowest)
    assert replicas.max_over_ranks(float(rank)) == 1.0
    assert replicas.sum_over_ranks(1.0) == 2.0
    replicas.barrier()
    replicas.shutdown()
    print(json.dumps({"rank": rank, "value": value}))
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_ranks_agree_on_whole_job_throughput(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err
        assert '"value": 300.0' in out


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_2203_02479_b200 import replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        assert k not in os.environ or os.environ[k] in ("0", "1")
    assert replicas.env_world()[2] in (1,)
    assert replicas.init("gloo") == 1
    replicas.barrier()  # no-op
    value, slowest = replicas.whole_job_throughput(50.0, 0.25)
    assert value == 200.0 and slowest == 0.25
