"""N > 1 path of bench.py on CPU: world_size-2 gloo processes run the replica timing protocol
(barrier, max over ranks, aggregate rate).  The hot path itself does not shard."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    from paper_2606_30985_b200 import replicas as R
    n = R.init("gloo")
    _, rank, _ = R.world()
    R.barrier()
    ms = 10.0 + 5.0 * rank                  # rank 1 is the slow replica
    ms_max = R.max_over_ranks(ms)
    assert abs(ms_max - 15.0) < 1e-12, ms_max
    rate = R.aggregate_rate(3, ms_max, n)
    assert abs(rate - 2 * 3 / 15e-3) < 1e-9, rate
    R.barrier()
    R.finish()
    print("rank", rank, "ok")
""") % ROOT


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_gloo_replicas(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for rank, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok" % rank in o


def test_single_process_is_a_noop():
    from paper_2606_30985_b200 import replicas as R
    assert R.max_over_ranks(7.5) == 7.5
    assert R.aggregate_rate(5, 100.0, 1) == 50.0


def test_bench_gpus_flag_spawns_one_replica_per_gpu(monkeypatch):
    """`python bench.py --gpus N` run directly (WORLD_SIZE unset) must start N replica processes itself:
    it re-launches the same command line under torch.distributed.run with --nproc-per-node N on 127.0.0.1."""
    import importlib
    sys.path.insert(0, ROOT)
    bench = importlib.import_module("bench")
    seen = {}
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "3", "--warmup", "3"])
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    assert bench.main() == 0
    cmd = seen["cmd"]
    assert "torch.distributed.run" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-6:] == ["--gpus", "4", "--steps", "3", "--warmup", "3"]
    # under torchrun (WORLD_SIZE set) the same flag does not spawn again
    monkeypatch.setenv("WORLD_SIZE", "4")
    seen.clear()
    monkeypatch.setattr(bench, "run_ours", lambda a: ({"ok": 1}, 1, 4))
    import paper_2606_30985_b200.replicas as R
    monkeypatch.setattr(R, "finish", lambda: None)
    assert bench.main() == 0 and "cmd" not in seen
