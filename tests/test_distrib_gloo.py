"""The N>1 plumbing of bench.py (replicas only) on CPU: world_size 2, gloo.

The path has no data-path collective; what N ranks share is the measurement: a barrier on both
sides of the timed region, the max over ranks of the device-timed milliseconds, and the
aggregate throughput = all ranks' cell-updates / that time.
"""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    from paper_1311_0861_b200 import distrib
    rank, local_rank, world = distrib.env_world()
    assert world == 2 and local_rank == rank
    distrib.init("gloo")
    distrib.barrier()
    ms = distrib.max_over_ranks(10.0 + 5.0 * rank)          # rank 1 is the slow one
    agg = distrib.aggregate_throughput(1000, 4, ms, world)
    distrib.barrier()
    distrib.shutdown()
    print(json.dumps({{"rank": rank, "ms": ms, "agg": agg}}))
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_replica_timing_takes_the_max_and_sums_the_work(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 15.0                                  # max over ranks, seen by every rank
        assert o["agg"] == 2 * 1000 * 4 / 15.0e-3               # whole-job cell-updates/s


def test_single_process_is_a_no_op():
    sys.path.insert(0, ROOT)
    from paper_1311_0861_b200 import distrib
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        assert k not in os.environ or os.environ[k] in ("0", "1")
    assert distrib.env_world()[2] == 1 or os.environ.get("WORLD_SIZE") == "1"
    distrib.barrier()
    assert distrib.max_over_ranks(3.5) == 3.5
    assert distrib.aggregate_throughput(10, 2, 4.0, 1) == 10 * 2 / 4.0e-3


LAUNCHED = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    from paper_1311_0861_b200 import distrib
    rank, local_rank, world = distrib.env_world()
    distrib.init("gloo")
    distrib.barrier()
    ms = distrib.max_over_ranks(7.0 + rank)
    distrib.barrier()
    distrib.shutdown()
    print(json.dumps({{"rank": rank, "local_rank": local_rank, "n_gpus": world, "ms": ms}}))   # every rank prints
""")


def test_launcher_starts_n_ranks_and_only_rank_0_reaches_stdout(tmp_path):
    """`bench.py --gpus N` outside torchrun: distrib.launch_replicas starts the N ranks itself (CPU stub, gloo)."""
    import json
    worker = tmp_path / "stub.py"
    worker.write_text(LAUNCHED.format(root=ROOT))
    driver = tmp_path / "driver.py"
    driver.write_text(textwrap.dedent(f"""
        import sys
        sys.path.insert(0, {ROOT!r})
        from paper_1311_0861_b200 import distrib
        sys.exit(distrib.launch_replicas(3, [sys.executable, {str(worker)!r}], timeout=120))
    """))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_PORT")}
    r = subprocess.run([sys.executable, str(driver)], env=env, capture_output=True, text=True, timeout=180)
    assert r.returncode == 0, r.stderr
    lines = [json.loads(x) for x in r.stdout.strip().splitlines()]
    assert lines == [{"rank": 0, "local_rank": 0, "n_gpus": 3, "ms": 9.0}]      # one line, rank 0's, max over 3 ranks


def test_bench_gpus_flag_goes_through_the_launcher():
    """bench.py hands --gpus N > 1 to the launcher unless torchrun's WORLD_SIZE is already set."""
    text = open(os.path.join(ROOT, "bench.py")).read()
    assert 'args.gpus > 1 and "WORLD_SIZE" not in os.environ' in text and "launch_replicas(args.gpus" in text
