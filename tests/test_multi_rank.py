"""The N > 1 path on CPU: two processes over `gloo`, the same plumbing bench.py uses under torchrun --
job sharding with no data-path collective, a barrier, max-over-ranks step time and summed unit count."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, os.environ["SET_REPO_ROOT"])
    from paper_2606_05495_b200 import multi
    rank, local_rank, world = multi.init_process_group("gloo")
    assert world == 2 and rank == int(os.environ["RANK"])
    multi.barrier("cpu")
    weak = list(multi.shard_jobs(10, rank, world, "weak"))
    strong = list(multi.shard_jobs(11, rank, world, "strong"))
    # rank r pretends its step took (r + 1) * 10 ms and processed len(strong) jobs
    ms, units = multi.aggregate((rank + 1) * 10.0, float(len(strong)), "cpu")
    multi.barrier("cpu")
    print(json.dumps({"rank": rank, "weak": weak, "strong": strong, "ms": ms, "units": units}), flush=True)
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(world, code=None, argv=None, extra_env=None):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), SET_REPO_ROOT=ROOT, **(extra_env or {}))
        cmd = [sys.executable, "-c", code] if code else [sys.executable] + argv
        procs.append(subprocess.Popen(cmd, env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    return outs


def test_two_ranks_shard_and_aggregate_over_gloo():
    outs = [json.loads(o.strip().splitlines()[-1]) for o in _spawn(2, code=WORKER)]
    outs.sort(key=lambda r: r["rank"])
    # weak scaling: every rank has its own 10 jobs, ids disjoint
    assert outs[0]["weak"] == list(range(0, 10)) and outs[1]["weak"] == list(range(10, 20))
    # strong scaling: home GPU = job_id mod world; together the ranks cover every job exactly once
    assert outs[0]["strong"] == [0, 2, 4, 6, 8, 10] and outs[1]["strong"] == [1, 3, 5, 7, 9]
    assert sorted(outs[0]["strong"] + outs[1]["strong"]) == list(range(11))
    for r in outs:
        assert r["ms"] == 20.0          # max over ranks, never the local time
        assert r["units"] == 11.0       # sum over ranks


def test_shard_jobs_single_rank_and_bad_arguments():
    import pytest
    from paper_2606_05495_b200 import multi
    assert list(multi.shard_jobs(5, 0, 1, "weak")) == [0, 1, 2, 3, 4] == list(multi.shard_jobs(5, 0, 1, "strong"))
    assert multi.aggregate(3.5, 7.0) == (3.5, 7.0)      # no process group: identity
    with pytest.raises(ValueError):
        multi.shard_jobs(5, 2, 2)
    with pytest.raises(ValueError):
        multi.shard_jobs(5, 0, 1, "neither")


def test_reference_arm_under_two_ranks_prints_once():
    """bench.py --impl reference under a 2-rank launch: rank 0 alone runs the oracle and prints the line, rank 1 exits 0."""
    outs = _spawn(2, argv=["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "0"])
    lines = [o.strip().splitlines()[-1] for o in outs if o.strip()]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["metric"] == "jobs/s" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
