"""N > 1 path of bench.py on CPU: two gloo ranks (DESIGN.md sec. 8 -- the hot path does not shard, so
`--gpus N` is N independent replicas; what the ranks share is the barrier, the max-over-ranks time and
the whole-job aggregation, and in the reference arm only rank 0 works)."""
import io
import os
import sys
from contextlib import redirect_stdout

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow replica
    dist.barrier()
    ms = bench.reduce_max(ms_local, world)
    value = bench.job_value(1000, 3, ms, world)
    # reference arm: ranks other than 0 print nothing and do no work
    out = io.StringIO()
    if rank != 0:
        class A:
            steps, warmup, gpus, config = 1, 0, world, 5
        with redirect_stdout(out):
            bench.run_reference(A, rank)
    q.put((rank, ms, value, out.getvalue()))
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value, out in res:
        assert ms == 15.0                               # max over ranks, on every rank
        assert value == pytest.approx(2 * 1000 * 3 / 0.015)
        assert out == ""


def test_capture_hash_covers_host_code_flags_and_switches(monkeypatch):
    """bench.py trusts the per-launch DRAM bytes of profiles/traffic.json only while ncu_summary.source_sha() is
    unchanged: the hash must move with hydro_api.cu (ring depths, grids, species grouping), with the build flags and
    with every run-time switch of include/hydro.h."""
    from paper_2007_05218_b200 import ncu_summary as N
    hdr = open(os.path.join(ROOT, "include", "hydro.h")).read()
    import re
    assert set(re.findall(r"^ \*   (HYDRO_[A-Z_]+)=", hdr, flags=re.M)) == set(N.KNOBS)
    assert "hydro_api.cu" in N.PATH_SOURCES
    for k in N.KNOBS:
        monkeypatch.delenv(k, raising=False)
    base = N.source_sha()
    for k in N.KNOBS:
        monkeypatch.setenv(k, "2")
        assert N.source_sha() != base, k
        monkeypatch.delenv(k)
    assert N.source_sha() == base
    monkeypatch.setattr(N, "build_flags", lambda: "fmad=0 extra=")
    assert N.source_sha() != base


def test_plain_gpus_2_invocation_starts_two_ranks():
    """`python bench.py --gpus 2` with no launcher around it must itself start one rank per GPU (it used to run ONE
    replica and print n_gpus 1).  --dry-run stops before CUDA: the ranks join a gloo group and rank 0 prints the
    line's skeleton, which must show both ranks, the max over ranks and the whole-job aggregate."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                     # rank 0 alone prints
    line = lines[0]
    assert line["dry_run"] is True and line["n_gpus"] == 2 and line["ranks"] == [0, 1]
    assert line["max_over_ranks_check_ms"] == 2.0          # ranks report 1.0 and 2.0: the slower one counts
    assert line["replica_aggregate_check"] == 2.0          # value = the zones of BOTH replicas over that time
    one = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--dry-run"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert one.returncode == 0 and json.loads(one.stdout.splitlines()[-1])["n_gpus"] == 1
