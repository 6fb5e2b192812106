"""The N>1 host logic of bench.py (replica plan, max-over-ranks timing, aggregate value) on the gloo backend,
world_size 2, CPU only.  The path shards as independent replicas: there is no data-path collective to test."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import bench
    r, l, w = bench.dist_init("gloo")
    plan = bench.replica_plan(r, w, 2048)
    ms = 10.0 + 5.0 * r                       # rank 1 is slower
    ms_max = bench.dist_max(ms)
    tot = bench.dist_sum(float(plan["tokens"]))
    bench.dist_barrier()
    q.put((r, plan, ms_max, tot))


def test_two_rank_replicas_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r, plan, ms_max, tot in res:
        assert ms_max == 15.0                                  # max over ranks, not this rank's own time
        assert plan["global_tokens"] == 4096 == tot            # whole-job aggregate
        assert plan["x_stream"] == f"rank{r}"                  # each replica draws its own batch
    assert res[0][1]["x_stream"] != res[1][1]["x_stream"]


def test_reference_arm_prints_contract_line(capsys, monkeypatch):
    sys.path.insert(0, ROOT)
    import json
    import bench
    import workloads as wl
    # shrink the workload so the CPU suite stays fast; the arm itself is unchanged
    monkeypatch.setitem(wl.CONFIGS, "tiny_ref", wl.scaled(wl.CONFIGS["tiny"], name="tiny_ref"))
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--workload", "tiny_ref", "--steps", "1",
                                      "--warmup", "0", "--ref-tokens", "16"])
    ap_choices = sorted(wl.CONFIGS)
    assert "tiny_ref" in ap_choices
    bench.main()
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "tokens/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
