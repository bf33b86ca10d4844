"""Host-side logic of the multi-rank bench path (replicas only, no data-path collective), on CPU with
the gloo backend and world_size 2: job time = max over ranks, value = whole-job aggregate, reference arm prints on
rank 0 only."""
import importlib.util
import io
import os
import socket
import sys
from contextlib import redirect_stdout

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load_bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    bench = load_bench()
    local_ms = 10.0 * (rank + 1)                 # rank 1 is the slow one
    job_ms = bench.max_over_ranks(local_ms, dist, "cpu")
    out.put((rank, job_ms, bench.whole_job_value(1000, 5, world, job_ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_job_time_is_max_over_ranks_and_value_is_whole_job():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, job_ms, value in res:
        assert job_ms == 20.0                                    # both ranks agree on the slowest rank's time
        assert value == pytest.approx(2 * 1000 * 5 / 20e-3)      # 2 replicas x 1000 atoms x 5 steps in 20 ms


def test_single_rank_helpers():
    bench = load_bench()
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.whole_job_value(1029000, 100, 1, 400.0) == pytest.approx(1029000 * 100 / 0.4)


def test_reference_arm_is_silent_on_other_ranks(monkeypatch):
    bench = load_bench()
    monkeypatch.setenv("RANK", "1")

    class Args:
        steps, warmup, gpus, cpu_sample_side = 1, 0, 2, 10

    buf = io.StringIO()
    with redirect_stdout(buf):
        bench.run_reference(Args())
    assert buf.getvalue() == ""
