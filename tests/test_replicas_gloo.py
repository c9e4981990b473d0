"""N > 1 path of the benchmark on CPU: world_size-2 gloo processes exercise the barrier, the
max-over-ranks timing and the whole-job rate (replicas only, no data-path collective)."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2507_19141_b200.replicas import Replicas
    rep = Replicas(backend="gloo")
    rep.barrier()
    ms_local = 2.0 if rank == 0 else 3.5            # rank 1 is the slow one
    rate, ms = rep.whole_job_rate(1_000_000, ms_local)
    q.put((rank, rep.is_reporter, rep.max_over_ranks(float(rank)), rate, ms))
    rep.barrier()
    rep.close()


def test_two_rank_gloo_replicas():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [True, False]                    # only rank 0 reports
    for _, _, mx, rate, ms in got:
        assert mx == 1.0 and ms == 3.5                             # max over ranks, same on both
        assert abs(rate - 2 * 1_000_000 / 3.5e-3) < 1e-3           # whole-job units / slowest time


def test_single_process_is_identity():
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2507_19141_b200.replicas import Replicas
    rep = Replicas()
    assert rep.world == 1 and rep.is_reporter
    rate, ms = rep.whole_job_rate(500, 2.0)
    assert ms == 2.0 and rate == 500 / 2e-3
    rep.barrier()


def test_bench_launcher_starts_n_ranks_itself():
    """`python bench.py --gpus 2` with no torchrun wrapper must start 2 ranks.  The launcher path
    is the product's; `--impl plumbing` swaps the CUDA step for a gloo barrier so it runs on the CPU box."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR",
                                                              "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "plumbing"],
                         env=env, capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                          # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["config"]["parallelism"] == "replicas x2"
    assert lines[0]["max_over_ranks_ms"] == 2.0                     # rank 1's value won the MAX


def test_bench_refuses_a_rank_count_that_contradicts_gpus():
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "plumbing"],
                         env=env, capture_output=True, text=True, timeout=120)
    assert res.returncode != 0 and "WORLD_SIZE" in res.stderr
