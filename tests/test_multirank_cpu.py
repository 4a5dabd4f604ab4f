"""The N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").

The level step has no data-path collective; what N ranks share is (1) a barrier on both sides of a timed region, (2) the max
over ranks of its duration, which every rank must receive, (3) the whole-job rate = N x the per-rank work / that maximum,
printed by rank 0 alone, and (4) in the reference arm, rank 0 alone runs the oracle while the other ranks exit 0 without
work or output.  bench.py's own helpers are driven here by two real processes."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def launch(world, argv, extra_env=None):
    port = free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), **(extra_env or {}))
        procs.append(subprocess.Popen([sys.executable] + argv, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


WORKER = textwrap.dedent("""
    import json, sys, time
    import bench
    rank, world, local, dist = bench.init_ranks("gloo")
    assert world == 2 and dist is not None and rank == local
    # (1) barrier: rank 1 arrives 0.4 s late; nobody leaves before it has arrived
    if rank == 1:
        time.sleep(0.4)
    t_arrive = time.time()
    dist.barrier()
    t_leave = time.time()
    # (2) max over ranks of a per-rank duration, received by every rank
    mine = 3.0 if rank == 0 else 5.0
    worst = bench.max_over_ranks(mine, dist, "cpu")
    # (3) whole-job rate from the per-rank work and the slowest rank
    rate = bench.job_rate(1000.0, world, worst * 1e-3)
    import torch
    arr = torch.tensor([t_arrive], dtype=torch.float64); dist.all_reduce(arr, op=dist.ReduceOp.MAX)
    if rank == 0:
        print(json.dumps({"rank": rank, "worst": worst, "rate": rate, "left_after_last_arrival": t_leave >= arr.item() - 1e-3}))
    else:
        assert worst == 5.0 and t_leave >= arr.item() - 1e-3
    dist.barrier()
    dist.destroy_process_group()
""")


def test_two_ranks_gloo_barrier_max_and_rate(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text("import sys; sys.path.insert(0, %r)\n" % ROOT + WORKER)
    res = launch(2, [str(w)])
    for rc, out, err in res:
        assert rc == 0, err[-2000:]
    assert res[1][1].strip() == ""                                   # rank 1 prints nothing
    d = json.loads(res[0][1].strip().splitlines()[-1])
    assert d["worst"] == 5.0                                          # the slowest rank's time, not rank 0's own 3.0
    assert d["rate"] == 2 * 1000.0 / 5.0e-3                           # N x per-rank work / max time
    assert d["left_after_last_arrival"]


def test_single_process_needs_no_group():
    import bench
    env = {k: os.environ.pop(k) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK") if k in os.environ}
    try:
        rank, world, local, dist = bench.init_ranks("gloo")
        assert (rank, world, local, dist) == (0, 1, 0, None)
        assert bench.max_over_ranks(7.5, None) == 7.5 and bench.job_rate(10.0, 1, 2.0) == 5.0
    finally:
        os.environ.update(env)


def test_reference_arm_runs_on_rank_0_only():
    """bench.py --impl reference under torchrun's environment with 2 ranks: rank 0 times the oracle and prints the one JSON
    line (n_gpus as given); rank 1 exits 0 with no output and without building or touching the oracle's work"""
    res = launch(2, ["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--n", "1024"])   # a small level: CPU suite
    for rc, out, err in res:
        assert rc == 0, err[-2000:]
    assert res[1][1].strip() == ""
    lines = [l for l in res[0][1].strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["steps"] == 1 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == (os.cpu_count() or 1) and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["gpu_launches"] == 0 and d["vs_baseline"] is None
