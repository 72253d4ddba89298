"""N > 1 host logic of bench.py on CPU: world_size 2, gloo.  The path does not shard (replicas
only), so what there is to check is: every rank gets its own seeded design, the job's time is the max over ranks, the
whole-job value counts every replica's cell updates, and `--impl reference` runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = bench.make_workload("C1", 40, seed_offset=bench.replica_seed_offset(rank))
    local_ms = [10.0 + 5.0 * rank, 4.0 - rank, 6.0 + 6.0 * rank]          # rank 1 is slower overall, faster forward
    tot, f, r = bench.reduce_max(local_ms, world)
    dist.barrier()
    out.put((rank, float(w.eps[8:24, 8:24, 8:24].sum()), tot, f, r, bench.whole_job_value(w.cells, w.nsteps, 3, world, tot)))
    dist.destroy_process_group()


def test_two_replicas_on_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, e0, t0, f0, b0, v0), (r1, e1, t1, f1, b1, v1) = res
    assert (r0, r1) == (0, 1)
    assert e0 != e1                                   # different seeded designs per replica
    assert t0 == t1 == 15.0 and f0 == f1 == 4.0 and b0 == b1 == 12.0   # max over ranks, per entry
    expect = 32 ** 3 * 40 * 3 * 2 / (15.0e-3) / 1e6   # both replicas' cell updates over the slowest replica's time
    assert abs(v0 - expect) < 1e-9 * expect and v0 == v1


def test_single_process_reduce_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max([1.5, 2.5], 1) == [1.5, 2.5]
    assert np.isclose(bench.whole_job_value(1000, 10, 2, 1, 1.0), 1000 * 10 * 2 / 1e-3 / 1e6)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1",
                        "--steps", "1", "--warmup", "0", "--ref-steps", "10"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "Mcell-updates/s"


def test_design_map_chain_rule_matches_finite_differences():
    """optimize.py (harness): filter + projection + broadcast and their hand-written backward pass."""
    import numpy as np
    from paper_2603_24027_b200 import optimize as O, workloads as W
    w = W.c2(nsteps=8)
    des = O.Design(w)
    rng = np.random.default_rng(3)
    rho = rng.uniform(0.2, 0.8, (des.nx, des.ny))
    c = rng.standard_normal((des.nx, des.ny, des.nzl))           # loss = <c, eps on the design box>
    lo, hi = w.design
    box = (slice(lo[0], hi[0]), slice(lo[1], hi[1]), slice(lo[2], hi[2]))

    def loss(r):
        eps, _ = des.forward(r, 3.0)
        return float(np.sum(c * eps[box].astype(np.float64)))
    des.forward(rho, 3.0)
    g = des.backward(c)
    for (i, j) in [(0, 0), (5, 17), (40, 63), (63, 31)]:
        h = 1e-3
        rp, rm = rho.copy(), rho.copy()
        rp[i, j] += h
        rm[i, j] -= h
        fd = (loss(rp) - loss(rm)) / (2 * h)
        assert abs(fd - g[i, j]) <= 2e-3 * max(abs(fd), 1e-3), (i, j, fd, g[i, j])
