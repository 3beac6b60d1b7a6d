"""Multi-GPU host logic on CPU: world_size-2 `gloo` processes.

Chains are independent (eq 54; "we can use multiple GPUs in parallel",
line 483): the ensemble is sharded by contiguous ranges of the GLOBAL chain index and the only
exchange of the path is the integer sum of the fixed-point stress sums.  Here each rank
produces the sums of ITS chain range with the oracle (the GPU kernels are not available on
the CPU box), converts them to the library's int64 fixed point, all-reduces them with the
product's `shard.allreduce_sums`, and the result must equal the single-process ensemble
bit for bit -- integer addition commutes, so the number of ranks cannot matter."""
import os
import socket

import numpy as np
import pytest

from paper_1106_2899_b200 import shard


def test_ranges_partition_the_ensemble():
    for total, world in ((10, 3), (1 << 20, 8), (7, 7), (5, 8)):
        ends = [shard.strong_range(total, r, world) for r in range(world)]
        assert ends[0][0] == 0 and ends[-1][1] == total
        assert all(ends[r][1] == ends[r + 1][0] for r in range(world - 1))
        sizes = [b - a for a, b in ends]
        assert max(sizes) - min(sizes) <= 1
    assert shard.weak_range(1 << 20, 3) == (3 << 20, 4 << 20)


def test_world_reads_the_torchrun_environment(monkeypatch):
    monkeypatch.setenv("RANK", "5"); monkeypatch.setenv("LOCAL_RANK", "1"); monkeypatch.setenv("WORLD_SIZE", "8")
    assert shard.world() == (5, 1, 8)
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        monkeypatch.delenv(k)
    assert shard.world() == (0, 0, 1)


def test_stress_means_undo_the_fixed_point():
    sums = np.array([[3 << 18] * 12], dtype=np.int64)
    m = shard.stress_means(sums, 3)
    assert np.allclose(m[0, :3], 0.0) and np.allclose(m[0, 3:], 1.0)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _fixed_point_sums(N, k0, k1, steps, seed):
    """int64 [steps][12]: sum over chains k0..k1-1 of round(2^18 x per-chain stress), the
    quantity the step kernel accumulates (per chain here, per lane share there)."""
    import oracle
    out = np.zeros((steps, 12), dtype=np.int64)
    e = oracle.Ensemble(N, k1 - k0, seed=seed, chain_offset=k0)
    for n in range(steps):
        e.run(1)
        for k in range(k1 - k0):
            sig, sv = e.chain_stress(k)
            sig = sig.copy(); sig[:3] += 1.0          # N - 1 of the -N are folded into the sums (shard.stress_means)
            out[n] += np.rint(np.concatenate([sig, sv]) * (1 << 18)).astype(np.int64)
    return out


def _worker(rank, world, port, N, M, steps, seed, q):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, _, w = shard.world()
        k0, k1 = shard.strong_range(M, r, w)
        t = torch.from_numpy(_fixed_point_sums(N, k0, k1, steps, seed))
        shard.allreduce_sums(t)
        q.put((rank, t.numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_gloo_allreduce_reproduces_the_single_process_ensemble():
    import torch.multiprocessing as mp
    N, M, steps, seed, world = 8, 37, 5, 3, 2          # 37 chains: uneven shards (19 + 18)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N, M, steps, seed, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=240) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = _fixed_point_sums(N, 0, M, steps, seed)
    assert np.array_equal(got[0], want) and np.array_equal(got[1], want)
    # and the means the library reports from such sums are the oracle's ensemble means
    import oracle
    e = oracle.Ensemble(N, M, seed=seed)
    ref = e.run(steps, stress_every=1)
    assert np.allclose(shard.stress_means(want, M), ref, atol=12 * 2.0 ** -19)


def test_bench_refuses_a_world_size_other_than_gpus_and_builds_the_drivers_launch_line():
    """bench.py --gpus N reports only when N ranks run: one rank must not stand in for an N-GPU measurement
    (SURVEY 8e).  Without a launcher it starts the ranks itself with the driver's torchrun line."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT="29511")
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0
    assert "--gpus 2 but the launcher started 1 rank" in r.stderr
    assert not any(line.startswith("{") for line in r.stdout.splitlines())        # no JSON line from a wrong world
    sys.path.insert(0, root)
    import bench
    cmd = bench.spawn_command(4, 29512, ["--gpus", "4", "--steps", "3"])
    assert cmd[:10] == [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "4",
                        "--master-addr", "127.0.0.1", "--master-port", "29512"]
    assert cmd[10] == os.path.join(root, "bench.py") and cmd[11:] == ["--gpus", "4", "--steps", "3"]
