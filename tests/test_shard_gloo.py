"""world_size-2 gloo tests (CPU) of the multi-GPU host logic: pairs shard over ranks with no
data-path collective; timing is the max over ranks."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")

from paper_2501_10653_b200 import shard  # noqa: E402


def test_pair_range_partitions_the_job():
    for total in (0, 1, 2, 7, 16, 33):
        for world in (1, 2, 3, 8):
            got = [i for r in range(world) for i in shard.pair_range(total, r, world)]
            assert got == list(range(total))
            sizes = [len(shard.pair_range(total, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.pair_range(4, 2, 2)


def test_weak_seeds_are_disjoint():
    seen = set()
    for r in range(8):
        s = shard.weak_seeds(32, r, 8, seed0=100)
        assert len(s) == 32 and not seen.intersection(s)
        seen.update(s)
    assert seen == set(range(100, 100 + 256))


def test_single_process_is_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    j = shard.job_throughput(32, 0.16)
    assert j["world"] == 1 and j["units"] == 32 and abs(j["us_per_unit"] - 5.0) < 1e-12


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dist.barrier()
        local_ms = 1.0 + rank                                  # rank 1 is the slow one
        j = shard.job_throughput(16, local_ms, dist)
        mine = list(shard.pair_range(5, rank, world))
        whole = torch.tensor([[float(i), float(10 * i)] for i in shard.weak_seeds(2, rank, world)])
        allw = shard.gather_whole(whole, dist)
        dist.barrier()
        q.put((rank, j, mine, allw.tolist()))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, j0, m0, w0), (r1, j1, m1, w1) = res
    assert (r0, r1) == (0, 1)
    assert j0 == j1                                            # every rank sees the same job numbers
    assert j0["world"] == 2 and j0["ms"] == 2.0 and j0["units"] == 32     # max over ranks, all ranks' units
    assert abs(j0["us_per_unit"] - 62.5) < 1e-9
    assert m0 == [0, 1, 2] and m1 == [3, 4]                    # disjoint, ordered, complete
    assert w0 == w1 == [[0.0, 0.0], [1.0, 10.0], [2.0, 20.0], [3.0, 30.0]]


# ----------------------------------------------------------------------------- one pair over several ranks
def test_band_rows_partition_the_image():
    for H, N_T in ((2048, 64), (100, 16), (65, 64), (7, 8), (1000, 128)):
        for world in (1, 2, 3, 8):
            bands = [shard.band_rows(H, N_T, r, world) for r in range(world)]
            assert bands[0][0] == 0 and bands[-1][1] == H
            for (a0, a1), (b0, b1) in zip(bands, bands[1:]):
                assert a1 == b0 and a0 <= a1
            for r0, r1 in bands:
                if r1 > r0:                                    # more ranks than tile rows: trailing bands are empty
                    assert r0 % N_T == 0 and (r1 % N_T == 0 or r1 == H)
            rows = [(r1 - r0 + N_T - 1) // N_T for r0, r1 in bands]
            assert max(rows) - min(rows) <= 1
    with pytest.raises(ValueError):
        shard.band_rows(64, 8, 2, 2)


def _band_worker(rank, world, port, q):
    """Each rank reduces ITS band of tile rows (per-tile values from the oracle: this test is about the
    host logic, not the kernels) to the four sums of Eqs. 3-4; one all-reduce; every rank finishes."""
    import numpy as np
    import torch.distributed as dist
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(0)                         # the same image on every rank
        x = rng.random((100, 72)).astype(np.float32)
        y = rng.random((100, 72)).astype(np.float32)
        N_T, C2, C = 16, 1e-6, 1e-6
        r0, r1 = shard.band_rows(100, N_T, rank, world)
        t = oracle.tiles_2d(x[r0:r1], y[r0:r1], N_T, 1e-6, C2, C, 5e-7)
        c2, c = float(np.float32(C2)), float(np.float32(C))
        sums4 = torch.tensor([np.sum(t["lisi"] * (np.maximum(t["X"], t["Y"]) + c2)),
                              np.sum(t["auglisi"] * (t["X"] + t["Y"] + c)), np.sum(t["X"]), np.sum(t["Y"])],
                             dtype=torch.float64)
        total = shard.allreduce_sums(sums4, dist)
        q.put((rank, (r0, r1), t["lisi"].shape, total.tolist()))
    finally:
        dist.destroy_process_group()


def test_two_ranks_share_one_pair_by_bands():
    import numpy as np
    import torch.multiprocessing as mp
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_band_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (_, b0, s0, t0), (_, b1, s1, t1) = res
    assert b0 == (0, 64) and b1 == (64, 100)                  # 7 tile rows: 4 + 3 (the last one ragged)
    assert s0 == (4, 5) and s1 == (3, 5)
    assert t0 == t1                                            # every rank holds the same all-reduced sums
    rng = np.random.default_rng(0)
    x = rng.random((100, 72)).astype(np.float32)
    y = rng.random((100, 72)).astype(np.float32)
    full = oracle.tiles_2d(x, y, 16, 1e-6, 1e-6, 1e-6, 5e-7)
    exp = oracle.aggregate(full["lisi"], full["auglisi"], full["X"], full["Y"], 1e-6, 1e-6)
    c2 = c = float(np.float32(1e-6))
    n = full["lisi"].size
    lisi = t0[0] / (max(t0[2], t0[3]) + c2)                    # Eq. 3 from the summed partials
    aug = (t0[1] - (n - 1) * c) / (t0[2] + t0[3] + c)          # Eq. 4
    assert abs(lisi - exp[0]) <= 1e-12 * abs(exp[0]) and abs(aug - exp[1]) <= 1e-12 * abs(exp[1])


def test_bench_gpus_n_starts_its_own_ranks():
    """`python bench.py --gpus 2` without WORLD_SIZE re-executes itself under torch.distributed.run with two ranks
    (the form the driver's 1-GPU command has).  --rank-map stops before CUDA: every rank joins a gloo group and reports
    its band of ONE config-[4] pair (--shard bands) and its seeds (replicas); the bands are shard.band_rows' partition."""
    import json
    import subprocess
    from paper_2501_10653_b200 import shard, synth
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items()
           if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--rank-map", "--workload", "cfg4",
                        "--shard", "bands"], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    cfg = synth.CONFIGS[4]
    assert d["n_gpus"] == 2 and [x["rank"] for x in d["ranks"]] == [0, 1]
    assert [tuple(x["band_rows"]) for x in d["ranks"]] == [shard.band_rows(cfg.N, cfg.N_T, k, 2) for k in range(2)]
    assert d["ranks"][0]["band_rows"][0] == 0 and d["ranks"][1]["band_rows"][1] == cfg.N
    assert d["ranks"][0]["band_rows"][1] == d["ranks"][1]["band_rows"][0]
    assert d["ranks"][0]["seeds"][1] < d["ranks"][1]["seeds"][0]           # replicas: no rank repeats another's pairs
