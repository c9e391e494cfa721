"""N > 1 path on CPU (gloo, world_size 2): the DM-block sharding bench.py uses.

The path shards by trial DM with no data-path collective; what multi-rank code exists is the
rank -> DM-block map, the barrier and the max-over-ranks of the step time.  The blocks are also
pushed through the oracle to show that the union of the ranks' outputs is the single-process
result on the concatenated DM list (every DM row is independent).
"""
import os
import sys
import types

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import synth
    from oracle import fdd_oracle as O
    args = types.SimpleNamespace(workload="tiny", ndm=None)
    w = bench.make_workload(args, rank, world)
    dms = torch.tensor(w.dm_list, dtype=torch.float64)
    gathered = [torch.zeros_like(dms) for _ in range(world)]
    dist.all_gather(gathered, dms)
    # same bytes on every rank (same seed), own DM block per rank
    u8 = synth.make_filterbank(w)
    digest = torch.tensor([int(u8.astype(np.int64).sum())])
    digests = [torch.zeros_like(digest) for _ in range(world)]
    dist.all_gather(digests, digest)
    d = O.delay_table(w.nchans, w.f_lo, w.f_hi, w.tsamp, w.dm_list)
    y = O.fdd_fft(u8, d, mode="time")[:, :64].copy()
    t = torch.tensor([10.0 + rank], dtype=torch.float64)        # per-rank "device time"
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.barrier()
    q.put((rank, [g.numpy() for g in gathered], [int(x) for x in digests], y, float(t)))
    dist.destroy_process_group()


def test_dm_block_sharding_world2():
    world, port = 2, 29000 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sys.path.insert(0, ROOT)
    import synth
    from oracle import fdd_oracle as O
    base = synth.workload("tiny")
    step = base.dm_list[1] - base.dm_list[0]
    all_dms = np.concatenate(res[0][1])
    # contiguous, disjoint blocks of the same uniform grid: trial r*ndm + i
    assert all_dms.shape == (world * base.ndm,)
    assert np.allclose(all_dms, base.dm_list[0] + step * np.arange(world * base.ndm), rtol=0, atol=1e-12)
    for r in res:
        assert np.array_equal(np.concatenate(r[1]), all_dms)        # every rank sees the same map
        assert r[2][0] == r[2][1]                                  # identical input bytes
        assert r[4] == 10.0 + world - 1                             # max over ranks
    # union of the ranks' outputs == one process over the concatenated DM list
    u8 = synth.make_filterbank(base)
    d = O.delay_table(base.nchans, base.f_lo, base.f_hi, base.tsamp, all_dms)
    full = O.fdd_fft(u8, d, mode="time")[:, :64]
    got = np.concatenate([r[3] for r in res], axis=0)
    assert np.abs(got - full).max() <= 1e-9 * np.abs(full).max()


def test_bench_gpus_n_starts_n_ranks_or_fails_loudly():
    """`python bench.py --gpus 2` outside torchrun must start 2 ranks itself; on a box with fewer
    than 2 GPUs (this one has none) it must refuse, never run one rank and call it two."""
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    if torch.cuda.device_count() >= 2:
        return                                   # on a multi-GPU box the GPU suite covers the launch
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1",
                        "--warmup", "1"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "CUDA device(s) are visible" in (r.stderr + r.stdout)
    assert '"n_gpus"' not in r.stdout
