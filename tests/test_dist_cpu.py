"""N > 1 host logic on CPU (gloo, world_size 2): event sharding by the global Philox counter and the
rank-0-only reference arm of bench.py.  No collective sits on the data path; the only exchange an integrator on top needs
is a scalar all-reduce of (sum w, sum w^2), exercised here with the oracle's weights standing in for device results."""
import json
import os
import subprocess
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_events, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path[:] = [ROOT] + [d for d in sys.path if os.path.abspath(d or ".") not in (ROOT, os.path.join(ROOT, "oracle"))]
    import paper_0909_5257_b200 as hg
    from oracle import oracle as O
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, cnt = hg.shard_range(n_events, rank, world)
    if torch.cuda.is_available():
        # on a GPU box the shard goes through the product's host-buffer entry point (heget_run_host: sample + evaluate on the
        # device, copies inside), both ranks sharing device 0; without a device the oracle's sampler stands in for it
        P = hg.Process("g g > g g g", 1000.0)
        mom_t = torch.empty(5, 4, cnt, dtype=torch.float64).pin_memory()
        w_t = torch.empty(cnt, dtype=torch.float64).pin_memory()
        me2 = P.run_host(1, cnt, first_event=lo, mom_out=mom_t, weight=w_t)
        assert bool((me2 > 0).all())
        mom, w = mom_t.numpy(), w_t.numpy()
    else:
        mom, w, tries = O.sample_momenta(3, 1000.0, 1, cnt, first_event=lo)
    ranges = [None] * world
    dist.all_gather_object(ranges, (lo, cnt))
    acc = torch.tensor([w.sum(), (w * w).sum(), float(cnt)], dtype=torch.float64)
    dist.all_reduce(acc)
    q.put((rank, ranges, acc.tolist(), mom[:, :, :3].tolist()))
    dist.destroy_process_group()


def test_two_rank_sharding_reproduces_single_rank_events():
    n, world, port = 1001, 2, 29731
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    from oracle import oracle as O
    whole, w, _ = O.sample_momenta(3, 1000.0, 1, n)
    for rank, ranges, acc, head in res:
        assert ranges == [(0, 500), (500, 501)]
        assert acc[2] == n and abs(acc[0] - w.sum()) <= 1e-12 * w.sum()
        lo = ranges[rank][0]
        if torch.cuda.is_available():      # device RAMBO vs the oracle's: equal to rounding (bitwise between the ranks' own shards, see test_gpu_parity)
            assert np.allclose(np.array(head), whole[:, :, lo:lo + 3], rtol=0, atol=1e-9)
        else:
            assert np.array_equal(np.array(head), whole[:, :, lo:lo + 3])       # a shard is the same slice of the whole batch, bitwise


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--config", "C1"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--config", "C1"], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "events/s"
