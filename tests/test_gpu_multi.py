"""The N > 1 path on GPUs: two ranks, one GPU each, NCCL.  Each rank solves its wavelength block of ONE
atmosphere with the CUDA library, J is all-gathered and Jbar all-reduced through torch.distributed, and both equal the
single-rank solve of the whole atmosphere bit for bit (wavelengths are independent formal solutions, PAPER.md:384, 573;
a block boundary at a multiple of 8 keeps every wavelength in the same lane batch).  Skipped, not failed, where fewer
than two GPUs are visible (the round's GPU box has one); bench.py --gpus N runs the same sharding."""
import os
import socket

import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A

pytestmark = pytest.mark.gpu


def _atmosphere(mode):
    if mode == "line":
        return A.line_config2(nx=256, ny=128, nlambda=32, ncascades=6)
    return A.make_config(4 if mode == "Jbar" else 2, nx=256, ny=128, nlambda=32, ncascades=6)


def _worker(rank, world, port, q, mode):
    import torch
    import torch.distributed as dist
    from paper_2408_14425_b200 import binding, sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device(f"cuda:{rank}"))
    accumulate = mode == "Jbar"
    atm = _atmosphere(mode)
    mine = sharding.shard_atmosphere(atm, rank, world)
    J, rc = binding.solve_atmosphere(mine, device=rank)
    if accumulate:
        out = sharding.allreduce_jbar(J)
    else:
        out = sharding.allgather_j(J, atm.nlambda)
    torch.cuda.synchronize(rank)
    if rank == 0:
        q.put(out.cpu().numpy())
    rc.close()
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("mode", ["J", "Jbar", "line"])
def test_two_ranks_nccl_match_one_rank(mode):
    accumulate = mode == "Jbar"
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    import torch.multiprocessing as mp
    from paper_2408_14425_b200 import binding
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, mode)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=600)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    atm = _atmosphere(mode)
    J, rc = binding.solve_atmosphere(atm)
    ref = J.cpu().numpy()
    rc.close()
    if accumulate:
        # two partial sums added by NCCL instead of one sum over all batches: same terms, another order
        assert np.allclose(got, ref, rtol=2e-6, atol=0)
    else:
        assert np.array_equal(got, ref)


def test_bench_shards_one_atmosphere_on_one_rank():
    """bench.py under a launcher environment of world size 1 (what the driver does at N = 1) prints one line whose
    unit count is the whole job's and whose keys the contract names; the sharding code path itself needs N > 1."""
    import json
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    out = subprocess.run([sys.executable, str(root / "bench.py"), "--config", "1", "--steps", "2", "--warmup", "3", "--no-cpu-baseline"],
                         capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["n_gpus"] == 1 and d["unit"] == "seg-lambda/s" and d["value"] > 0 and d["gpu_launches"] > 0
    assert d["roofline"]["bound"] in ("l2", "alu") and 0 < d["roofline"]["frac"] < 1.5
    assert d["config"]["early_exit"] is True and 0 < d["config"]["walked_fraction"] <= 1.0
    assert d["e2e"]["matches_device_path"] is True and d["e2e"]["steps"] == 2
    assert d["e2e"]["h2d_bytes_per_step"] == 2 * 512 * 512 * 16 * 4
