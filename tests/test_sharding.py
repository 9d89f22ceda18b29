"""The N > 1 path on CPU: wavelength blocks over a world-size-2 gloo group.
Each rank solves its block (with the oracle here — there is no GPU; on a GPU box bench.py does the
same with the CUDA library), J is all-gathered, Jbar all-reduced, and both equal the one-rank solve."""
import os
import socket

import numpy as np
import pytest

from paper_2408_14425_b200 import atmospheres as A
from paper_2408_14425_b200 import sharding


def test_wavelength_blocks_partition():
    for L in (1, 2, 5, 16, 64, 709):
        for world in (1, 2, 3, 4, 8):
            blocks = [sharding.wavelength_block(L, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == L
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1


def _atmosphere(line):
    if line:   # the moving line shards by x_lambda: every rank holds the six per-cell line parameters
        return A.line_config2(nx=64, ny=16, nlambda=5, ncascades=3)
    return A.make_config(4, nx=64, ny=16, nlambda=5, ncascades=3)


def _worker(rank, world, port, q, line):
    import torch
    import torch.distributed as dist
    from oracle import rc_oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    atm = _atmosphere(line)
    mine = sharding.shard_atmosphere(atm, rank, world)
    assert mine.nlambda == (3 if rank == 0 else 2) and (not line or (mine.line is atm.line and len(mine.xl) == mine.nlambda))
    out = rc_oracle.solve_atmosphere(mine, nthreads=2)
    J = sharding.allgather_j(torch.from_numpy(out["J"]), atm.nlambda)
    Jbar = sharding.allreduce_jbar(torch.from_numpy(out["Jbar"].copy()))
    if rank == 0:
        q.put((J.numpy(), Jbar.numpy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("line", [False, True])
def test_two_rank_gloo_matches_single_rank(oracle, line):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, line)) for r in range(2)]
    for p in procs:
        p.start()
    J, Jbar = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    atm = _atmosphere(line)
    ref = oracle.solve_atmosphere(atm)
    assert np.array_equal(J, ref["J"])
    assert np.allclose(Jbar, ref["Jbar"], rtol=1e-14, atol=0)


def test_bench_reference_arm_single_and_multi_rank():
    """bench.py --impl reference: rank 0 alone times the oracle and prints ONE JSON line with the contract's keys;
    under a multi-rank launch the other ranks exit 0 without work or output."""
    import json
    import os
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    cmd = [sys.executable, str(root / "bench.py"), "--impl", "reference", "--config", "0", "--steps", "2", "--warmup", "1"]
    env = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    out = subprocess.run(cmd + ["--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "seg-lambda/s" and d["value"] > 0 and d["n_gpus"] == 2
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    env["RANK"] = "1"
    out = subprocess.run(cmd + ["--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
