"""World-size-2 gloo test (CPU) of the N>1 path: ranks own blocks of GLOBAL chain ids, the only exchange
is the ensemble accumulator; the result must equal the single-rank run over all chains.  The per-rank
compute is the CPU oracle here (the GPU kernels use the same chain_id0 convention; see
tests/test_gpu_parity.py::test_noise_matches_oracle and test_init_random_walk_matches_oracle)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle as O
from paper_2208_06559_b200 import ensemble


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, C, N, steps, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        chain0 = ensemble.shard(rank, world, C)
        p = O.Params(n_rods=N, dt=1e-4, seed=3)
        r = O.init_random_walk(N, 1.0, 1002, range(chain0, chain0 + C))
        r, info = O.step_ensemble(p, r, 0, steps, chain0=chain0)
        _, ens = O.observables(p, r)
        ens_t = ensemble.reduce_ensemble(torch.from_numpy(ens.copy()))
        ms = ensemble.max_over_ranks(10.0 + rank)
        if rank == 0:
            np.save(out, np.concatenate([ens_t.numpy().reshape(-1), [ms]]))
    finally:
        dist.destroy_process_group()


def test_two_rank_ensemble_equals_single_rank(tmp_path):
    C, N, steps, world = 6, 12, 3, 2
    out = str(tmp_path / "ens.npy")
    mp.spawn(_worker, args=(world, _free_port(), C, N, steps, out), nprocs=world, join=True)
    got = np.load(out)
    p = O.Params(n_rods=N, dt=1e-4, seed=3)
    r = O.init_random_walk(N, 1.0, 1002, range(world * C))
    r, info = O.step_ensemble(p, r, 0, steps, chain0=0)
    _, ens = O.observables(p, r)
    assert np.allclose(got[:-1].reshape(2, -1), ens, rtol=1e-13, atol=1e-12)
    assert got[-1] == 11.0                                   # max over ranks of the per-rank time
    mean, se = ensemble.mean_and_se(torch.from_numpy(ens), world * C)
    assert abs(float(mean[0]) - N) < 6 * float(se[0]) + 0.5 * N


def test_shard_bounds():
    import pytest
    assert ensemble.shard(0, 4, 256) == 0 and ensemble.shard(3, 4, 256) == 768
    with pytest.raises(ValueError):
        ensemble.shard(4, 4, 1)


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` outside torchrun must start two ranks itself.  Run on the CPU
    through the reference arm (the oracle; the GPU arm needs CUDA): bench.py re-executes under torch.distributed.run,
    rank 0 alone prints ONE JSON line, and it refuses to print n_gpus != --gpus, so n_gpus = 2 proves WORLD_SIZE = 2."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "c1",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["config"]["workload"] == "c1"
    # inside a torchrun environment whose WORLD_SIZE disagrees with --gpus it refuses
    env2 = dict(env, WORLD_SIZE="1", RANK="0")
    bad = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "c1"],
                         capture_output=True, text=True, env=env2, timeout=600)
    assert bad.returncode != 0 and "refusing" in (bad.stderr + bad.stdout)
