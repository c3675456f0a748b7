"""The N > 1 data path on CPU: two gloo ranks shard the atoms (inputs.shard_bounds), exchange the P
partial structure factors and sum them in rank order -- the host-side logic of bench.py --gpus N
and of the rbe_set_rho / rbe_set_exchange contract.  The per-rank arithmetic
here is the oracle's (there is no GPU in this test); what is checked is the sharding, the
collective and the order of the sum."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2407_09315_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = inputs.CONFIGS["water_3k"]
        atoms = inputs.make_atoms(cfg)
        m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)       # replicated: same seed
        lo, hi = inputs.shard_bounds(cfg.N, world, rank, align=32)
        oracle.set_threads(1)
        part = torch.from_numpy(oracle.rho(atoms[lo:hi], cfg.L, m))         # this rank's atoms only
        gathered = [torch.empty_like(part) for _ in range(world)]
        dist.all_gather(gathered, part)
        total = torch.zeros_like(part)
        for g in gathered:                                                   # rank order: bitwise reproducible
            total = total + g
        S = oracle.S(cfg.L, cfg.alpha)
        F = oracle.force(atoms[lo:hi], cfg.L, m, S, total.numpy())
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), lo=lo, hi=hi, rho=total.numpy(), F=F)
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_exchange_and_rank_ordered_sum(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = [np.load(tmp_path / f"rank{k}.npz") for k in range(world)]
    assert int(r[0]["lo"]) == 0 and int(r[0]["hi"]) == int(r[1]["lo"]) and int(r[1]["hi"]) == cfg.N
    assert int(r[0]["hi"]) % 32 == 0                                  # shards are whole 32-atom windows
    assert np.array_equal(r[0]["rho"], r[1]["rho"])                   # bitwise the same sum on every rank
    rho_full = oracle.rho(atoms, cfg.L, m)
    assert np.abs(r[0]["rho"] - rho_full).max() <= 1e-12 * np.abs(atoms[:, 3]).sum()
    F_full = oracle.force(atoms, cfg.L, m, oracle.S(cfg.L, cfg.alpha), rho_full)
    F = np.concatenate([r[0]["F"], r[1]["F"]])
    assert np.linalg.norm(F - F_full) <= 1e-12 * np.linalg.norm(F_full)
    assert np.abs(F.sum(0)).max() <= 1e-10 * np.abs(F).sum()          # momentum conservation across shards


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--ref-atoms", "2000"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "ns/atom/step"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
