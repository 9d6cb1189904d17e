"""Multi-GPU host logic on CPU (gloo, world_size 2): the spin-shard rule and the one collective of the path
(spins are independent; the only coupling is the sum over spins per ADC sample,
:194).  The per-rank signals are produced by the oracle here, because no GPU exists on this box; what is under
test is paper_2301_02702_b200.dist (shard bounds + reduce_signal), not the kernels."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2301_02702_b200 import workloads as W
from paper_2301_02702_b200.dist import env_world, reduce_signal, shard_bounds


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_bounds_cover_every_spin_once():
    for n in (0, 1, 7, 1024, 1000003):
        for world in (1, 2, 3, 8):
            lo_prev = 0
            sizes = []
            for r in range(world):
                lo, hi = shard_bounds(n, r, world)
                assert lo == lo_prev and hi >= lo
                sizes.append(hi - lo)
                lo_prev = hi
            assert lo_prev == n and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(10, 2, 2)


def test_env_world_defaults(monkeypatch):
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        monkeypatch.delenv(k, raising=False)
    assert env_world() == (0, 0, 1)
    monkeypatch.setenv("RANK", "3"); monkeypatch.setenv("LOCAL_RANK", "1"); monkeypatch.setenv("WORLD_SIZE", "4")
    assert env_world() == (3, 1, 4)


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        w = W.small("1")
        lo, hi = shard_bounds(w.phantom.n, rank, world)
        part = oracle.simulate(w.phantom.subset(slice(lo, hi)), w.seq, n_threads=1)
        sig = torch.from_numpy(part.astype(np.complex64))
        reduce_signal(sig)                      # the path's one collective
        np.save(os.path.join(out_dir, f"sig{rank}.npy"), sig.numpy())
        # the rank-ordered variant: same sum, and bitwise what adding the shards in rank order gives
        det = torch.from_numpy(part.astype(np.complex64))
        reduce_signal(det, deterministic=True)
        np.save(os.path.join(out_dir, f"det{rank}.npy"), det.numpy())
        np.save(os.path.join(out_dir, f"part{rank}.npy"), part.astype(np.complex64))
        # a second, real-valued tensor goes through the same call
        t = torch.full((4,), float(rank + 1))
        reduce_signal(t)
        assert torch.all(t == 3.0)
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_sum_to_the_full_signal(tmp_path, oracle_mod):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = W.small("1")
    full = oracle_mod.simulate(w.phantom, w.seq)
    a = np.load(tmp_path / "sig0.npy")
    b = np.load(tmp_path / "sig1.npy")
    assert np.array_equal(a, b), "all-reduce must leave the same signal on every rank"
    scale = np.abs(full).max()
    assert np.abs(a - full).max() / scale < 1e-6   # complex64 rounding of the two partial sums
    d0, d1 = np.load(tmp_path / "det0.npy"), np.load(tmp_path / "det1.npy")
    want = np.load(tmp_path / "part0.npy") + np.load(tmp_path / "part1.npy")   # rank order, complex64 adds
    assert np.array_equal(d0, d1) and np.array_equal(d0.view(np.float32), want.view(np.float32))


def test_reduce_signal_is_a_noop_without_a_process_group():
    t = torch.arange(6, dtype=torch.float32).view(3, 2).contiguous()
    c = torch.view_as_complex(t.clone())
    assert reduce_signal(c) is c and torch.equal(torch.view_as_real(c), t)
