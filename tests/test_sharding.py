"""N > 1 path on CPU: two gloo ranks shard a batch on row / lens boundaries, evaluate their rows
(with the oracle standing in for the device kernels: the sharding logic is what is under test)
and all-gather logL; the result must equal the single-process evaluation."""
import os
import socket

import numpy as np
import pytest

from paper_2503_08586_b200 import sharding, workloads as W


def test_bounds_cover_everything_once():
    for B, L, world in ((4096, 1, 2), (4097, 1, 4), (512 * 10, 10, 4), (7 * 3, 7, 8), (5, 1, 8)):
        b = sharding.all_bounds(B, L, world)
        assert b[0][0] == 0 and b[-1][1] == B
        for (a0, a1), (c0, c1) in zip(b[:-1], b[1:]):
            assert a1 == c0 and a0 <= a1
        if L > 1:
            per = B // L
            assert all(x % per == 0 for pair in b for x in pair)
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 3, 0, 2)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, n_lens, rows_per_lens, out_path):
    import torch
    import torch.distributed as dist
    from oracle import oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.workload(3).scaled(batch=n_lens * rows_per_lens, n_lens=n_lens)
    w = W.Workload(**{**w.__dict__, "ny": 16, "nx": 16, "psf_size": 5})
    prob = W.make_problem(w, O.render_for_workloads)
    rows = W.batch_rows(w, rows_per_lens)
    sub, my_rows = sharding.shard_problem(prob, rows, rank, world)
    ll = np.zeros(0)
    if sub is not None and len(my_rows):
        ll, _ = O.loglike_batch(O.config_of(sub.workload), sub.psf, sub.data, sub.noise,
                                my_rows, n_lens=sub.workload.n_lens, threads=1)
    mine = torch.from_numpy(np.asarray(ll, np.float64))
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([mine.numel()], dtype=torch.int64))
    mx = int(max(s.item() for s in sizes))
    pad = torch.zeros(mx, dtype=torch.float64); pad[:mine.numel()] = mine
    parts = [torch.zeros(mx, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(parts, pad)
    if rank == 0:
        full = np.concatenate([p[:int(s.item())].numpy() for p, s in zip(parts, sizes)])
        np.save(out_path, full)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_matches_single_process(tmp_path, orc):
    import torch.multiprocessing as mp
    n_lens, per = 3, 4
    out = str(tmp_path / "ll.npy")
    mp.spawn(_worker, args=(2, _free_port(), n_lens, per, out), nprocs=2, join=True)
    got = np.load(out)
    w = W.workload(3).scaled(batch=n_lens * per, n_lens=n_lens)
    w = W.Workload(**{**w.__dict__, "ny": 16, "nx": 16, "psf_size": 5})
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, per)
    want, _ = orc.loglike_batch(orc.config_of(w), prob.psf, prob.data, prob.noise, rows, n_lens=n_lens)
    assert got.shape == want.shape and np.array_equal(got, want)
