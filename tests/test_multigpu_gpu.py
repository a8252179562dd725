"""the path shards over independent rows (or lenses) with no data-path collective.
Here the CUDA path itself runs on two devices of one node -- sharding.shard_problem + one context per
device -- and must reproduce the single-device result bit for bit.  Skipped on one-GPU boxes (the
CPU suite covers the host-side sharding logic with two gloo ranks, tests/test_sharding.py)."""
import numpy as np
import pytest

from paper_2503_08586_b200 import sharding, workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n_lens,per", [(1, 600), (4, 32)])
def test_two_devices_reproduce_one_device(orc, n_lens, per):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    from paper_2503_08586_b200 import api
    w = (W.workload(1) if n_lens == 1 else W.workload(3)).scaled(batch=n_lens * per, n_lens=n_lens)
    prob = W.make_problem(w, orc.render_for_workloads)
    rows = W.batch_rows(w, per)
    torch.cuda.set_device(0)
    ctx = api.LensContext.from_problem(prob)
    want = ctx.loglike(torch.from_numpy(rows).cuda()).cpu()
    ctx.close()
    parts = []
    for rank in range(2):
        sub, my = sharding.shard_problem(prob, rows, rank, 2)
        torch.cuda.set_device(rank)
        c = api.LensContext.from_problem(sub)
        parts.append(c.loglike(torch.from_numpy(np.ascontiguousarray(my)).cuda()).cpu())
        c.close()
    torch.cuda.set_device(0)
    assert torch.equal(torch.cat(parts), want)
