"""Row sharding for N GPUs: parameter rows are independent units, so a batch is
split across ranks with no data-path collective; at most the caller all-gathers logL[B].

With n_lens > 1 the split falls on lens boundaries (a rank then needs only its lenses' psf /
data / noise blocks).  Pure host logic, no arithmetic of the method.
"""
from __future__ import annotations

from typing import List, Tuple


def shard_bounds(B: int, n_lens: int, rank: int, world: int) -> Tuple[int, int]:
    """Rows [r0, r1) of rank `rank`.  B must be a multiple of n_lens."""
    if B % n_lens or not (0 <= rank < world):
        raise ValueError("bad shard request")
    if n_lens > 1:
        per = B // n_lens
        l0, l1 = (n_lens * rank) // world, (n_lens * (rank + 1)) // world
        return l0 * per, l1 * per
    return (B * rank) // world, (B * (rank + 1)) // world


def lens_bounds(n_lens: int, rank: int, world: int) -> Tuple[int, int]:
    return (n_lens * rank) // world, (n_lens * (rank + 1)) // world


def all_bounds(B: int, n_lens: int, world: int) -> List[Tuple[int, int]]:
    return [shard_bounds(B, n_lens, r, world) for r in range(world)]


def shard_problem(prob, rows, rank: int, world: int):
    """(problem, rows) of rank `rank`: with several lenses the rank keeps only its lenses' psf /
    data / noise blocks and their rows; with one lens the context is replicated and the rows split.
    `prob` is a workloads.Problem, `rows` the float32 [B, P] batch of the whole job."""
    from dataclasses import replace
    w = prob.workload
    B = rows.shape[0]
    r0, r1 = shard_bounds(B, w.n_lens, rank, world)
    if w.n_lens > 1:
        l0, l1 = lens_bounds(w.n_lens, rank, world)
        if l1 == l0:
            return None, rows[0:0]
        sub = replace(w, n_lens=l1 - l0, batch=(l1 - l0) * (B // w.n_lens))
        return replace(prob, workload=sub, psf=prob.psf[l0:l1], data=prob.data[l0:l1], noise=prob.noise[l0:l1],
                       truth=prob.truth[l0:l1]), rows[r0:r1]
    return prob, rows[r0:r1]
