"""Host-side partition of independent frozen-phonon configurations over ranks (images are
averaged over thermal-displacement configurations, each a full independent run).  No data-path collective:
rank r runs configurations r, r + N, ...; the only exchange is one all-reduce of the [probes][rings] sums."""
from __future__ import annotations


def phonons_for_rank(n_phonons: int, world: int, rank: int) -> list[int]:
    """Configurations of this rank.  With more ranks than configurations every rank still gets one
    (weak scaling: per-GPU work is fixed as N grows), numbered on from the workload's own."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world size")
    return [ph for ph in range(max(n_phonons, world)) if ph % world == rank]


def all_reduce_sum(acc, dist=None):
    """Sum of `acc` over ranks, in place (a collective, no arithmetic here): with every rank accumulating its
    configurations through ``prism_accumulate`` at weight 1 / (total configurations), the result is the mean."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(acc)
    return acc


def phonon_average(acc, count: int, dist=None):
    """Mean over all configurations of all ranks: acc holds this rank's sum of `count` outputs (a torch tensor,
    reduced in place).  dist: an initialised torch.distributed module, or None for a single process."""
    total = count
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        import torch
        n = torch.tensor([float(count)], dtype=torch.float64, device=acc.device)
        dist.all_reduce(acc)
        dist.all_reduce(n)
        total = int(round(float(n.item())))
    acc /= float(total)
    return acc
