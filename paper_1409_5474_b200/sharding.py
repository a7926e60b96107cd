"""Multi-GPU decomposition of one force call: i-sharding with a replicated j-set.

The i-particles of a call are independent ("embarrassingly parallel"), so rank r of P
takes a contiguous slice of the active list and evaluates it against all N j-particles held in
its own context; the pair loop needs no exchange.  (The paper's own multi-GPU scheme distributes j
and sums partial forces; DESIGN.md section 9 says why i-sharding is taken here.)
What does cross ranks is outside the pair loop: assembling the per-rank results in i_list order
(`gather_forces`), which an integrator needs before it corrects and re-broadcasts the updated
particles.  Host logic only; torch.distributed is the transport (nccl on GPUs, gloo in the CPU
tests).
"""
import torch
import torch.distributed as dist


def shard_bounds(ni, rank, world):
    """[lo, hi) of rank's slice of an i_list of length ni: slices differ by at most one entry,
    cover 0..ni without overlap, and keep i_list order."""
    if world < 1 or not (0 <= rank < world) or ni < 0:
        raise ValueError("bad shard request")
    q, r = divmod(ni, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def shard_i_list(i_list, rank, world):
    lo, hi = shard_bounds(len(i_list), rank, world)
    return i_list[lo:hi]


def gather_forces(acc, jrk, pot, ni, group=None):
    """All ranks get acc, jrk (3, ni) and pot (ni,) in i_list order from the per-rank slices
    (3, n_local), (3, n_local), (n_local,).  One all_gather of padded [7][max_local] blocks."""
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    lo, hi = shard_bounds(ni, rank, world)
    assert pot.shape[0] == hi - lo
    width = -(-ni // world) if ni else 0
    block = torch.zeros((7, width), dtype=torch.float64, device=pot.device)
    block[0:3, :hi - lo] = acc
    block[3:6, :hi - lo] = jrk
    block[6, :hi - lo] = pot
    blocks = [torch.empty_like(block) for _ in range(world)]
    dist.all_gather(blocks, block, group=group)
    out = torch.empty((7, ni), dtype=torch.float64, device=pot.device)
    for r in range(world):
        a, b = shard_bounds(ni, r, world)
        out[:, a:b] = blocks[r][:, :b - a]
    return out[0:3], out[3:6], out[6]
