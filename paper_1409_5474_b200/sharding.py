"""Multi-GPU decompositions of one force call.

(1) i-sharding with a replicated j-set (bench.py's N > 1 path):

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


# ---- (2) j-sharding: the paper's own multi-GPU scheme ---------------------------
#
# "Multi-GPU parallelization is achieved by distributing the j particles over the various GPUs ...
# This reduces the memory usage, transfer time and the time required to execute the optional
# prediction step on the j particles.  In this scheme the first kernel computes the partial forces
# ... and the second kernel sums these."  Rank r stores and predicts only particles
# [lo_r, hi_r) (contiguous blocks: the sum is order-free, so this equals the paper's round-robin).
# One force call on a global active list:
#   1. every rank takes the predicted state of the active particles it OWNS, with their flag;
#   2. one all_gather gives every rank the state of all active particles (6 fp64 + flag + global
#      index each);
#   3. every rank evaluates them BY VALUE against its own j-slice, telling the kernel which member of
#      the slice each active particle is (nb_force_ext_ids: self_idx = global index - lo for the
#      particles it owns, -1 for the others): the owner excludes the self pair by index (R5) and
#      every rank treats the pairs between a flagged active particle and the flagged members of
#      its slice as unsoftened (R7) -- exactly what nb_force does on one GPU;
#   4. one all_reduce(sum) of [7][ni] fp64 -- the paper's "second kernel", across GPUs.
# Nothing is added or taken back on the host: the sum of the ranks' partial forces IS the force.


def owned(i_list, lo, hi):
    """Positions k (ascending) of the global active list whose particle lies in [lo, hi)."""
    il = torch.as_tensor(i_list)
    return torch.nonzero((il >= lo) & (il < hi)).flatten()


def gather_active_state(state_local, pos_local, ni, group=None):
    """state_local: (R, n_owned) fp64 rows of the owned active particles (predicted x, y, z, vx, vy,
    vz, then whatever else travels: flag, global index), pos_local: their positions in the global
    active list.  Returns (R, ni) on every rank, in active-list order.  One all_gather of the
    counts + one of padded blocks."""
    world = dist.get_world_size(group)
    dev = state_local.device
    rows = state_local.shape[0]
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, torch.tensor([state_local.shape[1]], dtype=torch.int64, device=dev), group=group)
    width = max(int(c.item()) for c in counts)
    block = torch.zeros((rows + 1, max(width, 1)), dtype=torch.float64, device=dev)
    k = state_local.shape[1]
    block[:rows, :k] = state_local
    block[rows, :k] = pos_local.to(torch.float64)        # positions < 2^53: exact in fp64
    blocks = [torch.empty_like(block) for _ in range(world)]
    dist.all_gather(blocks, block, group=group)
    out = torch.empty((rows, ni), dtype=torch.float64, device=dev)
    for r in range(world):
        kr = int(counts[r].item())
        if kr:
            out[:, blocks[r][rows, :kr].to(torch.int64)] = blocks[r][:rows, :kr]
    return out


def force_j_sharded(force_by_value_ids, state_local, pos_local, ni, lo, hi, group=None):
    """Steps 2-4 above.  state_local: (8, n_owned) = predicted x, y, z, vx, vy, vz, flag (0/1) and
    GLOBAL index of the owned active particles.  force_by_value_ids(x (3, ni), v (3, ni), self_idx
    int32 (ni,), iflags uint8 (ni,)) -> (acc (3, ni), jrk (3, ni), pot (ni,)) against the CALLING
    rank's j-slice [lo, hi) (Context.force_ext_ids on a GPU).  Returns the complete acc, jrk, pot of
    the active list on every rank."""
    st = gather_active_state(state_local, pos_local, ni, group)
    gidx = st[7].to(torch.int64)
    mine = (gidx >= lo) & (gidx < hi)
    self_idx = torch.where(mine, gidx - lo, torch.full_like(gidx, -1)).to(torch.int32)
    iflags = st[6].to(torch.uint8)
    acc, jrk, pot = force_by_value_ids(st[0:3].contiguous(), st[3:6].contiguous(), self_idx, iflags)
    part = torch.cat([acc, jrk, pot.reshape(1, -1)], dim=0).contiguous()
    dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)
    return part[0:3], part[3:6], part[6]


# ---- (3) j-sharding with the exchange done by the kernels (nb.h: nb_xchg_*, nb_xforce) -----------
#
# Step 4 above -- the paper's "second kernel", across GPUs -- without a collective call: every rank
# owns a window in device memory, the pair kernel's reducing CTA stores the rank's partial forces into
# every rank's window over NVLink peer memory, raises a flag, waits for the peers' flags and adds the
# slots in rank order (csrc/xchg.h).  What is host logic is the one-time wiring: exchanging the
# windows' IPC handles.


def xchg_connect(ctx, ni_cap, group=None):
    """Create this rank's window (ctx.xchg_create), exchange the IPC handles with all ranks of the
    group (one all_gather_object), attach every peer's window, barrier.  ctx: a Context (or anything
    with xchg_create / xchg_export / xchg_attach).  Returns (rank, world)."""
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    ctx.xchg_create(rank, world, ni_cap)
    handle, _ = ctx.xchg_export()
    handles = [None] * world
    dist.all_gather_object(handles, handle, group=group)
    for r in range(world):
        if r != rank:
            ctx.xchg_attach(r, handle=handles[r])
    dist.barrier(group=group)                 # nobody pushes before everybody has attached
    return rank, world


def force_j_sharded_xchg(ctx, state_local, pos_local, ni, lo, hi, eps2, group=None):
    """force_j_sharded with step 4 inside the kernels: gathers the active particles' state (step 2,
    still one all_gather -- an integrator that keeps the active state replicated, as the paper's host
    does, needs none), then ONE ctx.xforce call returns the complete forces on every rank."""
    st = gather_active_state(state_local, pos_local, ni, group)
    gidx = st[7].to(torch.int64)
    mine = (gidx >= lo) & (gidx < hi)
    self_idx = torch.where(mine, gidx - lo, torch.full_like(gidx, -1)).to(torch.int32)
    iflags = st[6].to(torch.uint8)
    return ctx.xforce(st[0:3].contiguous(), st[3:6].contiguous(), self_idx, iflags, eps2)


# ---- (4) one block step of the j-sharded integrator (host logic around the C-ABI calls) -----------
#
# PAPER.md:41/:49 (block time steps: "only the particles are updated that require a force update at a
# certain time") on the j-sharded layout of PAPER.md:55: every rank schedules, predicts and corrects
# ITS slice; what crosses ranks per block step is one double (the block time), the state of the due
# particles (72 B each) and their partial forces (56 B each).


def step_j_sharded(ctx, lo, hi, flags_local, eps2, eta, dt_min, dt_max, group=None, exchange="xchg"):
    """One block step.  ctx: this rank's Context holding particles [lo, hi) with steps initialised
    (init_steps / set_dt); flags_local: device uint8 tensor (hi - lo,) of their flag bits.
    exchange: "xchg" = nb_xforce (partial forces exchanged and summed by the kernels over peer memory:
    xchg_connect first), "xchg_split" = the same with the two halves of the call separated by a host
    barrier (for ranks that share one GPU: no kernel then waits for another process's kernel), "nccl" =
    nb_force_ext_ids + all_reduce.  Returns (t, ni): the block time and the number of particles
    advanced over all ranks.  Every rank must call it."""
    dev = flags_local.device
    # 1. my slice's earliest time and who is due then (R21); the block time is the minimum over ranks
    t_loc, ni_loc, il_loc = ctx.next_block()
    tt = torch.tensor([t_loc if ni_loc > 0 else float("inf")], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MIN, group=group)
    t = float(tt.item())
    due = il_loc.to(torch.int64) if (ni_loc > 0 and t_loc == t) else torch.empty(0, dtype=torch.int64, device=dev)
    # 2. my slice predicted to t (R1, R8); the predicted state of my due particles travels to all ranks,
    #    in rank order = ascending global index (R21)
    ctx.predict(t)
    px, pv = ctx.predicted()
    k = due.shape[0]
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(dist.get_world_size(group))]
    dist.all_gather(counts, torch.tensor([k], dtype=torch.int64, device=dev), group=group)
    counts = [int(c.item()) for c in counts]
    ni, first = sum(counts), sum(counts[:dist.get_rank(group)])
    pos = first + torch.arange(k, dtype=torch.int64, device=dev)
    state = torch.cat([px[:, due], pv[:, due], flags_local[due].to(torch.float64)[None],
                       (due + lo).to(torch.float64)[None]], 0)
    st = gather_active_state(state, pos, ni, group)
    gidx = st[7].to(torch.int64)
    mine = (gidx >= lo) & (gidx < hi)
    self_idx = torch.where(mine, gidx - lo, torch.full_like(gidx, -1)).to(torch.int32)
    iflags = st[6].to(torch.uint8)
    x, v = st[0:3].contiguous(), st[3:6].contiguous()
    # 3. forces of ALL ranks' particles on the due ones
    if exchange == "xchg":
        acc, jrk, _ = ctx.xforce(x, v, self_idx, iflags, eps2)
    elif exchange == "xchg_split":
        part = ctx.xforce(x, v, self_idx, iflags, eps2, phase=1)
        ctx.sync()
        dist.barrier(group=group)
        acc, jrk, _ = ctx.xforce(None, None, None, None, eps2, phase=2, out=part)
    else:
        acc, jrk, pot = ctx.force_ext_ids(x, v, self_idx, iflags, eps2)
        part = torch.cat([acc, jrk, pot.reshape(1, -1)], 0).contiguous()
        dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)
        acc, jrk = part[0:3], part[3:6]
    # 4. corrector, new steps (R12, R18..R20): the owners, on their own particles
    if k:
        ctx.correct(due.to(torch.int32), t, acc[:, pos].contiguous(), jrk[:, pos].contiguous(), eta, dt_min, dt_max)
    return t, ni
