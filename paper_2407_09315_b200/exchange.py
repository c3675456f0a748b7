"""Plumbing of the fused multi-GPU exchange (include/rbe.h: rbe_set_exchange): allocate one
exchange buffer per rank in torch symmetric memory (peer-mapped over NVLink), hand every rank's
mapping of every buffer to the library.  torch.distributed is used for the rendezvous only; the
exchange itself happens inside the structure-factor and force kernels."""
from __future__ import annotations


def setup_fused_exchange(ctx, group=None):
    """Configure `ctx` (an rbe.Rbe) for the fused exchange over `group` (default: WORLD).
    Returns the symmetric-memory tensor (kept alive by ctx as well).  Collective: every rank of
    the group must call it."""
    import torch
    import torch.distributed as dist
    import torch.distributed._symmetric_memory as symm_mem

    group = group if group is not None else dist.group.WORLD
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    nbytes = ctx.rbe_exchange_bytes(world)
    if nbytes == 0:
        raise ValueError(f"fused exchange supports up to 16 ranks, got {world}")
    buf = symm_mem.empty(nbytes, dtype=torch.uint8, device=torch.device("cuda", torch.cuda.current_device()))
    hdl = symm_mem.rendezvous(buf, group)
    buf.zero_()                      # flags start below every epoch
    torch.cuda.synchronize()
    dist.barrier(group)              # nobody pushes before every buffer is zeroed
    ptrs = [int(p) for p in hdl.buffer_ptrs]
    assert len(ptrs) == world and ptrs[rank] == buf.data_ptr()
    ctx.rbe_set_exchange(rank, world, ptrs, nbytes, keep_alive=(buf, hdl))
    return buf
