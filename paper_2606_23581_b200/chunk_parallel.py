"""Chunk-parallel decode across GPUs: plumbing only.

A request's chunks are spread over the ranks of a process group (one process per GPU).  Every rank reads ITS chunks once
(kam_paged_decode_state), the per-rank softmax states (o, lse) are exchanged with ONE all-gather over NVLink/NVSwitch
(NCCL through torch.distributed; <= 2.1 MB per rank at BASELINE.json config 5) and every rank applies the same merge
(kam_lse_merge_states) in the same order, so all ranks end with identical bits.  Nothing here computes: sharding is
integer bookkeeping, the exchange is torch.distributed, the arithmetic is in the two C entry points.
"""
import torch
import torch.distributed as dist


def shard_chunks(n_chunks, rank, world):
    """Chunk indices rank `rank` owns: contiguous blocks, the first n_chunks % world ranks take one more."""
    base, extra = divmod(int(n_chunks), int(world))
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def all_gather_states(o_state, lse_state, group=None):
    """One all-gather of [o | lse] rows.  o_state [B, Hq, Dv] f32, lse_state [B, Hq] f32 (device tensors on NCCL, CPU
    tensors on gloo).  Returns (o_all [world, B, Hq, Dv], lse_all [world, B, Hq]) in rank order."""
    world = dist.get_world_size(group)
    B, Hq, Dv = o_state.shape
    packed = torch.cat([o_state.reshape(B * Hq, Dv), lse_state.reshape(B * Hq, 1)], dim=1).contiguous()
    gathered = torch.empty((world * packed.shape[0], packed.shape[1]), dtype=packed.dtype, device=packed.device)
    dist.all_gather_into_tensor(gathered, packed, group=group)          # rank-major concatenation along dim 0
    gathered = gathered.reshape(world, B * Hq, Dv + 1)
    o_all = gathered[:, :, :Dv].reshape(world, B, Hq, Dv).contiguous()
    lse_all = gathered[:, :, Dv].reshape(world, B, Hq).contiguous()
    return o_all, lse_all


def decode_chunk_parallel(ctx, q, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale, out, lse,
                          patches=None, group=None):
    """This rank's (block_tables, chunk_starts, chunk_offsets, n_chunks) describe only the chunks it holds (n_chunks[b] may
    be 0).  out [B, Hq, Dv] bf16 and lse [B, Hq] f32 receive the readout over ALL ranks' chunks."""
    B, Hq = lse.shape
    o_state = torch.empty((B, Hq, out.shape[2]), dtype=torch.float32, device=q.device)
    l_state = torch.empty((B, Hq), dtype=torch.float32, device=q.device)
    ctx.kam_paged_decode_state(q, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale, o_state, l_state,
                               patches=patches)
    o_all, l_all = all_gather_states(o_state, l_state, group)
    world = o_all.shape[0]
    ctx.kam_lse_merge_states([o_all[r] for r in range(world)], [l_all[r] for r in range(world)], B, out, lse)
    return out, lse
