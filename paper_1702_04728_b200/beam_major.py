"""Beam-major exchange: coarse channels are sharded over W ranks for the beamformer
(PAPER.md:47, :53 -- one channel per GPU in the paper; no collective there), the consumer of the beams
(dedispersion, the FRB search) wants ALL channels of a subset of beams: an all-to-all corner turn
channel-sharded -> beam-sharded.

Layouts (C order, uint8):  local beams      [C_local][R][1024][16]        (chime_bf_execute)
                           receive buffer   [C_total][R][1024 / W][16]    on the rank that owns the beams

Two ways to get there:
  * fused (the product): chime_bf_execute_beam_major -- the kernel's epilogue stores every beam's 16 bytes into the
    owner's receive buffer through peer-mapped pointers (NVLink); `peer_buffer_ptrs` obtains them from
    torch.distributed's symmetric memory.  No NCCL call on the data path.
  * `exchange_all_to_all` (baseline / check): re-layout with torch ops + one torch.distributed.all_to_all_single.
    Runs on any backend (gloo on CPU in the tests); it is what the fused path is compared against.
Host logic only; no beamformer arithmetic.
"""
N_BEAM, N_FINE = 1024, 16


def beam_shard(world, rank):
    """(first beam, count) owned by `rank`: contiguous blocks of 1024 / world beams (world must divide 1024)."""
    if world < 1 or N_BEAM % world or not (0 <= rank < world):
        raise ValueError("world must divide 1024 and 0 <= rank < world")
    per = N_BEAM // world
    return rank * per, per


def receive_shape(n_coarse_total, n_frames, world):
    return (n_coarse_total, n_frames, N_BEAM // world, N_FINE)


def exchange_all_to_all(local_beams, group=None):
    """local_beams: [C_local][R][1024][16] uint8 (this rank's channels; every rank the same C_local).
    Returns this rank's receive buffer [world * C_local][R][1024 / world][16]; channel order = rank-major."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    C, R, B, F = local_beams.shape
    assert B == N_BEAM and F == N_FINE and N_BEAM % world == 0
    per = N_BEAM // world
    # [C][R][W][per][16] -> [W][C][R][per][16]: block d is what rank d receives from this rank
    send = local_beams.view(C, R, world, per, F).permute(2, 0, 1, 3, 4).contiguous()
    if world == 1:
        return send.view(C, R, per, F)
    recv = torch.empty_like(send)
    dist.all_to_all_single(recv.view(-1), send.view(-1), group=group)
    return recv.view(world * C, R, per, F)          # block s = the C channels of source rank s


def peer_buffer_ptrs(recv_buffer, group=None):
    """Device pointers of every rank's receive buffer as seen from this rank (peer-mapped over NVLink), for
    chime_bf_execute_beam_major.  Single rank: the local pointer.  Multi-rank: torch symmetric memory
    (`recv_buffer` must have been allocated with torch.distributed._symmetric_memory.empty)."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return [recv_buffer.data_ptr()]
    import torch.distributed._symmetric_memory as symm_mem
    hdl = symm_mem.rendezvous(recv_buffer, group=group if group is not None else dist.group.WORLD)
    return [int(p) for p in hdl.buffer_ptrs]
