"""Multi-GPU range search over a replicated hierarchy: one batch of queries sharded across ranks (SURVEY.md 8(e)(i),
NEXT-4).

Algorithm 1 keeps no state across queries, so a batch splits into contiguous blocks, one per rank
(one process per GPU, ``torch.distributed``); every rank holds the whole hierarchy -- built locally from the same
primitives (the build is deterministic: the hierarchy is unique, P8) or received once with :func:`replicate_nodes` --
and runs the ordinary query path on its block.  There is NO collective inside the traversal.  What the ranks exchange is
one all-gather of their result sizes: the rows of rank r come after the rows of ranks < r, so its block of the global
CSR is its local CSR shifted by the number of results of the ranks before it, and the global arrays are the
concatenation of the blocks.

This module holds only that plumbing (block bounds, the all-gather, the offset shift, an optional gather to every
rank); it is device-agnostic, which is how the N > 1 path is tested on CPU with ``gloo``.  The tensors handed to a
collective live where the group's backend can reach them: on the GPU under ``nccl``, on the host otherwise (``gloo``
has no all-gather of CUDA tensors), so CUDA results can also be assembled by ranks that talk over ``gloo`` -- two
processes sharing one GPU in the tests.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def _comm_device(t: torch.Tensor, group=None) -> torch.device:
    """Where a tensor must live to go through a collective of ``group``: its own device under nccl, else the host."""
    if dist.is_initialized() and "nccl" in str(dist.get_backend(group)):
        return t.device
    return torch.device("cpu")


def block_bounds(q: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous block of rank ``rank``: the first q % world ranks get one query more."""
    base, extra = divmod(int(q), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


class ShardedCsr:
    """This rank's block of the global CSR.

    ``offsets``: int64[q_local + 1], already GLOBAL positions (offsets[0] = results of all earlier ranks);
    ``indices``: int32[nnz_local]; ``q_lo``/``q_hi``: the block of queries; ``nnz_before``/``nnz_total``."""

    __slots__ = ("q_lo", "q_hi", "offsets", "indices", "nnz_before", "nnz_total", "nnz_per_rank")


def assemble(local_offsets: torch.Tensor, local_indices: torch.Tensor, q: int, group=None) -> ShardedCsr:
    """local_offsets (int64[q_local + 1], starting at 0) and local_indices of this rank's block -> its block of the
    global CSR.  One all-gather of one int64 per rank."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    out = ShardedCsr()
    out.q_lo, out.q_hi = block_bounds(q, rank, world)
    if local_offsets.numel() != out.q_hi - out.q_lo + 1:
        raise ValueError(f"rank {rank}: expected offsets of {out.q_hi - out.q_lo + 1} entries, got {local_offsets.numel()}")
    nnz_local = local_offsets[-1].reshape(1).to(torch.int64)
    if world > 1:
        nnz_local = nnz_local.to(_comm_device(nnz_local, group))
        sizes = [torch.zeros_like(nnz_local) for _ in range(world)]
        dist.all_gather(sizes, nnz_local, group=group)
        sizes = torch.cat(sizes).cpu()
    else:
        sizes = nnz_local.cpu()
    out.nnz_per_rank = [int(x) for x in sizes.tolist()]
    out.nnz_before = sum(out.nnz_per_rank[:rank])
    out.nnz_total = sum(out.nnz_per_rank)
    out.offsets = local_offsets.to(torch.int64) + out.nnz_before
    out.indices = local_indices[: out.nnz_per_rank[rank]]
    return out


def gather_global(csr: ShardedCsr, q: int, group=None) -> tuple[torch.Tensor, torch.Tensor]:
    """Every rank receives the whole CSR (offsets int64[q + 1], indices int32[nnz_total]).  For callers that need it in
    one place and for tests; the blocks are padded to the largest one for the all-gather."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        return csr.offsets, csr.indices
    dev = csr.offsets.device
    max_rows = max(block_bounds(q, r, world)[1] - block_bounds(q, r, world)[0] for r in range(world))
    max_nnz = max(csr.nnz_per_rank)
    off_pad = torch.zeros(max_rows, dtype=torch.int64, device=dev)
    off_pad[: csr.q_hi - csr.q_lo] = csr.offsets[:-1]
    idx_pad = torch.zeros(max(max_nnz, 1), dtype=torch.int32, device=dev)
    idx_pad[: csr.indices.numel()] = csr.indices
    comm = _comm_device(off_pad, group)
    off_pad, idx_pad = off_pad.to(comm), idx_pad.to(comm)
    offs = [torch.zeros_like(off_pad) for _ in range(world)]
    idxs = [torch.zeros_like(idx_pad) for _ in range(world)]
    dist.all_gather(offs, off_pad, group=group)
    dist.all_gather(idxs, idx_pad, group=group)
    offs, idxs = [t.to(dev) for t in offs], [t.to(dev) for t in idxs]
    rows = [offs[r][: block_bounds(q, r, world)[1] - block_bounds(q, r, world)[0]] for r in range(world)]
    offsets = torch.cat(rows + [torch.tensor([csr.nnz_total], dtype=torch.int64, device=dev)])
    indices = torch.cat([idxs[r][: csr.nnz_per_rank[r]] for r in range(world)])
    return offsets, indices


def replicate_nodes(nodes: torch.Tensor, src: int = 0, group=None) -> None:
    """Broadcast a finished hierarchy (the ``nodes`` buffer of a build on rank ``src``) to every rank: 64 n bytes over
    NVLink, once per build, instead of building on every rank."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.broadcast(nodes, src=src, group=group)


def sharded_query(local_query, queries: torch.Tensor, group=None) -> ShardedCsr:
    """queries: the WHOLE batch (every rank passes the same tensor or at least its own block in place);
    local_query(block) -> (offsets int64[len(block) + 1] from 0, indices int32[>= nnz]) runs the ordinary query path
    (``binding.query`` on this rank's GPU) on this rank's block."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    q = int(queries.shape[0])
    lo, hi = block_bounds(q, rank, world)
    block = queries[lo:hi]
    if block.data_ptr() % 16 != 0:      # the C ABI wants 16-byte aligned queries: a block of 24-byte boxes may start off that
        block = block.clone()
    off, idx = local_query(block)
    return assemble(off, idx, q, group=group)
