"""EvoSP-3D row sharding of triangle attention over an SP group (
PAPER.md Sec. IV-B, Fig. 10).

The pair tensor is partitioned along one sequence axis, "with different SP groups operating on disjoint
contiguous shards".  For the starting-node operator the broadcast rows i are independent, so a rank
that holds rows [r0, r0 + n) of Q, K, V, G needs nothing from its peers but the bias:

  forward    bias [B,H,N,N] is "replicated across device via an all_gather that is launched asynchronously"
             (P:L201): each rank produced the n query lines j of its own shard  ->  gather_bias()
             then tri_attn_rows_fwd on the local rows (R = n, include/tri_attn.h)
  backward   tri_attn_rows_bwd on the local rows gives dQ, dK, dV, dG of those rows and a PARTIAL
             dBias = sum over the local rows of dS; the sum over ranks, handed back in the same sharding as
             the bias came in, is a reduce-scatter                                      ->  scatter_dbias()
  rotation   the ending-node operator attends along the other pair axis; "all_to_all collectives are used
             to rearrange the layout of token_pair" so that the axis that was sharded becomes
             local and the other one sharded; with the two axes swapped as well the ending-node operator
             is the starting-node one (include/tri_attn.h: ending = T . starting . T)   ->  rotate()

Only plumbing lives here (torch.distributed collectives, slicing, axis permutes); every step of the
attention itself runs in the CUDA kernels behind tri_attn_rows_fwd / tri_attn_rows_bwd.  The compute needs a
GPU (there is no CPU path); the collectives work on any backend, which is how the gloo tests drive them.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import binding


def shard_rows(N: int, world: int, rank: int) -> tuple[int, int]:
    """First row and row count of `rank`'s contiguous shard of N rows.  N must divide evenly:
    the collectives below exchange equal blocks."""
    if world <= 0 or not 0 <= rank < world:
        raise ValueError(f"rank {rank} outside world {world}")
    if N % world:
        raise ValueError(f"N={N} is not a multiple of the SP group size {world}")
    n = N // world
    return rank * n, n


def _world(group) -> int:
    return dist.get_world_size(group)


def gather_bias(bias_shard: torch.Tensor, group=None, async_op: bool = False):
    """bias_shard [B,H,n,N] (the n = N/P query lines of this rank's shard) -> bias [B,H,N,N] on every rank.
    With async_op=True returns (work, finish): call finish() after work.wait() to get the tensor (P:L201:
    the all_gather is launched asynchronously and overlapped with computation)."""
    P = _world(group)
    B, H, n, N = bias_shard.shape
    if n * P != N:
        raise ValueError(f"bias shard {tuple(bias_shard.shape)} is not 1/{P} of a square plane")
    buf = torch.empty((P, B, H, n, N), dtype=bias_shard.dtype, device=bias_shard.device)
    work = dist.all_gather_into_tensor(buf.view(-1), bias_shard.contiguous().view(-1), group=group, async_op=async_op)

    def finish():
        # [P,B,H,n,N] -> [B,H,P*n,N]: rank p's lines are query lines p*n .. p*n+n-1
        return buf.permute(1, 2, 0, 3, 4).reshape(B, H, N, N)

    return (work, finish) if async_op else finish()


def scatter_dbias(dbias_partial: torch.Tensor, group=None) -> torch.Tensor:
    """dbias_partial [B,H,N,N] fp32 (sum over this rank's rows) -> [B,H,n,N]: the sum over all ranks of the
    query lines this rank owns (reduce-scatter; Sec. 8(e))."""
    P = _world(group)
    B, H, N, N2 = dbias_partial.shape
    if N != N2 or N % P:
        raise ValueError(f"dBias {tuple(dbias_partial.shape)} cannot be scattered over {P} ranks")
    n = N // P
    src = dbias_partial.view(B, H, P, n, N).permute(2, 0, 1, 3, 4).contiguous()  # block p first
    out = torch.empty((B, H, n, N), dtype=dbias_partial.dtype, device=dbias_partial.device)
    dist.reduce_scatter_tensor(out.view(-1), src.view(-1), group=group)
    return out


def rotate(x_shard: torch.Tensor, row_dim: int = 1, col_dim: int = 3, group=None) -> torch.Tensor:
    """Axis rotation of a pair-shaped tensor between attention stages (all_to_all, Fig. 10).

    x_shard holds rows [r0, r0+n) of X along `row_dim` and all N positions along `col_dim`
    (e.g. [B,n,H,N,d] with row_dim=1, col_dim=3, or a pair tensor [B,n,N,c] with col_dim=2).
    Returns this rank's shard of X^T, T = swap of the two pair axes: the same shape, where
    out[..., j_local, ..., i, ...] = X[..., i, ..., r0 + j_local, ...] -- the formerly sharded axis is whole and
    local, the other one is sharded, and the ending-node operator on X is the starting-node one on X^T.
    Communication volume per rank: the local shard (O(N^2 c / P))."""
    P = _world(group)
    n, N = x_shard.shape[row_dim], x_shard.shape[col_dim]
    if n * P != N:
        raise ValueError(f"shard {tuple(x_shard.shape)} is not 1/{P} of a square pair tensor")
    # block p = my rows, columns of rank p; all_to_all hands it to rank p
    send = torch.stack(x_shard.split(n, dim=col_dim), dim=0).contiguous()  # [P, ..., n_i, ..., n_j, ...]
    recv = torch.empty_like(send)
    dist.all_to_all_single(recv.view(-1), send.view(-1), group=group)
    # recv[p] = rows of rank p (i = p*n + i_local), my columns j_local: swap the two axes, then lay the P blocks
    # along the (new) column axis
    blocks = [recv[p].transpose(row_dim, col_dim) for p in range(P)]  # [..., n_j, ..., n_i, ...]
    return torch.cat(blocks, dim=col_dim).contiguous()


class PeerReduceScatter:
    """The dBias reduce-scatter as ONE kernel over peer memory (tri_attn_dbias_reduce_scatter) instead of an NCCL call:
    every rank's partial dBias lives in a torch symmetric-memory buffer that its peers can load over NVLink / NVSwitch; each
    rank sums its own N / P query lines out of all P buffers in rank order (fixed order: bitwise reproducible).

        rs = PeerReduceScatter(B, H, N, group)       # collective: allocates and exchanges the buffers once
        tri_attn_rows_bwd(..., out=(dQ, dK, dV, dG, rs.buffer))
        dbias_shard = rs()                           # barrier, reduce kernel, barrier
    """

    def __init__(self, B: int, H: int, N: int, group=None, device=None):
        import torch.distributed._symmetric_memory as symm_mem

        group = dist.group.WORLD if group is None else group
        device = torch.device("cuda", torch.cuda.current_device()) if device is None else device
        shard_rows(N, _world(group), dist.get_rank(group))  # N must divide evenly
        self.shape = (B, H, N)
        self.buffer = symm_mem.empty((B, H, N, N), dtype=torch.float32, device=device)
        self.handle = symm_mem.rendezvous(self.buffer, group)

    def __call__(self, out=None):
        B, H, N = self.shape
        h = self.handle
        h.barrier()  # every rank's backward has written its buffer (stream-ordered on each rank)
        out = binding.tri_attn_dbias_reduce_scatter(list(h.buffer_ptrs), h.rank, B, H, N, out=out, device=self.buffer.device)
        h.barrier()  # nobody overwrites its buffer before every rank has read it
        return out


class PeerAllGather:
    """The bias all-gather as a pull over peer memory (tri_attn_bias_all_gather): every rank puts its shard [B,H,n,N] into a
    torch symmetric-memory buffer and copies the lines of all shards into its own full bias with one kernel.

        ag = PeerAllGather(B, H, N, dtype, group)     # collective: allocates and exchanges the buffers once
        bias = ag(bias_shard)                          # local copy into the buffer, barrier, pull kernel, barrier
    """

    def __init__(self, B: int, H: int, N: int, dtype, group=None, device=None):
        import torch.distributed._symmetric_memory as symm_mem

        group = dist.group.WORLD if group is None else group
        device = torch.device("cuda", torch.cuda.current_device()) if device is None else device
        _, n = shard_rows(N, _world(group), dist.get_rank(group))
        self.shape = (B, H, N)
        self.buffer = symm_mem.empty((B, H, n, N), dtype=dtype, device=device)
        self.handle = symm_mem.rendezvous(self.buffer, group)

    def __call__(self, bias_shard, out=None):
        B, H, N = self.shape
        h = self.handle
        self.buffer.copy_(bias_shard)
        h.barrier()  # every rank's shard is in its buffer
        out = binding.tri_attn_bias_all_gather(list(h.buffer_ptrs), B, H, N, self.buffer.dtype, out=out, device=self.buffer.device)
        h.barrier()  # nobody refills its buffer before every rank has read it
        return out


class RowShardedTriAttention:
    """Starting-node triangle attention on this rank's shard of the broadcast rows.

    forward(Q, K, V, G, bias_shard, mask) with Q,K,V,G [B,n,H,N,d] (rows r0..r0+n-1), bias_shard [B,H,n,N],
    mask [B,n,N] or None returns O [B,n,H,N,d] and LSE [B,n,H,N]; backward(dO) returns dQ, dK, dV, dG of
    the local rows and dBias_shard [B,H,n,N] fp32 (already summed over the group; by NCCL reduce-scatter, or with
    peer_reduce=True the bias all-gather and the dBias reduce-scatter both run as our kernels over peer memory:
    PeerAllGather, PeerReduceScatter).  For the ending-node operator rotate() the
    operands first.  CUDA only."""

    def __init__(self, group=None, peer_reduce: bool = False):
        self.group = group
        self._saved = None
        self._peer = peer_reduce  # both exchanges by the peer-memory kernels (symmetric memory) instead of NCCL
        self._rs = None
        self._ag = None

    def forward(self, Q, K, V, G, bias_shard, mask=None):
        if not Q.is_cuda:
            raise binding.TriAttnError("RowShardedTriAttention needs CUDA tensors (there is no CPU path)")
        if self._peer:
            B, H, n, N = bias_shard.shape
            if self._ag is None or self._ag.shape != (B, H, N) or self._ag.buffer.dtype != bias_shard.dtype:
                self._ag = PeerAllGather(B, H, N, bias_shard.dtype, self.group, Q.device)
            bias = self._ag(bias_shard)
        else:
            work, finish = gather_bias(bias_shard, self.group, async_op=True)
            work.wait()  # stream-ordered for NCCL: the kernels below are enqueued behind the all-gather
            bias = finish().contiguous()
        O, LSE = binding.tri_attn_rows_fwd(Q, K, V, G, bias, mask)
        self._saved = (Q, K, V, G, bias, mask, O, LSE)
        return O, LSE

    def backward(self, dO):
        if self._saved is None:
            raise binding.TriAttnError("backward() before forward()")
        Q, K, V, G, bias, mask, O, LSE = self._saved
        self._saved = None
        if not self._peer:
            dQ, dK, dV, dG, dBias = binding.tri_attn_rows_bwd(dO, Q, K, V, G, bias, mask, O, LSE)
            return dQ, dK, dV, dG, scatter_dbias(dBias, self.group)
        B, _, H, N, _ = Q.shape
        if self._rs is None or self._rs.shape != (B, H, N):
            self._rs = PeerReduceScatter(B, H, N, self.group, Q.device)
        grads = tuple(torch.empty_like(Q) for _ in range(4))
        binding.tri_attn_rows_bwd(dO, Q, K, V, G, bias, mask, O, LSE, out=grads + (self._rs.buffer,))
        return grads + (self._rs(),)
