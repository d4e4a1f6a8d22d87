"""N_m-sharded application of F and F^T over several ranks (one process per GPU).

How the path shards: along the spatial parameter axis.
Rank g holds the spectrum of its own parameter slice, Fhat[:, :, P_g], and the slice m[:, P_g]:

    F m    = sum_g F[:, :, P_g] m[:, P_g]   -> local tt_matvec, then ONE all-reduce (sum) of d
                                               (N_d*N_t reals: 160 KB at C3, latency-bound)
    F^T d  -> d is replicated, every rank produces its own slice of m': no collective at all
    F^T F m = rmatvec(matvec(m))            -> one all-reduce in the middle

The north star of this build is the one-GPU path (bench.py's default is independent replicas);
this wrapper is the recorded, tested route to more GPUs: torch.distributed (NCCL on GPUs, gloo in
the CPU tests) does the only exchange step the method has.  It holds none of the method's
arithmetic: the local operator is passed in (a tt Plan on a GPU; the CPU oracle in the gloo test).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


class _AllReduce:
    """In-place sum over the ranks of `group` (NCCL on GPUs, gloo in the CPU tests); nothing to do for a single rank.
    The classes below take any callable with this signature instead, which is how the one-GPU test stands in for the
    exchange step (tests/test_gpu_sharded.py: the emulated ranks' partials are summed in one process)."""

    def __init__(self, group=None):
        self.group = group

    def __call__(self, t: torch.Tensor) -> None:
        if dist.is_available() and dist.is_initialized() and dist.get_world_size(self.group) > 1:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)


def shard_range(N_m: int, rank: int, world: int, align: int = 16) -> tuple[int, int]:
    """Contiguous parameter range [p0, p1) of `rank`: equal shares, boundaries on multiples of `align`
    (the row pitch granularity of Fhat) except the last one; empty ranges only if N_m < world*align."""
    blocks = (N_m + align - 1) // align
    b0 = blocks * rank // world
    b1 = blocks * (rank + 1) // world
    return min(N_m, b0 * align), min(N_m, b1 * align)


class ShardedOperator:
    """F, F^T, F^T F with the parameter axis split over the ranks of `group`.

    local_matvec(m_local)  -> this rank's partial d  (tensor [N_t, N_d], same shape on all ranks)
    local_rmatvec(d)       -> this rank's slice of m' (tensor [N_t, p1 - p0])
    """

    def __init__(self, local_matvec, local_rmatvec, group=None, all_reduce=None):
        self.local_matvec, self.local_rmatvec, self.group = local_matvec, local_rmatvec, group
        self.all_reduce = all_reduce or _AllReduce(group)

    def matvec(self, m_local: torch.Tensor) -> torch.Tensor:
        d = self.local_matvec(m_local)
        self.all_reduce(d)                                               # the path's only exchange step
        return d

    def rmatvec(self, d: torch.Tensor) -> torch.Tensor:
        return self.local_rmatvec(d)

    def normal(self, m_local: torch.Tensor) -> torch.Tensor:
        return self.rmatvec(self.matvec(m_local))


def from_plan(plan, group=None, all_reduce=None) -> ShardedOperator:
    """Wraps a tt Plan built on this rank's slice F[:, :, p0:p1] of the block column."""
    return ShardedOperator(plan.matvec, plan.rmatvec, group, all_reduce)


class ShardedMapInference:
    """The online MAP point of eq (4.13) with the parameter axis split over the ranks.

    G* and F shard exactly like F^T and F above: G* y needs no collective (every rank owns its slice of the
    parameter field), b = F G* y is the local partial followed by the ONE all-reduce of the data vector; the
    data-space steps (Gamma_noise^{-1}, the K-solve with the replicated Cholesky factor) are replicated - they
    act on n = N_d N_t numbers.  This is what lets the paper's fp64 spectra (2 x 103 GB at its test shape) be
    held by two or more GPUs.  Like ShardedOperator this class holds none of the method's arithmetic:

      partial(d_obs) -> b_partial      the first half of eq (4.13) on the local slices (tt_map_infer_partial)
      finish(b)      -> m_map slice    the second half (tt_map_infer_finish)
      gain(d_obs)    -> m_map slice    G* K^{-1} d_obs (tt_map_infer TT_MAP_GAIN): no collective at all
    """

    def __init__(self, partial, finish, gain, group=None, all_reduce=None):
        self.partial, self.finish, self.gain, self.group = partial, finish, gain, group
        self.all_reduce = all_reduce or _AllReduce(group)

    def infer(self, d_obs: torch.Tensor, gain_form: bool = False) -> torch.Tensor:
        """This rank's slice of m_map."""
        if gain_form:
            return self.gain(d_obs)
        b = self.partial(d_obs)
        self.all_reduce(b)                                                   # the path's only exchange step
        return self.finish(b)


def map_from_binding(mp, group=None, all_reduce=None) -> ShardedMapInference:
    """Wraps a binding.MapInference built on this rank's slices of the block columns of F and G*."""
    from . import binding as tt
    state = {}

    def partial(d_obs):
        state["a"], b = mp.infer_partial(d_obs)
        return b

    def finish(b):
        return mp.infer_finish(b, state.pop("a"))

    return ShardedMapInference(partial, finish, lambda d: mp.infer(d, tt.TT_MAP_GAIN), group, all_reduce)


def assemble_K_sharded(local_product, add_noise, group=None, all_reduce=None) -> torch.Tensor:
    """K = Gamma_noise + F G* with the parameter axis sharded: F G* = sum_g F[:, :, P_g] G[:, :, P_g]^* is a sum over the ranks'
    parameter slices, so every rank forms the product of its own slices WITHOUT noise (`local_product()`:
    binding.assemble_K_direct(..., noise_var=None) on a GPU, the oracle with zero noise in the gloo test), ONE all-reduce (sum)
    of the n x n matrix follows (4.8 GB at the paper's shape), and the noise is added once, after it, by `add_noise(K)`
    (binding.tt_K_add_noise on a GPU).  No arithmetic happens here."""
    K = local_product()
    (all_reduce or _AllReduce(group))(K)
    add_noise(K)
    return K
