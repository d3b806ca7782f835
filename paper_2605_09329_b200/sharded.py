"""The distillation step sharded over the vocabulary (include/tts.h "f4"): one process per GPU, rank g
owns a contiguous range of vocabulary rows of W / master / m / v and the matching teacher columns.  This module only
does the plumbing between the library's shard calls -- the partition, two tiny collectives per step
(all-gather of [T, 8] row tuples, all-reduce of gh [T, d]) and one per mask (all-gather of [T] (max, index) pairs)
through torch.distributed: NCCL over NVLink / NVSwitch on GPUs, gloo in the CPU tests.  Every arithmetic step,
including the merge of the gathered tuples, runs in the library's kernels.

Why plain NCCL calls: the exchanged tensors are 512 B .. 8 MB against 2.2 GB of local HBM traffic per rank at 8 GPUs
(DESIGN.md "Multi-GPU"); both collectives are latency-bound and sit between kernels whose inputs they are, so there
is no transfer to overlap tile by tile with the contraction that precedes them.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

from . import tts


def shard_range(V: int, rank: int, world: int, align: int = 128):
    """Rows [v0, v1) of rank `rank`: V / align blocks dealt out as evenly as possible (151936 = 128 x 1187 does not
    split evenly), every shard a multiple of `align` rows so that it stays on the tensor path."""
    if V % align != 0:
        raise ValueError("V = %d is not a multiple of %d" % (V, align))
    blocks = V // align
    if world > blocks:
        raise ValueError("more ranks (%d) than %d-row blocks (%d)" % (world, align, blocks))
    return align * (blocks * rank // world), align * (blocks * (rank + 1) // world)


def all_gather_rows(x: torch.Tensor, group=None) -> torch.Tensor:
    """[...] on every rank -> [world, ...] on every rank, rank order (identity for one process)."""
    if not (dist.is_initialized() and dist.get_world_size(group) > 1):
        return x.unsqueeze(0)
    world = dist.get_world_size(group)
    out = torch.empty((world,) + tuple(x.shape), dtype=x.dtype, device=x.device)
    if x.is_cuda:
        dist.all_gather_into_tensor(out, x.contiguous(), group=group)
    else:
        dist.all_gather(list(out.unbind(0)), x.contiguous(), group=group)
    return out


def all_reduce_sum_(x: torch.Tensor, group=None) -> torch.Tensor:
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
    return x


class ShardExchange:
    """What vocabulary shards exchange per round, as an interface: three tiny collectives between library calls.
    `TorchDistExchange` (NCCL on GPUs, gloo in the CPU tests) is the implementation shipped; a one-shot multimem /
    NVLS reduction over NVSwitch peer memory can replace it later without touching VocabShardedStep or the C ABI.
    `bytes_per_step(T, d)` is the traffic per rank and round, for bench.py's `comm` record."""

    n_shards = 1

    def gather_stats(self, stats):        # [T, 8] fp32 -> [n_shards, T, 8], rank order
        raise NotImplementedError

    def reduce_gh(self, gh):              # [T, d] fp32, summed over shards in place
        raise NotImplementedError

    def gather_argmax(self, val, idx):    # ([T] fp32, [T] i32) -> ([n_shards, T], [n_shards, T])
        raise NotImplementedError

    def bytes_per_step(self, T, d):
        n = self.n_shards
        return {"all_gather_row_tuples": {"send": 32 * T, "recv": 32 * T * n},
                "all_reduce_gh": {"bytes": 4 * T * d},
                "all_gather_argmax": {"send": 8 * T, "recv": 8 * T * n}}


class TorchDistExchange(ShardExchange):
    def __init__(self, group=None):
        self.group = group
        self.n_shards = dist.get_world_size(group) if dist.is_initialized() else 1
        self.backend = dist.get_backend(group) if dist.is_initialized() else "none"

    def gather_stats(self, stats):
        return all_gather_rows(stats, self.group)

    def reduce_gh(self, gh):
        return all_reduce_sum_(gh, self.group)

    def gather_argmax(self, val, idx):
        return all_gather_rows(val, self.group), all_gather_rows(idx, self.group)


class VocabShardedStep:
    """One rank's half of the sharded round.  `cfg_local` is this rank's tts_config (its V is the shard's row count)."""

    def __init__(self, cfg_local: tts.tts_config, v_offset: int, device: int = 0, group=None, exchange=None):
        self.cfg, self.v_offset, self.group = cfg_local, v_offset, group
        self.exchange = exchange if exchange is not None else TorchDistExchange(group)
        self.dev = torch.device("cuda", device)
        self.ctx = tts.tts_ctx_create(cfg_local, device)
        T = cfg_local.T_max
        self.stats = torch.empty((T, 8), dtype=torch.float32, device=self.dev)
        self.am_val = torch.empty(T, dtype=torch.float32, device=self.dev)
        self.am_idx = torch.empty(T, dtype=torch.int32, device=self.dev)

    def close(self):
        if self.ctx is not None:
            tts.tts_ctx_destroy(self.ctx)
            self.ctx = None

    def accept_mask(self, teacher_local, draft_tokens, T, mask_out, tau_out, teacher_argmax_out=None, stream=None):
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        with torch.cuda.stream(s):
            tts.tts_shard_argmax(self.ctx, teacher_local, T, self.v_offset, self.am_val, self.am_idx, s)
            val_all, idx_all = self.exchange.gather_argmax(self.am_val[:T], self.am_idx[:T])
            tts.tts_shard_accept_mask(self.ctx, val_all, idx_all, val_all.shape[0], draft_tokens, T, mask_out, tau_out,
                                      teacher_argmax_out, s)
        return val_all.shape[0]

    def distill_step(self, teacher_local, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_scale,
                     loss_out, kl_rows_out=None, gh_out=None, gW_debug_out=None, stream=None, **extras):
        """gh_out holds the FULL gradient w.r.t. h on return (all-reduced); loss_out the global loss."""
        s = stream if stream is not None else torch.cuda.current_stream(self.dev)
        with torch.cuda.stream(s):
            tts.tts_shard_begin_step(self.ctx, teacher_local, h, W_in, T, self.stats, side_stream=s, **extras)
            stats_all = self.exchange.gather_stats(self.stats[:T])
            tts.tts_shard_finish_step(self.ctx, stats_all, stats_all.shape[0], teacher_local, h, W_in, W_out, W_master,
                                      adam_m, adam_v, pos_weight, mask, T, loss_scale, loss_out, kl_rows_out, gh_out,
                                      gW_debug_out, side_stream=s, **extras)
            if gh_out is not None:
                self.exchange.reduce_gh(gh_out)
        return stats_all.shape[0]
