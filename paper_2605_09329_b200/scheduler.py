"""Strided, asynchronous scheduling of the TTS update around the C-ABI step (Fig. 7).

    "Every S speculation rounds, a gradient update is dispatched to a side CUDA stream and overlaps with the next
     S-1 rounds on the main stream ... A synchronization barrier is inserted after S-1 rounds to ensure that the
     speculator is adjusted with the prior update before the next canvas of draft tokens are generated."

`DraftHeadUpdater` owns what that needs and nothing else: the side stream, the library context, the W_in / W_out
double buffer (R18: draft rounds keep reading the old weights while the update writes the new ones; the
buffers swap at the barrier), the device outputs of the last step, and a snapshot of the pristine head for the
paper's reset between requests.  Every step of the method runs in libtts_b200.so; this file only
orders calls and swaps pointers.  Each update consumes the signal of the most recent round only, "without any
accumulation across the S-1 skipped rounds".
"""
from __future__ import annotations

import torch

from . import tts


class DraftHeadUpdater:
    def __init__(self, W, master, adam_m, adam_v, *, seg_len, T_max, stride=1, lr=1e-5, beta1=0.9, beta2=0.999,
                 eps=1e-8, weight_decay=0.0, optimizer=tts.TTS_ADAMW, logits_dtype=tts.TTS_BF16,
                 mask_mode=tts.TTS_ROWS_ALL, max_ctas=0, host_barrier=False, want_gh=True, keep_snapshot=False,
                 use_graph=False, moment_dtype=tts.TTS_MOMENT_F32, flags=0, priority=None):
        assert stride >= 1
        V, d = W.shape
        self.V, self.d, self.seg_len, self.T_max, self.stride = V, d, seg_len, T_max, int(stride)
        self.device = W.device
        self.W = [W, torch.empty_like(W)]
        self.cur = 0
        self.master, self.m, self.v = master, adam_m, adam_v
        self.host_barrier = host_barrier          # CPU-side barrier in front of CUDA-graph replay
        # priority: CUDA stream priority of the side stream (None = default; -1 = high, 0 = low on this device)
        self.side = (torch.cuda.Stream(device=self.device) if priority is None else
                     torch.cuda.Stream(device=self.device, priority=priority))
        cfg = tts.make_config(V, d, T_max, seg_len, tts.TTS_BF16, logits_dtype, optimizer, lr, beta1, beta2, eps,
                              weight_decay, mask_mode, max_ctas, moment_dtype=moment_dtype, flags=flags)
        self.ctx = tts.tts_ctx_create(cfg, self.device.index or 0)
        self.mask = torch.zeros(T_max, dtype=torch.uint8, device=self.device)
        self.tau = torch.zeros(T_max // seg_len, dtype=torch.int32, device=self.device)
        self.loss = torch.zeros(1, dtype=torch.float32, device=self.device)
        self.kl_rows = torch.zeros(T_max, dtype=torch.float32, device=self.device)
        self.gh = torch.zeros(T_max, d, dtype=torch.float32, device=self.device) if want_gh else None
        # CUDA-graph replay of the whole step (include/tts.h "CUDA-graph capture"): one captured graph
        # per parity of the W double buffer, fed from static input buffers; captured lazily for (T, loss_scale)
        self.use_graph = bool(use_graph)
        self._graphs, self._graph_key, self._static = None, None, None
        self.round = 0                 # rounds seen since the last reset
        self.pending_since = None      # round index at which the in-flight update was dispatched
        self.updates = 0
        self.launches = 0
        self._snap = None
        if keep_snapshot:
            self.snapshot()

    # ------------------------------------------------------------------ what the drafter reads
    def weights(self):
        """The working weights the next draft round must use (valid on the main stream)."""
        return self.W[self.cur]

    # ------------------------------------------------------------------ per round
    def on_round_end(self, teacher_logits, h, draft_tokens, pos_weight, T, loss_scale=1.0, main_stream=None):
        """Call once per speculation round after verification produced `teacher_logits` on the main stream.
        Round r with r % S == 0 dispatches an update on the side stream; the barrier falls S-1 rounds later, at the
        end of round r + S - 1, i.e. before the draft of round r + S.  The buffers passed on a dispatching round
        must stay untouched until that barrier (R17).  Returns True when this round dispatched an update."""
        main = main_stream or torch.cuda.current_stream(self.device)
        r = self.round
        self.round += 1
        dispatched = False
        if r % self.stride == 0:
            assert self.pending_since is None
            if self.use_graph:
                self._dispatch_graph(teacher_logits, h, draft_tokens, pos_weight, T, loss_scale, main)
            else:
                self.side.wait_stream(main)        # the round's signal exists once main reaches this point
                self._enqueue(teacher_logits, h, draft_tokens, pos_weight, T, loss_scale, self.cur)
            self.pending_since = r
            self.updates += 1
            dispatched = True
        if self.pending_since is not None and r - self.pending_since == self.stride - 1:
            self.barrier(main)
        return dispatched

    def _enqueue(self, teacher_logits, h, draft_tokens, pos_weight, T, loss_scale, parity):
        tts.tts_accept_mask(self.ctx, teacher_logits, draft_tokens, T, self.mask, self.tau, None, self.side)
        n = tts.tts_last_launch_count(self.ctx)
        tts.tts_distill_step(self.ctx, teacher_logits, h, self.W[parity], self.W[1 - parity], self.master, self.m,
                             self.v, pos_weight, self.mask, T, loss_scale, self.loss, self.kl_rows, self.gh, None,
                             self.side)
        self._launches_per_step = n + tts.tts_last_launch_count(self.ctx)
        self.launches += self._launches_per_step

    def _dispatch_graph(self, teacher_logits, h, draft_tokens, pos_weight, T, loss_scale, main):
        key = (T, float(loss_scale), teacher_logits.dtype)
        if self._graph_key != key:
            st = dict(teacher=torch.empty_like(teacher_logits[:T]), h=torch.empty_like(h[:T]),
                      tok=torch.empty_like(draft_tokens[:T]), pw=torch.empty_like(pos_weight[:T]))
            graphs = []
            for parity in (0, 1):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=self.side):
                    self._enqueue(st["teacher"], st["h"], st["tok"], st["pw"], T, loss_scale, parity)
                self.launches -= self._launches_per_step      # captured, not launched
                graphs.append(g)
            self._graphs, self._graph_key, self._static = graphs, key, st
        self.side.wait_stream(main)
        st = self._static
        with torch.cuda.stream(self.side):                    # the round's signal -> the graph's static inputs
            st["teacher"].copy_(teacher_logits[:T], non_blocking=True)
            st["h"].copy_(h[:T], non_blocking=True)
            st["tok"].copy_(draft_tokens[:T], non_blocking=True)
            st["pw"].copy_(pos_weight[:T], non_blocking=True)
            self._graphs[self.cur].replay()
        tts.tts_record_done(self.ctx, self.side)
        self.launches += self._launches_per_step

    def barrier(self, main_stream=None):
        """The paper's barrier: the main stream (or, with host_barrier, the CPU) waits for the in-flight update;
        then the double buffer swaps so that the next draft reads the updated weights."""
        if self.pending_since is None:
            return
        main = main_stream or torch.cuda.current_stream(self.device)
        if self.host_barrier:
            tts.tts_sync_step(self.ctx)
        else:
            tts.tts_wait_step(self.ctx, main)
        self.cur ^= 1
        self.pending_since = None

    # ------------------------------------------------------------------ per request
    def snapshot(self):
        """Keep a copy of the head as it is now (normally the pristine, pre-trained head)."""
        self.barrier()
        self._snap = dict(W=self.W[self.cur].clone(), master=self.master.clone(),
                          m=None if self.m is None else self.m.clone(), v=None if self.v is None else self.v.clone(),
                          step=tts.tts_get_step_count_on(self.ctx, self.side))   # waits for the side stream only

    def restore(self):
        """"resets the speculator between requests so per-request adaptation is bounded"."""
        assert self._snap is not None, "snapshot() first"
        self.barrier()
        torch.cuda.current_stream(self.device).wait_stream(self.side)
        self.W[self.cur].copy_(self._snap["W"])
        self.master.copy_(self._snap["master"])
        if self.m is not None:
            self.m.copy_(self._snap["m"])
            self.v.copy_(self._snap["v"])
        tts.tts_set_step_count_async(self.ctx, self._snap["step"], self.side)   # ordered before the next step, no host sync
        self.round = 0

    def close(self):
        if self.ctx is not None:
            tts.tts_ctx_destroy(self.ctx)
            self.ctx = None
