#!/usr/bin/env python
"""bench.py -- throughput of the TTS online-distillation step on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one pass of the whole hot path over one round of synthetic input:
tts_accept_mask (a1) + tts_distill_step (a2-a7) enqueued on a side stream, then the barrier (a8).
Default workload: BASELINE.json configs[2], the Qwen3-8B-shaped draft head (V=151936, d=4096, T=16,
bf16 weights + fp32 master, AdamW) -- the configuration the metric's >=70%-of-roofline target is
quoted on.  Inputs are seeded and synthetic (workloads/synth.py).

  value      steps/s with all inputs resident in HBM (CUDA events on the side stream, max over ranks)
  e2e        the same metric through tts_round_host: the round's teacher logits / hidden states /
             tokens / weights come from pinned HOST buffers and loss / tau / mask go back to the host
             inside the timed region
  roofline   dominant kernel (a6+a7, gW contraction fused with the AdamW update): ALGORITHMIC bytes per
             launch / mean launch duration (CUDA events recorded on the launching stream by the library's
             tts_profile_* calls) against MEASURED_PEAKS.json's copy bandwidth
  cpu_baseline  the fp64 oracle (oracle/tts_oracle.py, as it stands) timed on this box's host cores on a
             bounded vocabulary sample of the same workload

N > 1: "replicas only": every rank runs an independent replica of the step on its
own rounds, no data-path collective; value = steps of all ranks / max-over-ranks time.
--impl reference: the oracle arm (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FALLBACK_HBM_GBS = 6650.0   # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--blocks", type=int, default=5,
                    help="timed blocks of --steps steps each (barrier + events around every block); ms_per_step is the "
                         "MEDIAN block, ms_per_step_min / _max the spread (VERDICT r2: one block hid an 8%% box-to-box spread)")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel-path", default="auto", choices=["auto", "simt"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-sample-rows", type=int, default=8192, help="vocabulary rows in the oracle sample")
    ap.add_argument("--cpu-sampled-only", action="store_true",
                    help="cpu_baseline from the vocabulary sample only (skip the measured whole oracle step, ~25 s)")
    ap.add_argument("--draft-logits", default="computed", choices=["computed", "given"],
                    help="given: the drafter's own logits are passed in (tts_distill_step_ex, SURVEY 8(f) f1) and pass "
                         "a2 is skipped; the default computes them, as BASELINE.json's north_star describes")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "vocab"],
                    help="N > 1: independent replicas of the step (weak scaling, no data-path collective), or ONE step "
                         "sharded over the vocabulary (strong scaling; SURVEY 8(e): all-gather of [T,8] row tuples and "
                         "all-reduce of gh [T,d] per step over NCCL)")
    ap.add_argument("--n-seq", type=int, default=0,
                    help="override the number of concurrent sequences (rows = 16 x n_seq <= 512): the T-scaling of the "
                         "batched shape between BASELINE configs[2] (1 sequence) and configs[3] (32)")
    ap.add_argument("--moments", default="f32", choices=["f32", "bf16"],
                    help="storage format of Adam's moments: f32 (every BASELINE.json configuration) or the opt-in bf16 "
                         "variant (TTS_MOMENT_BF16, SURVEY 8(f) f4: 20 instead of 28 bytes per parameter per step)")
    ap.add_argument("--max-ctas", type=int, default=0,
                    help="SM budget of the step's persistent kernels (tts_config.max_ctas; 0 = all SMs): what the main "
                         "stream keeps while the update overlaps it (PAPER.md:426)")
    ap.add_argument("--side-priority", default="default", choices=["default", "high", "low"],
                    help="--stream: CUDA priority of the update's side stream relative to the main stream (low = the "
                         "harness's main stream is created with high priority instead)")
    ap.add_argument("--stream", action="store_true",
                    help="also run the long-generation stream protocol (BASELINE.json configs[4]; use --config 5)")
    ap.add_argument("--rounds", type=int, default=4000, help="--stream: speculation rounds per pass")
    ap.add_argument("--strides", default="1,5", help="--stream: update strides S to run")
    ap.add_argument("--standins", default="hbm,compute", help="--stream: stand-in verification kernels to run")
    ap.add_argument("--standin-gb", type=float, default=64.0,
                    help="--stream: bytes the HBM-bound stand-in reads per round (64 GB ~ one bf16 pass over a 32B target)")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                j = json.load(f)
            return float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def profiled_traffic(cfg_id):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed
    `ncu --set full` capture of this workload (profiles/r2_README.md has the command); None when there is none."""
    import csv
    p = os.path.join(ROOT, "profiles", "r2_ncu_full_config%d.csv" % cfg_id)
    if not os.path.exists(p):
        return None
    try:
        rows = list(csv.reader(open(p)))
        hdr, units = rows[0], rows[1]
        ki, ri, wi = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
        mult = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}
        for r in rows[2:]:
            if "tc_update" in r[ki]:
                return int(float(r[ri]) * mult[units[ri]] + float(r[wi]) * mult[units[wi]])
    except Exception:
        return None
    return None


def algorithmic_bytes(V, d, T, adam=True, moments="f32"):
    """SURVEY.md 8(d) / DESIGN.md "Algorithmic bytes": what the method must move per step."""
    state = (12 if moments == "f32" else 8) if adam else 4     # fp32 master (+ m, v in fp32 or bf16)
    step = V * d * (2 + state + state + 2)         # bf16 W read once, state read+written once, bf16 W written once
    step += T * V * 2 + T * d * 2 + T * d * 4      # teacher logits, h, gh
    update_kernel = V * d * (state + state + 2) + T * V * 2 + T * d * 2   # a6+a7 launch alone
    return step, update_kernel


class ClockSampler(threading.Thread):
    """Samples SM clocks and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(0.02)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def _np_bits(t):
    """bf16 torch tensor -> uint16 numpy bit patterns (what the oracle consumes)."""
    import numpy as np
    import torch
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def host_sample(case, rows):
    """The first ``rows`` vocabulary rows of a device case, as the oracle's numpy inputs."""
    Vs = min(rows, case["V"])
    return dict(teacher=_np_bits(case["teacher"][:, :Vs]), h=_np_bits(case["h"]), W=_np_bits(case["W"][:Vs]),
                master=case["master"][:Vs].cpu().numpy(), m=case["m"][:Vs].float().cpu().numpy(),
                v=case["v"][:Vs].float().cpu().numpy(), tok=case["draft_tokens"].cpu().numpy(),
                pw=case["pos_weight"].cpu().numpy(), Vs=Vs)


def time_oracle(case, sample, repeats=1):
    """One oracle step (mask + loss + gradients + AdamW, fp64) on the vocabulary sample.  Returns seconds."""
    from oracle import tts_oracle as O
    c = case["cfg"]
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        mask, tau, am = O.accept_mask(sample["teacher"], sample["tok"], case["seg_len"])
        O.distill_step(sample["teacher"], sample["h"], sample["W"], sample["master"], sample["m"], sample["v"],
                       sample["pw"], mask, seg_len=case["seg_len"], loss_scale=case["loss_scale"],
                       optimizer="sgd" if sample["m"] is None else "adamw", lr=c["lr"], beta1=c["beta1"],
                       beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], step=1)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best


def host_full(case):
    """A whole device case as the oracle's numpy inputs (bit for bit)."""
    z = lambda x: None if x is None else x.cpu().numpy()
    return dict(teacher=_np_bits(case["teacher"]), h=_np_bits(case["h"]), W=_np_bits(case["W"]), master=z(case["master"]),
                m=z(case["m"]), v=z(case["v"]), tok=case["draft_tokens"].cpu().numpy(), pw=case["pos_weight"].cpu().numpy())


def oracle_full_step(case, hc, slab=8192):
    """ONE WHOLE oracle step at full size, measured (not extrapolated): mask, full-vocabulary logits and normalisers,
    loss, gh, and gW + AdamW on EVERY vocabulary row, streamed over slabs of `slab` rows exactly as the full-size parity
    tests do (oracle/tts_oracle.py as it stands: row_normalisers, gh_full, distill_step_rows).  Returns (seconds, loss)."""
    import numpy as np
    from oracle import tts_oracle as O
    c = case["cfg"]
    V, C = case["V"], case["seg_len"]
    t0 = time.perf_counter()
    mask, tau, am = O.accept_mask(hc["teacher"], hc["tok"], C)
    z, lse_t, lse_z, kl = O.row_normalisers(hc["teacher"], hc["h"], hc["W"], slab=slab)
    omega = O.row_weights(hc["pw"], mask, O.ROWS_ALL, C)
    loss = case["loss_scale"] * float((omega * kl).sum())
    O.gh_full(z, lse_t, lse_z, hc["teacher"], hc["W"], omega, case["loss_scale"], slab=slab)
    for v0 in range(0, V, slab):
        rows = np.arange(v0, min(V, v0 + slab))
        r = O.distill_step_rows(rows, z, lse_t, lse_z, hc["teacher"], hc["h"], hc["W"][v0:v0 + slab],
                                hc["master"][v0:v0 + slab], hc["m"][v0:v0 + slab], hc["v"][v0:v0 + slab], omega,
                                loss_scale=case["loss_scale"], optimizer="adamw", lr=c["lr"], beta1=c["beta1"],
                                beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], step=1)
        O.working_copy_bits(r["master"])
    return time.perf_counter() - t0, loss


def peak_rss_gb():
    import resource
    return resource.getrusage(resource.RUSAGE_SELF).ru_maxrss / 1e6     # Linux: kilobytes


def cpu_threads():
    try:
        from threadpoolctl import threadpool_info
        n = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        n = 1
    return max(1, min(n, len(os.sched_getaffinity(0))))   # BLAS threads the matmuls use; elementwise numpy is 1 thread


def run_reference(args, rank, world):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only).

    One-canvas configurations (2, 3, 5): every step is ONE WHOLE oracle step at full size, measured.  A step takes
    ~20-40 s, so the number of steps actually run is bounded to about two minutes of work; `steps` in the line is what
    ran, `steps_requested` what was asked.  The inputs are the seeded device recipe copied to the host when a GPU is
    there (seconds), the host recipe otherwise (minutes); the oracle itself never touches the GPU.
    Config 1 is the whole (tiny) problem; config 4 (512 rows: ~2 TFLOP of fp64 per step) stays a vocabulary sample,
    scaled, and says so."""
    if rank != 0:
        return
    import numpy as np
    from workloads import synth
    cfgc = synth.CONFIGS[args.config]
    V, d = cfgc["V"], cfgc["d"]
    cores = cpu_threads()
    T_full = cfgc["n_seq"] * cfgc["seg_len"]
    if args.config in (2, 3, 5):
        import torch
        if torch.cuda.is_available():
            case = synth.make_case_device(args.config, "cuda:0")
            hc = host_full(case)
            case = {k: case[k] for k in ("cfg", "V", "d", "T", "seg_len", "loss_scale")}
            torch.cuda.empty_cache()
        else:
            hcase = synth.make_case(args.config)
            hc = dict(teacher=hcase["teacher"], h=hcase["h"], W=hcase["W"], master=hcase["master"], m=hcase["m"],
                      v=hcase["v"], tok=hcase["draft_tokens"], pw=hcase["pos_weight"])
            case = {k: hcase[k] for k in ("cfg", "V", "d", "T", "seg_len", "loss_scale")}
        first, loss = oracle_full_step(case, hc)
        budget_s = 120.0
        n = max(1, min(args.steps, int(budget_s / max(first, 1e-3))))
        times = [first]
        for _ in range(n - 1):
            times.append(oracle_full_step(case, hc)[0])
        dt = sum(times) / len(times)
        sps = 1.0 / dt
        what = ("ONE WHOLE oracle step per step, measured at full size (V=%d, d=%d, T=%d; every vocabulary row through "
                "gW + AdamW in slabs of 8192): %d step(s) run of %d requested, no warm-up, %.1f s each, peak RSS %.1f GB"
                % (V, d, T_full, n, args.steps, dt, peak_rss_gb()))
        steps_run, warm_run = n, 0
    else:
        rows = min(args.cpu_sample_rows, 4096, V)   # config 1: the whole problem
        case = synth.make_case(args.config, V=rows, n_seq=min(cfgc["n_seq"], 2) if args.config == 4 else None)
        sample = dict(teacher=case["teacher"], h=case["h"], W=case["W"], master=case["master"], m=case["m"],
                      v=case["v"], tok=case["draft_tokens"], pw=case["pos_weight"], Vs=rows)
        for _ in range(args.warmup):
            time_oracle(case, sample)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            time_oracle(case, sample)
        dt = (time.perf_counter() - t0) / args.steps
        scale = (V / rows) * (T_full / case["T"])
        sps = 1.0 / (dt * scale)
        what = "vocabulary rows 0..%d of %d (full d=%d, T=%d of %d), time scaled by %.1f (an extrapolation)" % (
            rows, V, d, case["T"], T_full, scale)
        steps_run, warm_run = args.steps, args.warmup
    line = {"impl": "reference", "metric": "distill_steps_per_sec", "value": sps, "unit": "steps/s",
            "n_gpus": args.gpus, "steps": steps_run, "warmup": warm_run, "steps_requested": args.steps,
            "warmup_requested": args.warmup, "ms_per_step": 1e3 / sps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(args.config, world, "oracle-cpu"),
            "cpu_baseline": {"value": sps, "unit": "steps/s", "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": sps, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg_id, world, path, parallelism="replicas"):
    from workloads import synth
    c = synth.CONFIGS[cfg_id]
    par = "single GPU"
    if world > 1:
        par = ("replicas x%d (no data-path collective)" % world if parallelism == "replicas" else
               "vocabulary shards x%d (all-gather [T,8] row tuples + all-reduce gh [T,d] per step, NCCL)" % world)
    kind = ("fp32 throughout, plain SGD lr=1e-3" if c["param"] == synth.F32 else "bf16 W + fp32 master, AdamW lr=1e-5")
    return {"workload": "BASELINE.json configs[%d] %s: V=%d d=%d T=%d (seg_len %d x %d seq), %s"
                        % (cfg_id - 1, c["name"], c["V"], c["d"], c["seg_len"] * c["n_seq"], c["seg_len"], c["n_seq"], kind),
            "V": c["V"], "d": c["d"], "T": c["seg_len"] * c["n_seq"],
            "optimizer": "sgd" if c["optimizer"] == synth.SGD else "adamw",
            "parallelism": par,
            "kernel_path": path,
            "l2": "working set per step (17 GB of weight state) exceeds the 126 MB L2: every step is L2-cold"}


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    from paper_2605_09329_b200 import dist_util, tts
    from workloads import synth

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the distillation step has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    tdev = torch.device(dev)
    dist_util.init("nccl", tdev)

    def barrier():
        dist_util.barrier(tdev)

    vocab = world > 1 and args.parallelism == "vocab"
    V_full = synth.CONFIGS[args.config]["V"]
    if vocab:
        # one step, every rank owns a slice of the vocabulary (rows of W / master / m / v, columns of the teacher)
        import torch.distributed as dist
        from paper_2605_09329_b200 import sharded
        v0, v1 = sharded.shard_range(V_full, rank, world)
        case = synth.make_case_device(args.config, dev, seed_offset=rank, V=v1 - v0, shared_h=True)
        dist.broadcast(case["draft_tokens"], 0)      # replicated inputs: canvas tokens (global ids), h, pos_weight
    else:
        case = synth.make_case_device(args.config, dev, seed_offset=rank, n_seq=args.n_seq or None)
    c = case["cfg"]
    V, d, T, C = case["V"], case["d"], case["T"], case["seg_len"]
    kpath = tts.TTS_PATH_AUTO if args.kernel_path == "auto" else tts.TTS_PATH_SIMT
    cfg = tts.make_config(V, d, T, C, tts.TTS_BF16, tts.TTS_BF16, tts.TTS_ADAMW, c["lr"], c["beta1"], c["beta2"],
                          c["eps"], c["weight_decay"], tts.TTS_ROWS_ALL, args.max_ctas, kpath,
                          moment_dtype=tts.TTS_MOMENT_BF16 if args.moments == "bf16" else tts.TTS_MOMENT_F32)
    if args.moments == "bf16":
        case["m"], case["v"] = case["m"].to(torch.bfloat16), case["v"].to(torch.bfloat16)
    shard = sharded.VocabShardedStep(cfg, v0, local_rank) if vocab else None
    ctx = shard.ctx if vocab else tts.tts_ctx_create(cfg, local_rank)
    W = [case["W"], torch.empty_like(case["W"])]        # W_in / W_out double buffer, swapped at the barrier (R18)
    master, m, v = case["master"], case["m"], case["v"]
    teacher, h, tok, pw = case["teacher"], case["h"], case["draft_tokens"], case["pos_weight"]
    mask = torch.zeros(T, dtype=torch.uint8, device=dev)
    tau = torch.zeros(T // C, dtype=torch.int32, device=dev)
    loss = torch.zeros(1, dtype=torch.float32, device=dev)
    gh = torch.zeros(T, d, dtype=torch.float32, device=dev)
    side = torch.cuda.Stream(device=dev)
    main = torch.cuda.current_stream()
    launches = [0]
    cur = [0]

    z_given = None
    if args.draft_logits == "given":      # what the drafter already holds after generating the canvas
        z_given = torch.cat([h[i:i + 64].float() @ case["W"].float().T for i in range(0, T, 64)], 0).contiguous()

    def step_vocab():
        shard.accept_mask(teacher, tok, T, mask, tau, None, side)
        launches[0] += 3
        shard.distill_step(teacher, h, W[cur[0]], W[1 - cur[0]], master, m, v, pw, mask, T, case["loss_scale"], loss,
                           None, gh, None, side)
        launches[0] += 2 + tts.tts_last_launch_count(ctx)      # begin (logits + sweep) + finish
        tts.tts_wait_step(ctx, main)
        cur[0] ^= 1

    def step():
        if vocab:
            return step_vocab()
        tts.tts_accept_mask(ctx, teacher, tok, T, mask, tau, None, side)
        n = tts.tts_last_launch_count(ctx)
        if z_given is None:
            tts.tts_distill_step(ctx, teacher, h, W[cur[0]], W[1 - cur[0]], master, m, v, pw, mask, T,
                                 case["loss_scale"], loss, None, gh, None, side)
        else:
            tts.tts_distill_step_ex(ctx, teacher, h, W[cur[0]], W[1 - cur[0]], master, m, v, pw, mask, T,
                                    case["loss_scale"], loss, None, gh, None, draft_logits=z_given, side_stream=side)
        launches[0] += n + tts.tts_last_launch_count(ctx)
        tts.tts_wait_step(ctx, main)      # the paper's barrier before the next draft round
        cur[0] ^= 1

    side.wait_stream(main)
    for _ in range(args.warmup):
        step()
    barrier()
    used_tensor = tts.tts_last_step_used_tensor_path(ctx)
    if not vocab:
        tts.tts_profile_enable(ctx, 1)
    launches[0] = 0
    sampler = ClockSampler(local_rank)
    sampler.start()
    # B blocks of exactly K steps, each bracketed by a barrier (which synchronises) and by CUDA events on the stream the
    # step runs on; per block the max over ranks.  The reported step time is the median block.
    block_ms, block_phase, n_prof = [], [], 0
    for _ in range(max(1, args.blocks)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(side)
        for _ in range(args.steps):
            step()
        e1.record(side)
        barrier()
        block_ms.append(dist_util.max_over_ranks(e0.elapsed_time(e1), tdev))
        if not vocab:
            ph, n = tts.tts_profile_read(ctx)      # mean per phase over this block's steps; resets the recorder
            if n > 0:
                block_phase.append(ph)
                n_prof += n
    clocks = sampler.stop()
    tts.tts_profile_enable(ctx, 0)
    loss_val = float(loss.item())

    def med(xs):
        s = sorted(xs)
        return s[len(s) // 2] if len(s) % 2 else 0.5 * (s[len(s) // 2 - 1] + s[len(s) // 2])

    ms_total = med(block_ms)
    phase_ms = [med([b[i] for b in block_phase]) for i in range(tts.TTS_NUM_PHASES)] if block_phase else \
        [0.0] * tts.TTS_NUM_PHASES
    upd_blocks = [b[4] for b in block_phase]

    # ---- end to end through HOST buffers: tts_round_host (H2D of the round's inputs, D2H of loss/tau/mask) ----
    e2e = None
    if not args.no_e2e and not vocab:
        ht = teacher.view(torch.int16).cpu().pin_memory()
        hh = h.view(torch.int16).cpu().pin_memory()
        htok, hpw = tok.cpu().pin_memory(), pw.cpu().pin_memory()
        # two result sets: at most two rounds are pending (tts_round_host_begin / _end, include/tts.h)
        hout = [(torch.zeros(1).pin_memory(), torch.zeros(T // C, dtype=torch.int32).pin_memory(),
                 torch.zeros(T, dtype=torch.uint8).pin_memory()) for _ in range(2)]
        n_begun = [0]

        def round_begin():
            hloss, htau, hmask = hout[n_begun[0] & 1]
            tts.tts_round_host_begin(ctx, ht, hh, htok, hpw, T, case["loss_scale"], W[cur[0]], W[1 - cur[0]], master, m,
                                     v, gh, hloss, htau, hmask, side)
            cur[0] ^= 1
            n_begun[0] += 1

        def rounds(k):
            # round i + 1's inputs are copied (and its a2 queued) while round i's step runs: the updates are
            # asynchronous by design; every round's H2D and D2H copies lie inside the timed region
            round_begin()
            for _ in range(k - 1):
                round_begin()
                tts.tts_round_host_end(ctx)
            tts.tts_round_host_end(ctx)

        rounds(max(3, args.warmup // 2))
        barrier()
        t0 = time.perf_counter()
        rounds(args.steps)
        barrier()
        dt = dist_util.max_over_ranks(time.perf_counter() - t0, tdev)
        # the same rounds one at a time (tts_round_host: each ends with a synchronise before the next begins)
        t1 = time.perf_counter()
        for _ in range(args.steps):
            hloss, htau, hmask = hout[0]
            tts.tts_round_host(ctx, ht, hh, htok, hpw, T, case["loss_scale"], W[cur[0]], W[1 - cur[0]], master, m, v, gh,
                               hloss, htau, hmask, side)
            cur[0] ^= 1
        dt_serial = dist_util.max_over_ranks(time.perf_counter() - t1, tdev)
        e2e = {"value": world * args.steps / dt, "unit": "steps/s",
               "h2d_bytes_per_step": int(ht.numel() * 2 + hh.numel() * 2 + htok.numel() * 4 + hpw.numel() * 4),
               "d2h_bytes_per_step": int(4 + hout[0][1].numel() * 4 + hout[0][2].numel()),
               "timing": "host clock around K rounds through tts_round_host_begin / _end from pinned host buffers, two "
                         "rounds in flight (round i + 1's H2D copy runs under round i's step); every round's copies "
                         "and its result read-back are inside the timed region",
               "one_round_at_a_time": world * args.steps / dt_serial}

    # ---- CPU baseline, rank 0 at N=1 only: ONE WHOLE oracle step, measured (one canvas: ~25 s of CPU work); the
    # 512-row configuration (~2 TFLOP of fp64 per step) keeps a vocabulary sample, scaled, and says so ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sample = host_sample(case, args.cpu_sample_rows if T <= 64 else max(512, args.cpu_sample_rows // 8))
        time_oracle(case, sample)
        sec = time_oracle(case, sample, repeats=2)
        scale = V / sample["Vs"]
        sampled = {"value": 1.0 / (sec * scale), "sample": "vocabulary rows 0..%d of %d (full d=%d, T=%d): %.2f s, "
                   "scaled by %.1f (an extrapolation)" % (sample["Vs"], V, d, T, sec, scale)}
        if T <= 64 and not args.cpu_sampled_only and args.moments == "f32":
            # the inputs of the step the GPU just timed would need its PRE-step state; the oracle's time does not
            # depend on the values, so it runs on the state as it is now (same shapes, same bits the GPU holds)
            full_s, _ = oracle_full_step(case, host_full(case))
            cpu = {"value": 1.0 / full_s, "unit": "steps/s", "cores": cpu_threads(), "kind": "oracle",
                   "sample": "ONE WHOLE oracle step, measured at full size (V=%d, d=%d, T=%d, every vocabulary row): "
                             "%.1f s, peak RSS %.1f GB, %d BLAS threads" % (V, d, T, full_s, peak_rss_gb(), cpu_threads()),
                   "sampled_estimate": sampled}
        else:
            cpu = {"value": sampled["value"], "unit": "steps/s", "cores": cpu_threads(), "kind": "oracle",
                   "sample": sampled["sample"]}

    tts.tts_ctx_destroy(ctx)
    stream = None
    if args.stream and world == 1:
        stream = run_stream(args, case, dev)
    if rank != 0:
        return
    ms_step = ms_total / args.steps
    sps = (1 if vocab else world) * 1e3 / ms_step          # shards: all ranks together take ONE step
    if vocab:
        V = V_full
    step_bytes, upd_bytes = algorithmic_bytes(V, d, T, moments=args.moments)
    if vocab:
        step_bytes //= world
    if z_given is not None:
        step_bytes += T * V * 4 - V * d * 2      # fp32 draft logits read instead of the bf16 W pass
    peak, peak_src = measured_peaks()
    upd_ms = phase_ms[4] if n_prof > 0 and phase_ms[4] > 0 else None
    roof = {"bound": "hbm", "kernel": "a6+a7 gW contraction fused with AdamW update (phase 4)",
            "achieved": (upd_bytes / (upd_ms * 1e-3) / 1e9) if upd_ms else None, "peak": peak, "unit": "GB/s",
            "frac": (upd_bytes / (upd_ms * 1e-3) / 1e9 / peak) if upd_ms else None,
            "traffic": profiled_traffic(args.config) if (z_given is None and not vocab and args.moments == "f32") else None,
            "traffic_source": "NOT measured by this run: dram__bytes_read.sum + dram__bytes_write.sum of one launch from "
                              "the committed ncu --set full capture profiles/r2_ncu_full_config%d.csv (commit d9a41c9, "
                              "2026-11-05; the update kernels' data movement is unchanged since)" % args.config,
            "peak_source": peak_src, "algorithmic_bytes_per_launch": upd_bytes, "kernel_ms": upd_ms,
            "step_algorithmic_bytes": step_bytes, "step_achieved": step_bytes / (ms_step * 1e-3) / 1e9,
            "step_frac_of_measured_copy": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
            "step_frac_of_nominal_8TBs": step_bytes / (ms_step * 1e-3) / 1e9 / 8000.0,
            "kernel_ms_min": min(upd_blocks) if upd_blocks else None,
            "kernel_ms_max": max(upd_blocks) if upd_blocks else None,
            "phase_ms": dict(zip(tts.PHASE_NAMES, phase_ms)), "profiled_steps": n_prof}
    line = {"metric": "distill_steps_per_sec", "value": sps, "unit": "steps/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
            "blocks": len(block_ms), "ms_per_step_min": min(block_ms) / args.steps,
            "ms_per_step_max": max(block_ms) / args.steps, "higher_is_better": True,
            "scaling": "strong" if vocab else "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": dict(workload_config(args.config, world, "tcgen05+tma" if used_tensor else "cuda-core",
                                           args.parallelism), **({"T": T, "n_seq_override": args.n_seq} if args.n_seq else {}),
                           draft_logits=args.draft_logits, adam_moments=args.moments),
            "rows_V_per_sec": sps * T * V, "loss": loss_val, "clocks": clocks, "e2e": e2e,
            "gpu_launches": launches[0] // len(block_ms), "gpu_launches_all_blocks": launches[0],
            "roofline": roof, "cpu_baseline": cpu}
    if stream is not None:
        line["stream"] = stream
    # what crosses the fabric per step, for the driver's rank check: replicas exchange nothing on the data path
    if world > 1:
        line["comm"] = ({"ranks": world, "backend": shard.exchange.backend, "pattern": "vocabulary shards",
                         "per_rank_bytes_per_step": shard.exchange.bytes_per_step(T, d)} if vocab else
                        {"ranks": world, "backend": "nccl", "pattern": "replicas: no data-path collective; one "
                         "max-over-ranks / sum-over-ranks scalar reduction around the timed region",
                         "per_rank_bytes_per_step": {}})
    print(json.dumps(line), flush=True)


def run_stream(args, case, dev):
    """BASELINE.json configs[4] / SURVEY 8(d): `rounds` consecutive speculation rounds on one head.  Per round the
    harness (main stream) draws h_t, builds the round's teacher ON THE DEVICE from the CURRENT weights,
    t_t = rn_bf16(h_t W_cur^T + mu_t u + 1.5 eps_t) (R16), and runs a stand-in verification kernel;
    scheduler.DraftHeadUpdater dispatches the TTS update on the side stream every S rounds and places the barrier
    S-1 rounds later.  The harness ops (torch matmul / randn / sum) stand in for the drafter and the
    verifier and are not the product; every step of the update runs in libtts_b200.so.

    Reported per (stand-in, S): rounds/s with and without updates, steady-state update steps/s from device
    timestamps recorded behind each step on the side stream (rounds >= 200), and the EXPOSED step time
    (time with updates - time without) / number of updates.  Two stand-ins because they bracket the answer: an
    HBM-bound verifier competes with the (HBM-bound) update for the same bandwidth, a tensor-bound one does not."""
    import torch
    from paper_2605_09329_b200 import tts
    from workloads import synth
    from paper_2605_09329_b200.scheduler import DraftHeadUpdater

    c = case["cfg"]
    V, d, C = case["V"], case["d"], case["seg_len"]
    T = C
    tdev = torch.device(dev)
    if args.side_priority == "low":       # the main stream outranks the side stream
        torch.cuda.set_stream(torch.cuda.Stream(device=tdev, priority=-1))
    main = torch.cuda.current_stream()
    side_prio = -1 if args.side_priority == "high" else None
    W0, master0 = case["W"].clone(), case["master"].clone()
    u = torch.from_numpy(synth.stream_direction(V, c["seed"])).to(tdev)
    pw = case["pos_weight"][:T].contiguous()
    rounds, skip = args.rounds, min(200, args.rounds // 4)
    mu_max = c.get("mu_max", 3.0)

    free, _ = torch.cuda.mem_get_info()
    nbytes = int(min(args.standin_gb * 1e9, free - 8e9))
    big = torch.empty(nbytes // 4, dtype=torch.float32, device=tdev)
    big.zero_()
    ga = torch.randn(8192, 8192, device=tdev, dtype=torch.bfloat16)
    gb = torch.randn(8192, 8192, device=tdev, dtype=torch.bfloat16)
    gc = torch.empty(8192, 8192, device=tdev, dtype=torch.bfloat16)
    sink = torch.zeros(1, device=tdev)

    def standin_hbm():
        sink.add_(big.sum())

    def time_of(fn, n=3):
        fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    hbm_ms = time_of(standin_hbm)
    mm_ms = time_of(lambda: torch.matmul(ga, gb, out=gc))
    n_mm = max(1, int(round(hbm_ms / mm_ms)))      # same duration as the HBM-bound stand-in, tensor-bound instead

    def standin_compute():
        for _ in range(n_mm):
            torch.matmul(ga, gb, out=gc)

    standins = {"hbm": (standin_hbm, "%.1f GB read-reduce, %.2f ms alone" % (nbytes / 1e9, hbm_ms)),
                "compute": (standin_compute, "%d x bf16 8192^3 matmul, %.2f ms alone" % (n_mm, n_mm * mm_ms))}
    bufs = [dict(teacher=torch.empty(T, V, dtype=torch.bfloat16, device=tdev),
                 h=torch.empty(T, d, dtype=torch.bfloat16, device=tdev),
                 tok=torch.empty(T, dtype=torch.int32, device=tdev)) for _ in range(2)]
    noise = torch.empty(T, V, dtype=torch.float32, device=tdev)
    hf = torch.empty(T, d, dtype=torch.float32, device=tdev)

    def one_pass(kind, stride, with_updates):
        m, v = torch.zeros_like(master0), torch.zeros_like(master0)
        master, W = master0.clone(), W0.clone()
        up = DraftHeadUpdater(W, master, m, v, seg_len=C, T_max=T, stride=stride, lr=c["lr"], beta1=c["beta1"],
                              beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], want_gh=True,
                              max_ctas=args.max_ctas, priority=side_prio)
        g = torch.Generator(device=tdev)
        g.manual_seed(1000003 * (c["seed"] + 1))
        fn = standins[kind][0]
        marks = []
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        for t in range(rounds):
            if t == skip:
                e0.record(main)
            b = bufs[0] if t % stride == 0 else bufs[1]     # a dispatching round's buffers rest until the barrier (R17)
            hf.normal_(0.0, 1.0, generator=g)
            b["h"].copy_(hf)
            z = torch.matmul(b["h"], up.weights().T).float()            # the drafter's logits from the CURRENT head
            noise.normal_(0.0, 1.0, generator=g)
            b["tok"].copy_(torch.argmax(z, dim=1))
            b["teacher"].copy_(z.add_(u, alpha=synth.stream_mu(t, rounds, mu_max)).add_(noise, alpha=1.5))
            fn()                                                           # stand-in verification
            if with_updates:
                if up.on_round_end(b["teacher"], b["h"], b["tok"], pw, T, 1.0, main) and t >= skip:
                    ev = torch.cuda.Event(enable_timing=True)
                    ev.record(up.side)
                    marks.append(ev)
        up.barrier(main)
        e1.record(main)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        out = {"ms": ms, "updates_timed": len(marks)}
        if with_updates:
            out["steps_per_s"] = (len(marks) - 1) / (marks[0].elapsed_time(marks[-1]) * 1e-3) if len(marks) > 1 else None
            out["launches"] = up.launches
            out["final_loss"] = float(up.loss.item())
            ok = bool(torch.isfinite(master).all()) and bool(torch.isfinite(m).all()) and bool(torch.isfinite(v).all())
            ok = ok and bool((up.weights() == master.to(torch.bfloat16)).all())
            ok = ok and tts.tts_get_step_count(up.ctx) == up.updates == (rounds + stride - 1) // stride
            out["invariants_ok"] = ok
        up.close()
        return out

    res = {"rounds": rounds, "timed_rounds": rounds - skip, "max_ctas": args.max_ctas,
           "side_priority": args.side_priority, "runs": []}
    for kind in [k for k in args.standins.split(",") if k in standins]:
        base = one_pass(kind, 1, False)
        for S in [int(x) for x in args.strides.split(",")]:
            w = one_pass(kind, S, True)
            n_upd = w["updates_timed"]
            res["runs"].append({
                "standin": kind, "standin_desc": standins[kind][1], "stride": S,
                "rounds_per_s_without_updates": (rounds - skip) / (base["ms"] * 1e-3),
                "rounds_per_s_with_updates": (rounds - skip) / (w["ms"] * 1e-3),
                "steady_state_steps_per_s": w["steps_per_s"],
                "exposed_step_ms": (w["ms"] - base["ms"]) / max(1, n_upd),
                "updates_timed": n_upd, "gpu_launches": w["launches"], "final_loss": w["final_loss"],
                "invariants_ok": w["invariants_ok"]})
    return res


def run_tiny(args):
    """BASELINE.json configs[0]: V=1024, d=64, T=8, fp32 throughout, plain SGD -- the CUDA-core kernels.  786 KB of
    state: the step is launch-latency-bound ("report us/step only"), so the roofline object carries the
    step's bytes over its time for the record and says so; the numbers that mean something are ms_per_step, the
    number of launches and the oracle's time on the same (whole) problem."""
    import numpy as np
    import torch
    from paper_2605_09329_b200 import tts
    from workloads import synth
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the distillation step has no CPU fallback")
    case = synth.make_case(1)
    c = case["cfg"]
    V, d, T, C = case["V"], case["d"], case["T"], case["seg_len"]
    cfg = tts.make_config(V, d, T, C, tts.TTS_F32, tts.TTS_F32, tts.TTS_SGD, c["lr"], max_ctas=args.max_ctas)
    ctx = tts.tts_ctx_create(cfg, 0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    teacher, h, tok, pw = dev(case["teacher"]), dev(case["h"]), dev(case["draft_tokens"]), dev(case["pos_weight"])
    W = [dev(case["W"]), torch.empty(V, d, device="cuda")]
    mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
    tau = torch.zeros(T // C, dtype=torch.int32, device="cuda")
    loss = torch.zeros(1, device="cuda")
    gh = torch.zeros(T, d, device="cuda")
    side, main = torch.cuda.Stream(), torch.cuda.current_stream()
    cur, launches = [0], [0]

    def step():
        tts.tts_accept_mask(ctx, teacher, tok, T, mask, tau, None, side)
        n = tts.tts_last_launch_count(ctx)
        tts.tts_distill_step(ctx, teacher, h, W[cur[0]], W[1 - cur[0]], None, None, None, pw, mask, T, 1.0, loss, None,
                             gh, None, side)
        launches[0] += n + tts.tts_last_launch_count(ctx)
        tts.tts_wait_step(ctx, main)
        cur[0] ^= 1

    side.wait_stream(main)
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    launches[0] = 0
    sampler = ClockSampler(0)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(side)
    for _ in range(args.steps):
        step()
    e1.record(side)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms_step = e0.elapsed_time(e1) / args.steps
    # the same steps replayed from CUDA graphs (one per parity of the W double buffer): at 786 KB the step is nothing
    # but launch latency, which is what capture removes (include/tts.h "CUDA-graph capture")
    graphs = []
    for parity in (0, 1):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            tts.tts_accept_mask(ctx, teacher, tok, T, mask, tau, None, side)
            tts.tts_distill_step(ctx, teacher, h, W[parity], W[1 - parity], None, None, None, pw, mask, T, 1.0, loss, None,
                                 gh, None, side)
        graphs.append(g)
    with torch.cuda.stream(side):
        for i in range(4):
            graphs[(cur[0] + i) & 1].replay()
        torch.cuda.synchronize()
        e0.record(side)
        for i in range(args.steps):
            graphs[(cur[0] + i) & 1].replay()
        e1.record(side)
    tts.tts_record_done(ctx, side)
    torch.cuda.synchronize()
    cur[0] = (cur[0] + 4 + args.steps) & 1
    ms_graph = e0.elapsed_time(e1) / args.steps
    # end to end through host buffers
    ht, hh = case["teacher"], case["h"]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    pt, ph, ptok, ppw = pin(ht), pin(hh), pin(case["draft_tokens"]), pin(case["pos_weight"])
    hloss, htau, hmask = torch.zeros(1).pin_memory(), torch.zeros(T // C, dtype=torch.int32).pin_memory(), torch.zeros(T, dtype=torch.uint8).pin_memory()
    for _ in range(3):
        tts.tts_round_host(ctx, pt, ph, ptok, ppw, T, 1.0, W[cur[0]], W[1 - cur[0]], None, None, None, gh, hloss, htau, hmask, side)
        cur[0] ^= 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        tts.tts_round_host(ctx, pt, ph, ptok, ppw, T, 1.0, W[cur[0]], W[1 - cur[0]], None, None, None, gh, hloss, htau, hmask, side)
        cur[0] ^= 1
    dt = time.perf_counter() - t0
    tts.tts_ctx_destroy(ctx)
    # the oracle on the whole problem
    from oracle import tts_oracle as O
    def oracle_step():
        m_, _, _ = O.accept_mask(case["teacher"], case["draft_tokens"], C)
        O.distill_step(case["teacher"], case["h"], case["W"], None, None, None, case["pos_weight"], m_, seg_len=C,
                       loss_scale=1.0, optimizer="sgd", lr=c["lr"])
    oracle_step()
    t0 = time.perf_counter()
    for _ in range(20):
        oracle_step()
    osec = (time.perf_counter() - t0) / 20
    step_bytes = V * d * (4 + 4 + 4) + T * V * 4 + T * d * 8
    peak, peak_src = measured_peaks()
    ach = step_bytes / (ms_step * 1e-3) / 1e9
    line = {"metric": "distill_steps_per_sec", "value": 1e3 / ms_step, "unit": "steps/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[0] tiny_fp32: V=1024 d=64 T=8, fp32 throughout, plain SGD lr=1e-3",
                       "V": V, "d": d, "T": T, "optimizer": "sgd", "parallelism": "single GPU", "kernel_path": "cuda-core",
                       "l2": "786 KB of state: L2-resident, the step is launch-latency-bound"},
            "rows_V_per_sec": 1e3 / ms_step * T * V, "loss": float(loss.item()), "clocks": clocks,
            "graph_replay_ms_per_step": ms_graph,
            "e2e": {"value": args.steps / dt, "unit": "steps/s", "h2d_bytes_per_step": int(pt.numel() * 4 + ph.numel() * 4 + T * 8),
                    "d2h_bytes_per_step": int(4 + T // C * 4 + T),
                    "timing": "host clock around K tts_round_host calls (each ends with a stream synchronise)"},
            "gpu_launches": launches[0],
            "roofline": {"bound": "hbm", "kernel": "whole step (latency-bound: %d launches of CUDA-core kernels over 786 KB)" % (launches[0] // max(args.steps, 1)),
                         "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": step_bytes, "kernel_ms": ms_step},
            "cpu_baseline": {"value": 1.0 / osec, "unit": "steps/s", "cores": cpu_threads(), "kind": "oracle",
                             "sample": "the whole configuration (V=1024, d=64, T=8): %.2f ms per oracle step" % (osec * 1e3)}}
    print(json.dumps(line), flush=True)


def launch_ranks(n, argv, device_count, script=None, run=None):
    """`bench.py --gpus N` started as ONE plain process (no torchrun around it, WORLD_SIZE unset): start the N ranks
    here, one per GPU, the way the contract's torchrun line does, and return their exit code.  Refuses, loudly, to
    pretend: with fewer than N devices there is no N-GPU number to print."""
    import socket
    import subprocess
    if device_count < n:
        raise SystemExit("bench.py --gpus %d: this node has %d CUDA device(s); refusing to run %d ranks on fewer GPUs "
                         "(a rank per GPU is the only configuration this bench measures)" % (n, device_count, n))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n),
           "--master-addr", "127.0.0.1", "--master-port", str(port), script or os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")      # the communicator / transport lines the driver's rank check reads
    return (run or subprocess.call)(cmd, env=env)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        import torch
        sys.exit(launch_ranks(args.gpus, sys.argv[1:], torch.cuda.device_count()))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and args.impl != "reference" and rank == 0:
        sys.stderr.write("bench.py: --gpus %d but WORLD_SIZE=%d; n_gpus in the line is the ranks that joined (%d)\n"
                         % (args.gpus, world, world))
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.config == 1:
        if rank == 0:
            run_tiny(args)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
