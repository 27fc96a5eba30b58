#!/usr/bin/env python
"""bench.py — LVSA block-sparse attention forward on B200.

One "step" = one pass of the whole hot path for one denoising step: build the block index on the
GPU (a1-a5) and run the attention forward (a6) on one batch of synthetic Wan-2.1-1.3B 6x-horizon
tensors (BASELINE.json configs[2]: T=121, P=1560, N=188760, H=12, d=128, bf16).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

Prints ONE JSON line (rank 0).  `value` = effective TFLOP/s counting only computed tiles.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2605_31057_b200 import inputs  # noqa: E402

METRIC = "ms/attention call and effective TFLOPS (% of B200 bf16 peak) vs all-tiles dense"
UNIT = "TFLOP/s"   # both arms print this unit; what each arm counts is in the line's "unit_detail"
UNIT_DETAIL = "bf16 in / fp32 accumulate; FLOPs of the computed tiles only (4 d per computed (row, column) pair)"
REF_UNIT_DETAIL = "fp64; exact Eq. 2 FLOPs (4 d per attended (row, key) pair)"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


class ClockSampler:
    """Samples nvidia-smi SM clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu: int):
        self.gpu, self.rows, self.proc, self.first = gpu, [], None, 0

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "25"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def mark(self):
        """Call at the start of the timed region: stop() then reports only the samples taken after it."""
        self.first = len(self.rows)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows, window = self.rows[self.first:], "timed region"
        if not rows and self.rows:      # a region shorter than one sampling period: the sample just before it
            rows, window = self.rows[-1:], "last sample before the timed region (region shorter than the sampling period)"
        for r in rows:
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for n, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm), "window": window}


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one attention launch and the tensor-pipe busy
    percentage (sm__pipe_tensor_cycles_active), from the committed `ncu --set full` capture of this
    workload (profiles/traffic.csv names the summary they came from); never measured live, None when
    no capture exists for this workload."""
    import csv
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None, None, None
    with open(p, newline="") as f:
        for row in csv.DictReader(f):
            if row["workload"] == workload:
                pct = row.get("tensor_pipe_active_pct")
                src = row["source"]
                if row.get("captured"):      # when and on which commit the capture was taken: a stale row shows
                    src = "captured " + row["captured"] + "; " + src
                return int(row["dram_bytes_per_launch"]), src, (float(pct) if pct else None)
    return None, None, None


def dist_setup(n_gpus: int):
    from paper_2605_31057_b200 import replicas
    return replicas.setup("nccl")


# ------------------------------------------------------------------------------------------
def run_ours(args):
    from paper_2605_31057_b200 import binding
    rank, world, local, dist = dist_setup(args.gpus)
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    w = inputs.WORKLOADS[args.workload]
    if args.window is not None or args.anchors is not None:
        import dataclasses
        w = dataclasses.replace(w, W=w.W if args.window is None else args.window,
                                a=w.a if args.anchors is None else args.anchors)
    pk = peaks()
    from paper_2605_31057_b200 import replicas
    shard = args.shard == "heads"
    H_full = w.H
    if shard:
        # strong scaling: heads [h_lo, h_hi) of ONE call (same seed on every rank), H_r heads per rank,
        # no collective; the sub-tensor is made contiguous once, outside any timing
        import dataclasses
        h_lo, h_hi = replicas.head_shard(w.H, world, rank)
        qf, kf, vf = inputs.make_qkv(w, f"cuda:{local}", torch.bfloat16, seed=w.seed)
        q, k, v = (x[:, :, h_lo:h_hi, :].contiguous() for x in (qf, kf, vf))
        del qf, kf, vf
        w = dataclasses.replace(w, H=h_hi - h_lo)
    else:
        q, k, v = inputs.make_qkv(w, f"cuda:{local}", torch.bfloat16, seed=w.seed + rank)
    layout_kw = {}
    if args.layout == "hnd":   # [B, H, N, d]: every head's tokens contiguous (lvsa_params_t.layout)
        q, k, v = (x.transpose(1, 2).contiguous() for x in (q, k, v))
        layout_kw["layout"] = binding.LAYOUT_HND
    out = torch.empty_like(q)
    lse = torch.empty((w.B, w.H, w.N), device=dev, dtype=torch.float32)
    stream = torch.cuda.current_stream()
    steps_cycle = list(w.steps) if w.steps else [0]

    kernel_of = {"default": binding.KERNEL_AUTO, "quad": binding.KERNEL_TCGEN05_QUAD, "hybrid": binding.KERNEL_TCGEN05_HYBRID,
                 "v0": binding.KERNEL_TCGEN05_V0}

    def build(s, **kw):
        kw.setdefault("kernel", kernel_of[args.kernel])
        kw.update(layout_kw)
        return binding.lvsa_build_block_index_ex(
            stream=stream.cuda_stream, T=w.T, P=w.P, H=w.H, d=w.d, B=w.B, window=w.W, anchors=w.a,
            step=s, layer=w.layers[0] if w.layers else 0, n_text=w.n_text, initial_anchors=w.k0, **kw)

    def tile_flop(kept_cols):
        """Computed-tile work: S = Q K^T and O += P V over tile_q rows x the kept kv columns."""
        return float(kept_cols) * w.tile * 4.0 * w.d * w.H * w.B

    # kept tiles / columns per distinct step of the cycle (lvsa_index_info synchronises, so it stays
    # out of the timed region)
    nnz_of, cols_of = {}, {}
    for s in sorted(set(steps_cycle)):
        ix0 = build(s)
        i0 = ix0.info()
        nnz_of[s], cols_of[s] = i0.nnz, i0.kept_cols
        ix0.destroy()

    def one_step(i):
        # the index lives in stream-ordered memory: destroying it right after the launch frees it
        # behind the attention kernel, with no host synchronisation anywhere in the step
        ix = build(steps_cycle[i % len(steps_cycle)])
        binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
        n = ix.launches()
        ix.destroy()
        return n

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: K whole steps
    # nvidia-smi needs a few hundred ms to deliver its first sample: start it before the warm-up and
    # report only what it saw from the start of the timed region on (sampler.mark below)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for i in range(args.warmup):
        one_step(i)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # the dominant kernel is timed where it runs: one event pair around the attention launch of
    # every timed step, on the launching stream (events cost nothing on the device)
    ka = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    kb = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    barrier()
    sampler.mark()
    e0.record(stream)
    attn_launches, build_launches = 1, 4
    for i in range(args.steps):
        ix = build(steps_cycle[i % len(steps_cycle)])
        ka[i].record(stream)
        binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
        kb[i].record(stream)
        attn_launches, build_launches = ix.launches(), ix.build_launches()
        ix.destroy()
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = e0.elapsed_time(e1)
    launches_per_step = build_launches + attn_launches   # index-builder kernels (4; 7 with quad lists) + attention
    step_nnz = [nnz_of[steps_cycle[i % len(steps_cycle)]] for i in range(args.steps)]
    tile_flops = sum(tile_flop(cols_of[steps_cycle[i % len(steps_cycle)]]) for i in range(args.steps))
    nnz_mean = float(np.mean(step_nnz))
    kern_all = [a.elapsed_time(b) for a, b in zip(ka, kb)]
    kern_ms = float(np.mean(kern_all))                                        # sustained, inside the step
    kern_median, kern_min = float(np.median(kern_all)), float(np.min(kern_all))
    kern_flops = tile_flops / args.steps

    # ---- the same kernel timed alone after an idle gap (burst clocks, no power cap yet): min of 5
    ix_k = build(steps_cycle[min(1, len(steps_cycle) - 1)])
    burst_flops = tile_flop(cols_of[steps_cycle[min(1, len(steps_cycle) - 1)]])
    burst = []
    for _ in range(5):
        torch.cuda.synchronize()
        time.sleep(0.25)
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record(stream)
        binding.lvsa_attn_fwd(q, k, v, ix_k, out, lse, stream.cuda_stream)
        k1.record(stream)
        torch.cuda.synchronize()
        burst.append(k0.elapsed_time(k1))
    burst_ms = float(min(burst))

    # ---- the frame-aligned kv tiling (row f4, reading R25) on the same inputs: same timing recipe as
    # the headline kernel (back to back inside a loop, and alone after an idle gap)
    fa_line = None
    if rank == 0 and not args.no_dense and args.kernel == "default":
        s_fa = steps_cycle[min(1, len(steps_cycle) - 1)]
        ix_fa = build(s_fa, kv_tiling=binding.KV_TILES_FRAME_ALIGNED)
        i_fa = ix_fa.info()

        def time_loop(ix, n):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(3):
                binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
            a.record(stream)
            for _ in range(n):
                binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
            b.record(stream)
            torch.cuda.synchronize()
            return a.elapsed_time(b) / n
        # the two tilings alternate (A B A B) so that neither always runs on the warmer chip
        n_fa = max(5, min(args.steps, 10))
        t4 = [time_loop(ix, n_fa) for ix in (ix_fa, ix_k, ix_fa, ix_k)]
        fa_ms, tok_ms = 0.5 * (t4[0] + t4[2]), 0.5 * (t4[1] + t4[3])
        fa_line = {"ms": round(fa_ms, 4), "ms_token0_same_loop": round(tok_ms, 4), "nnz": int(i_fa.nnz),
                   "kept_cols": int(i_fa.kept_cols), "kept_cols_token0": int(cols_of[s_fa]),
                   "tflops_computed": round(tile_flop(i_fa.kept_cols) / (fa_ms * 1e-3) / 1e12, 1),
                   "note": "fewer computed columns, more tile visits: no gain, the kernel's time follows the tile visits (DESIGN.md 7.2c)"}
        ix_fa.destroy()

    # ---- the 4-CTA-cluster variant (row f4: K/V shared by two MMA pairs through one multicast load):
    # same loops, alternating with the default kernel, SM clock sampled during each loop
    quad_line = None
    # (timed only on shapes whose QUAD results are checked against the oracle: tests/test_gpu_quad.py)
    quad_checked = args.workload in ("wan1.3b_1x", "wan1.3b_6x", "wan14b_6x", "hv1.5_2x")
    if rank == 0 and not args.no_dense and w.d == 128 and args.kernel == "default" and quad_checked:
        s_q = steps_cycle[min(1, len(steps_cycle) - 1)]
        ix_q = build(s_q, kernel=binding.KERNEL_TCGEN05_QUAD)

        def timed(ix, n):
            smp = ClockSampler(local)
            smp.start()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(3):
                binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
            a.record(stream)
            for _ in range(n):
                binding.lvsa_attn_fwd(q, k, v, ix, out, lse, stream.cuda_stream)
            b.record(stream)
            torch.cuda.synchronize()
            return a.elapsed_time(b) / n, smp.stop()["sm_mhz"]
        n_q = max(10, min(args.steps, 20))
        r4 = [timed(ix, n_q) for ix in (ix_q, ix_k, ix_q, ix_k)]
        mhz = lambda a, b: None if a is None or b is None else round(0.5 * (a + b), 0)
        quad_line = {"ms": round(0.5 * (r4[0][0] + r4[2][0]), 4), "ms_pair_kernel_same_loops": round(0.5 * (r4[1][0] + r4[3][0]), 4),
                     "sm_mhz": mhz(r4[0][1], r4[2][1]), "sm_mhz_pair_kernel": mhz(r4[1][1], r4[3][1]),
                     "grid_ctas": ix_q.grid(), "grid_ctas_pair_kernel": ix_k.grid(),
                     "note": "K/V loaded once per 4-CTA cluster (half the L2 -> SM traffic); 4-CTA clusters cannot cover every SM (DESIGN.md 7.2d)"}
        ix_q.destroy()

    # ---- index build alone (a1-a5): 4 kernels, enqueue only; device time by events, host time by clock
    torch.cuda.synchronize()
    nb = 20
    b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    b0.record(stream)
    for i in range(nb):
        build(i).destroy()
    b1.record(stream)
    build_host_us = (time.perf_counter() - t0) / nb * 1e6
    torch.cuda.synchronize()
    build_us = b0.elapsed_time(b1) / nb * 1e3

    # ---- the allocation-free builder (lvsa_build_csr_static: CSR into caller arrays, fixed scratch in the
    # library image), same steps, for callers whose allocator owns the GPU; None beyond its size limits
    static_us = None
    if rank == 0 and w.T + (1 if w.n_text else 0) <= binding.STATIC_MAX_FRAMES and -(-w.N // w.tile) <= binding.STATIC_MAX_Q_TILES:
        nq_s, cap_s = -(-w.N // w.tile), max(nnz_of.values())
        s_arr = (torch.empty(nq_s + 1, dtype=torch.int32, device=dev), torch.empty(cap_s, dtype=torch.int32, device=dev),
                 torch.empty(cap_s, dtype=torch.uint8, device=dev), torch.empty(1, dtype=torch.int32, device=dev))
        s_kw = dict(T=w.T, P=w.P, d=w.d, window=w.W, anchors=w.a, n_text=w.n_text, initial_anchors=w.k0)
        for i in range(3):
            binding.lvsa_build_csr_static(*s_arr, stream=stream.cuda_stream, step=steps_cycle[i % len(steps_cycle)], **s_kw)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        for i in range(nb):
            binding.lvsa_build_csr_static(*s_arr, stream=stream.cuda_stream, step=steps_cycle[i % len(steps_cycle)], **s_kw)
        s1.record(stream)
        torch.cuda.synchronize()
        static_us = s0.elapsed_time(s1) / nb * 1e3
        assert int(s_arr[3].item()) == nnz_of[steps_cycle[(nb - 1) % len(steps_cycle)]]   # same kept-tile count as the handle path
        del s_arr

    # ---- whole-schedule driver: all T_per phase indices built once, then an
    # S x L replay is attention launches only; here one launch per phase replayed from a CUDA graph
    sched_line = None
    if rank == 0 and not args.no_schedule:
        torch.cuda.synchronize()
        # warm-up: the first creation grows the stream-ordered pool by T_per arenas (milliseconds)
        binding.lvsa_schedule_create(stream=stream.cuda_stream, T=w.T, P=w.P, H=w.H, d=w.d, B=w.B,
                                     window=w.W, anchors=w.a, **layout_kw).destroy()
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        sched = binding.lvsa_schedule_create(stream=stream.cuda_stream, T=w.T, P=w.P, H=w.H, d=w.d, B=w.B,
                                             window=w.W, anchors=w.a, **layout_kw)
        c1.record(stream)
        torch.cuda.synchronize()
        phases = sched.num_phases()
        side = torch.cuda.Stream()
        side.wait_stream(stream)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                for r in range(phases):
                    binding.lvsa_schedule_attn_fwd(sched, r, q, k, v, out, lse, stream=side.cuda_stream)
        stream.wait_stream(side)
        graph.replay()
        torch.cuda.synchronize()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        graph.replay()
        g1.record(stream)
        torch.cuda.synchronize()
        S_sched = 50   # denoising steps of the schedule the configs name ("step 25 of 50")
        sched_line = {"phases": phases, "create_all_phases_us": round(c0.elapsed_time(c1) * 1e3, 1),
                      "index_us_per_step_amortised_over_%d_steps" % S_sched: round(c0.elapsed_time(c1) * 1e3 / S_sched, 2),
                      "index_us_per_step_rebuilt": round(build_us, 1),
                      "graph_replay_ms_per_attention_call": round(g0.elapsed_time(g1) / phases, 4),
                      "paper_cpu_rebuild_us": "< 200 per step on one CPU core (PAPER.md:91), frame-level metadata only"}
        del graph
        sched.destroy()

    # ---- all-tiles (dense, Eq. 1) path of the same kernel, for the speedup line (rank 0, N = 1)
    dense_ms = None
    if rank == 0 and not args.no_dense:
        ixd = binding.lvsa_build_block_index_ex(
            stream=stream.cuda_stream, T=w.T, P=w.P, H=w.H, d=w.d, B=w.B, window=w.W,
            anchors=binding.ALL_TILES, step=0, layer=0, **layout_kw)
        binding.lvsa_attn_fwd(q, k, v, ixd, out, lse, stream.cuda_stream)
        torch.cuda.synchronize()
        n_dense = 5
        dev_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_dense)]
        for d0, d1 in dev_ev:
            d0.record(stream)
            binding.lvsa_attn_fwd(q, k, v, ixd, out, lse, stream.cuda_stream)
            d1.record(stream)
        torch.cuda.synchronize()
        dense_all = sorted(d0.elapsed_time(d1) for d0, d1 in dev_ev)
        dense_ms = float(np.median(dense_all))
        dense_nnz = ixd.info().nnz
        dense_cols = ixd.info().kept_cols
        ixd.destroy()
        # restore the LVSA result in `out`
        binding.lvsa_attn_fwd(q, k, v, ix_k, out, lse, stream.cuda_stream)

    # ---- end to end through the C ABI with HOST buffers (H2D + kernels + D2H inside the region)
    e2e = None
    if not args.no_e2e:
        qh, kh, vh = (x.cpu().pin_memory() for x in (q, k, v))
        oh = torch.empty_like(qh).pin_memory()
        lh = torch.empty((w.B, w.H, w.N), dtype=torch.float32).pin_memory()
        n_e2e = max(1, args.steps)          # every one of the K steps, like the device-timed loop
        ixh = build(steps_cycle[0])
        binding.lvsa_attn_fwd_host(qh, kh, vh, ixh, oh, lh, stream.cuda_stream)   # warm-up: allocates the workspace
        ixh.destroy()
        barrier()
        h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        h0.record(stream)
        fl_e2e = 0.0
        for i in range(n_e2e):
            s_i = steps_cycle[i % len(steps_cycle)]
            ixh = build(s_i)
            binding.lvsa_attn_fwd_host(qh, kh, vh, ixh, oh, lh, stream.cuda_stream)   # H2D + kernel + D2H + sync
            ixh.destroy()
            fl_e2e += tile_flop(cols_of[s_i])
        h1.record(stream)
        barrier()
        e2e_ms = h0.elapsed_time(h1) / n_e2e
        bi = 3 * q.numel() * q.element_size()
        bo = out.numel() * out.element_size() + lse.numel() * 4
        e2e = {"ms": e2e_ms, "flops": fl_e2e / n_e2e, "h2d": bi, "d2h": bo, "calls": n_e2e}
        del qh, kh, vh, oh, lh

    # ---- max over ranks, aggregate
    ms_step, kern_ms, e2e_max = replicas.max_over_ranks(
        dist, [total_ms / args.steps, kern_ms, e2e["ms"] if e2e else 0.0], device=dev)
    if e2e:
        e2e["ms"] = e2e_max
    if shard:   # the ranks hold different numbers of heads: sum their work, divide by the slowest
        job_flops, job_e2e_flops = replicas.sum_over_ranks(
            dist, [tile_flops / args.steps, e2e["flops"] if e2e else 0.0], device=dev)
        value = replicas.job_throughput_sharded(job_flops, ms_step) / 1e12
        e2e_value = replicas.job_throughput_sharded(job_e2e_flops, e2e["ms"]) / 1e12 if e2e else None
    else:
        value = replicas.job_throughput(world, tile_flops / args.steps, ms_step) / 1e12
        e2e_value = replicas.job_throughput(world, e2e["flops"], e2e["ms"]) / 1e12 if e2e else None

    # ---- CPU baseline: the oracle as it stands, bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(w, q, k, v, steps_cycle[0], args.cpu_rows)
        # the same oracle on ONE core (a sixteenth of the sample), and its frame-level mask builder per
        # denoising step next to the paper's "1.4 us per call, < 200 us per rebuild"
        one = cpu_baseline(w, q, k, v, steps_cycle[0], max(8, args.cpu_rows // 16), nthreads=1)
        from oracle import lvsa_oracle as orc
        sec_rebuild, it_max, it_mean = orc.time_rebuild(w.T, w.W, w.a, 50, reps=20)
        cpu["one_core"] = {"value": one["value"], "seconds": one["seconds"], "sample": one["sample"]}
        cpu["mask_builder"] = {"us_per_step_one_core": round(sec_rebuild * 1e6, 2),
                               "us_per_frame_call": round(sec_rebuild * 1e6 / w.T, 3),
                               "alg1_loop_max": it_max, "alg1_loop_mean": round(it_mean, 3),
                               "paper": "1.4 us per call, < 200 us per rebuild, loop <= 8 (mean 1.21), PAPER.md:91"}

    if rank == 0:
        peak_sus = pk["bf16_tflops_sustained"]
        achieved = kern_flops / (kern_ms * 1e-3) / 1e12
        burst_tf = burst_flops / (burst_ms * 1e-3) / 1e12
        traffic, traffic_src, tensor_pct = ncu_traffic(args.workload)
        # the exact Eq. 2 work of the same calls (4 d flop per attended key and query row), from the
        # frame-level pattern the library reports (a_bits): what the computed tiles are an upper bound of
        frame_len = np.array([w.P] * w.T + ([w.n_text] if w.n_text else []), dtype=np.float64)
        useful_of = {}
        for s_e in sorted(set(steps_cycle)):
            ix_e = build(s_e)
            ab = ix_e.copy_host().a_bits
            ix_e.destroy()
            Tf = ab.shape[0]
            bits = ((ab[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1).reshape(Tf, -1)[:, :Tf]
            useful_of[s_e] = float((frame_len[:, None] * bits * frame_len[None, :]).sum()) * 4.0 * w.d * w.H * w.B
        # the timed steps cycle through steps_cycle: average the exact work over the same steps as kern_flops
        useful = sum(useful_of[steps_cycle[i % len(steps_cycle)]] for i in range(args.steps)) / args.steps
        line = {
            "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world,
            "unit_detail": UNIT_DETAIL,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms_step, 4),
            "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic (i.i.d. N(0,1) bf16, seeded Philox; stands in for Wan 2.1 latents)",
            "config": {"workload": args.workload, "T": w.T, "P": w.P, "N": w.N, "H": H_full, "d": w.d,
                       "B": w.B, "tile": w.tile, "window": w.W, "anchors": w.a,
                       "steps_cycled": steps_cycle, "nnz_mean": nnz_mean, "kernel": args.kernel, "layout": args.layout,
                       "l2": "inputs (3 x %.0f MB) exceed the 126 MB L2; no flush" % (q.numel() * 2 / 1e6),
                       "parallelism": ("heads of one call sharded over %d GPUs (%d heads on rank 0; no collective)" % (world, w.H)) if shard
                                      else ("replicas only (one independent call per GPU)" if world > 1 else "1 GPU")},
            "ms_per_attention_call": round(kern_ms, 4),
            "ms_per_attention_call_median": round(kern_median, 4), "ms_per_attention_call_min": round(kern_min, 4),
            "tflops_exact_eq2_work": round(useful / (kern_ms * 1e-3) / 1e12, 1),
            "computed_over_exact_work": round(kern_flops / useful, 4),
            "index_build_us": round(build_us, 1), "index_build_host_enqueue_us": round(build_host_us, 1),
            "index_build_static_scratch_us": None if static_us is None else round(static_us, 1),
            "pct_of_peak": {"sustained_kernel_vs_sustained_peak_%.1f" % pk["bf16_tflops_sustained"]: round(100 * achieved / pk["bf16_tflops_sustained"], 2),
                            "burst_kernel_vs_burst_peak_%.1f" % pk["bf16_tflops"]: round(100 * burst_tf / pk["bf16_tflops"], 2),
                            "sustained_kernel_vs_burst_peak": round(100 * achieved / pk["bf16_tflops"], 2),
                            "sustained_kernel_vs_nominal_2250": round(100 * achieved / 2250.0, 2)},
            "all_tiles": None if dense_ms is None else {
                "ms": round(dense_ms, 3), "ms_min": round(dense_all[0], 3), "ms_max": round(dense_all[-1], 3),
                "launches_timed": len(dense_all), "nnz": int(dense_nnz),
                "speedup_lvsa_vs_all_tiles": round(dense_ms / kern_ms, 3),
                "tflops": round(tile_flop(dense_cols) / (dense_ms * 1e-3) / 1e12, 1)},
            "frame_aligned_kv_tiles": fa_line,
            "quad_cluster_multicast": quad_line,
            "schedule": sched_line,
            "roofline": {"bound": "tensor", "achieved": round(achieved, 2), "peak": peak_sus,
                         "unit": "TFLOP/s", "frac": round(achieved / peak_sus, 4),
                         "frac_exact_eq2": round(useful / (kern_ms * 1e-3) / 1e12 / peak_sus, 4), "traffic": traffic,
                         "peak_source": pk["_source"] + " bf16 SUSTAINED peak: the kernel is timed inside the "
                                        "long step (event pair around each of the %d launches)" % args.steps,
                         "kernel": "lvsa_attn_sm100_pair_kernel", "flops_per_launch": kern_flops,
                         "ms_per_launch": round(kern_ms, 4),
                         "traffic_source": traffic_src,
                         "tensor_pipe_active_pct": tensor_pct,
                         "frac_sustained_time_vs_burst_peak": round(achieved / pk["bf16_tflops"], 4),
                         "burst": {"ms_per_launch": round(burst_ms, 4), "achieved": round(burst_tf, 2),
                                   "peak": pk["bf16_tflops"], "frac": round(burst_tf / pk["bf16_tflops"], 4),
                                   "how": "one launch after a 0.25 s idle gap, min of 5, vs the burst peak"}},
            "cpu_baseline": cpu,
            "e2e": None if e2e is None else {
                "value": round(e2e_value, 3), "unit": UNIT,
                "ms_per_step": round(e2e["ms"], 3), "calls_timed": e2e["calls"], "h2d_bytes_per_step": e2e["h2d"],
                "d2h_bytes_per_step": e2e["d2h"]},
            "gpu_launches": launches_per_step * args.steps,
            "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def cpu_baseline(w, q, k, v, step, n_rows, nthreads=0):
    """Times oracle O8 (fp64 Eq. 2) on a bounded sample of query rows of the same workload."""
    from oracle import lvsa_oracle as orc
    p = orc.pattern(w.T, w.W, w.a, step)
    rows = inputs.sample_rows(w, n_uniform=n_rows, n_edge=0, seed=1)[:n_rows]
    qa, ka, va = (inputs.to_oracle_array(x[0]) for x in (q, k, v))
    t0 = time.perf_counter()
    orc.attn_rows(qa, ka, va, w.T, w.P, p.A, rows, nthreads=nthreads)
    sec = time.perf_counter() - t0
    keys = sum(int(p.A[r // w.P].sum()) * w.P for r in rows)
    flops = 4.0 * w.d * w.H * keys
    cores = orc.num_threads() if nthreads == 0 else nthreads
    return {"value": flops / sec / 1e12, "unit": UNIT, "unit_detail": REF_UNIT_DETAIL, "cores": cores,
            "kind": "oracle", "seconds": round(sec, 2),
            "sample": f"{len(rows)} seeded query rows x {w.H} heads of {w.name} at step {step}",
            "extrapolated_ms_per_full_call": round(sec * 1e3 * w.N / len(rows), 1)}


def run_reference(args):
    """Reference arm = the oracle on the host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = inputs.WORKLOADS[args.workload]
    q, k, v = inputs.make_qkv(w, "cpu", torch.bfloat16)
    steps_cycle = list(w.steps) if w.steps else [0]
    rows_per_step = args.cpu_rows
    for i in range(args.warmup):
        cpu_baseline(w, q, k, v, steps_cycle[i % len(steps_cycle)], max(1, rows_per_step // 8))
    t0 = time.perf_counter()
    fl, last = 0.0, None
    for i in range(args.steps):
        last = cpu_baseline(w, q, k, v, steps_cycle[i % len(steps_cycle)], rows_per_step)
        fl += last["value"] * 1e12 * last["seconds"]
    sec = time.perf_counter() - t0
    val = fl / sec / 1e12
    ref_unit = UNIT
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": ref_unit, "unit_detail": REF_UNIT_DETAIL,
            "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3 / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic (same seeded tensors as the CUDA arm)",
            "config": {"workload": args.workload, "T": w.T, "P": w.P, "N": w.N, "H": w.H, "d": w.d,
                       "B": w.B, "tile": w.tile, "window": w.W, "anchors": w.a, "steps_cycled": steps_cycle},
            "cpu_baseline": {"value": val, "unit": ref_unit, "cores": last["cores"], "kind": "oracle",
                             "sample": f"each step: {last['sample']} (exact Eq. 2 flops, fp64)"},
            "e2e": {"value": val, "unit": ref_unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="wan1.3b_6x", choices=sorted(inputs.WORKLOADS))
    ap.add_argument("--cpu-rows", type=int, default=None, help="query rows in the oracle's timed sample")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-dense", action="store_true")
    ap.add_argument("--no-schedule", action="store_true")
    ap.add_argument("--kernel", default="default", choices=["default", "quad", "hybrid", "v0"],
                    help="attention kernel of the timed steps (default: the CTA-pair kernel); for A/B runs and ncu captures")
    ap.add_argument("--layout", default="nhd", choices=["nhd", "hnd"],
                    help="memory order of q, k, v, out: [B,N,H,d] (default, what a QKV projection yields) or [B,H,N,d]")
    ap.add_argument("--shard", default="none", choices=["none", "heads"],
                    help="none: every GPU runs a full replica of the call (weak scaling, the default the driver's SCALE run reads); "
                         "heads: the H heads of ONE call are dealt to the GPUs (strong scaling; PAPER.md:240's Ulysses shards)")
    ap.add_argument("--window", type=int, default=None, help="override W of the workload (sensitivity runs)")
    ap.add_argument("--anchors", type=int, default=None, help="override a = C - (2W+1) of the workload")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.cpu_rows is None:
        # ~15 s of oracle time on the GPU box's 16 host cores at the Wan 6x shape (5 s per 768 rows
        # measured there); scaled by heads and by the keys per row relative to Wan 6x
        wl = inputs.WORKLOADS[args.workload]
        args.cpu_rows = max(16, int(2304 * 12 / wl.H * min(4.0, 188760.0 / wl.N)))
        if args.impl == "reference":
            args.cpu_rows = max(8, args.cpu_rows // 4)
    if args.impl == "reference":
        run_reference(args)
    else:
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
        run_ours(args)


if __name__ == "__main__":
    main()
