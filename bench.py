#!/usr/bin/env python
"""bench.py -- SegPagedAttention on B200: useful TFLOP/s, roofline fraction, ms per layer.

A "step" is one pass of the whole hot path over one batch of synthetic
input, all through the C ABI (include/segpa.h):
    segpa_append_pages   (a1: scatter the batch's K/V rows, resident in HBM, into per-head pages)
    segpa_build_segments (a2-a5: page selection, translation, descriptor packing, tile schedule, H2D)
    segpa_attention_fwd  (a6-a8: fused attention [+ split-KV combine]; heads merged by layout)
Default workload: BASELINE.json configs[1] (Llama-3-8B-shaped layer).  `--config {1..5,4d,fig9-{decode,prefill}-{8,32,128}k}`
selects another one.  Multi-GPU: the path does not shard (BASELINE north_star: one GPU, no
collectives) -> N independent replicas, "scaling": "weak".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "segpa_useful_tflops"
UNIT = "TFLOP/s (useful: 4*D per attended (query, key, q-head) pair)"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return d, "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback (B200_PROFILING.md)"


def ncu_traffic(workload: str):
    """(DRAM bytes read + written by one attention launch, what that launch was) from the committed ncu --set full
    capture of this workload (profiles/r2_traffic.csv; commands in profiles/r2_ncu_full_attention_tc.md), or
    (None, None) when none was taken."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            f = line.split(",")
            if f[0] == workload:
                return int(f[-1]), ",".join(f[1:-1])
    except Exception:
        pass
    return None, None


def max_over_ranks(x: float, dist, device) -> float:
    """Replicas: the job's time is the slowest rank's (one all-reduce MAX; `dist` None = single process)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def get_workload(name: str):
    from paper_2606_06256_b200 import workloads as wl
    if name == "4d":
        return wl.config4(decode_only=True)
    if name.startswith("fig9-"):      # fig9-decode-8k, fig9-prefill-32k, ...: the paper's micro-benchmark shape
        _, mode, ctx = name.split("-")
        return wl.fig9(int(ctx.rstrip("k")) * 1024, mode)
    return wl.CONFIGS[int(name)]()


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.samples = []
        self.proc = None
        self.idx = gpu_index
        self.nvml = None          # (module, handle): NVML read from a thread every ~2 ms; nvidia-smi -lms is the fallback
        self.nv_samples = []      # (sm_mhz, reasons bitmask)
        self.nv_max = None
        self.stop_flag = False

    def _cuda_index_to_nvml(self, pynvml):
        """NVML enumerates all GPUs of the box, CUDA only the visible ones: map through CUDA_VISIBLE_DEVICES / UUID."""
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ent = [x.strip() for x in vis.split(",") if x.strip()]
            if self.idx < len(ent):
                e = ent[self.idx]
                if e.isdigit():
                    return pynvml.nvmlDeviceGetHandleByIndex(int(e))
                return pynvml.nvmlDeviceGetHandleByUUID(e.encode() if hasattr(e, "encode") else e)
        return pynvml.nvmlDeviceGetHandleByIndex(self.idx)

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = self._cuda_index_to_nvml(pynvml)
            self.nv_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
            self.nvml = (pynvml, h)
            self.th = threading.Thread(target=self._poll, daemon=True)
            self.th.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _poll(self):
        pynvml, h = self.nvml
        while not self.stop_flag:
            try:
                sm = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                try:
                    rs = int(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    rs = int(pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                self.nv_samples.append((sm, rs))
            except Exception:
                pass
            time.sleep(0.002)

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self):
        if self.nvml is not None:
            self.stop_flag = True
            self.th.join(timeout=1)
            pynvml, _ = self.nvml
            bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}
            sm = [a for a, _ in self.nv_samples]
            reasons = sorted(n for n, b in bits.items() if any(r & b for _, r in self.nv_samples))
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.nv_max, "reasons": reasons,
                    "samples": len(sm), "how": "NVML, every 2 ms during the timed region"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            f = [x.strip() for x in s.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "how": "nvidia-smi -lms 100"}


# ---------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the oracle as it stands on the host cores
# ---------------------------------------------------------------------------------------------
def oracle_sample(w, budget_rows: int, seed: int = 0, k_pool=None, v_pool=None, q=None):
    """Times the oracle on a bounded row sample of layer 0 of `w`. Returns (tflops, seconds, cores, pairs, desc)."""
    import torch  # noqa: F401
    import oracle
    from paper_2606_06256_b200 import workloads as wl
    if k_pool is None:
        k_pool, v_pool = wl.pool_values(w, "cpu")
        q = wl.q_values(w, 0, "cpu")
    rng = np.random.default_rng(seed)
    T = w.T[0]
    rows = np.sort(rng.choice(T, size=min(budget_rows, T), replace=False)).astype(np.int64)
    table, offs, kv_lens, index = wl.csr_page_tables(w, 0)
    segs = [(index[(s.kv_head, s.seq_id)], s.kv_head, s.head_class, s.window, s.n_sink, s.q_row_start, s.q_len)
            for s in w.layer_segments(0)]
    t0 = time.perf_counter()
    res = oracle.oracle_attention(Hq=w.Hq, Hkv=w.Hkv, D=w.D, P=w.P, k_pool=k_pool, v_pool=v_pool, page_table=table,
                                  pt_offsets=offs, kv_lens=kv_lens, segments=segs, q=q, T=T, scale=w.scale,
                                  row_subset=rows)
    dt = time.perf_counter() - t0
    flops = res.pairs * 4 * w.D
    desc = "%d uniformly sampled query rows of %d (all heads, layer 0) of %s; %d attended pairs" % (len(rows), T, w.name, res.pairs)
    return flops / dt / 1e12, dt, oracle.num_threads(), res.pairs, desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = get_workload(args.config or HEADLINE)
    from paper_2606_06256_b200 import workloads as wl
    k_pool, v_pool = wl.pool_values(w, "cpu")
    q = wl.q_values(w, 0, "cpu")
    rows = args.ref_rows if args.ref_rows > 0 else oracle_rows_for(w, args.ref_pairs)
    vals, times = [], []
    for i in range(args.warmup + args.steps):
        tf, dt, cores, pairs, desc = oracle_sample(w, rows, seed=i, k_pool=k_pool, v_pool=v_pool, q=q)
        if i >= args.warmup:
            vals.append(tf)
            times.append(dt)
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "note": "fp64 CPU oracle on a bounded row sample per step"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# context only: the same shapes as dense attention with an explicit mask ("Dense+mask")
# ---------------------------------------------------------------------------------------------
def dense_mask_ms(w, k_pool, v_pool, q, layer: int = 0, reps: int = 3):
    """Time of torch SDPA with a boolean attn_mask over gathered dense [1, H, L, D] K/V for one layer of `w`:
    per request, one call per group of KV heads sharing (class, window, q_len).  The gather is not timed.
    Library code, used as context for the paper's mask-penalty statement, not as a baseline to beat."""
    import torch
    import torch.nn.functional as F
    from paper_2606_06256_b200 import workloads as wl
    sm = w.stream_map()
    groups = {}
    for s in w.layer_segments(layer):
        groups.setdefault((s.seq_id, s.head_class, s.window if s.head_class == wl.LOCAL else 0, s.q_row_start, s.q_len), []).append(s.kv_head)
    calls = []
    for (seq, cls, W, q0, ql), heads in groups.items():
        L = sm[(layer, heads[0], seq)].kv_len
        kd = torch.stack([wl.stream_rows(k_pool, sm[(layer, h, seq)], w.P) for h in heads])      # [n_kvh, L, D]
        vd = torch.stack([wl.stream_rows(v_pool, sm[(layer, h, seq)], w.P) for h in heads])
        kd = kd.repeat_interleave(w.G, dim=0).unsqueeze(0)
        vd = vd.repeat_interleave(w.G, dim=0).unsqueeze(0)
        qh = torch.cat([torch.arange(h * w.G, (h + 1) * w.G) for h in heads]).to(q.device)
        qd = q[q0:q0 + ql][:, qh].permute(1, 0, 2).unsqueeze(0).contiguous()                      # [1, Hg, ql, D]
        i = torch.arange(L - ql, L, device=q.device).unsqueeze(1)
        j = torch.arange(L, device=q.device).unsqueeze(0)
        mask = (j <= i) if cls == wl.GLOBAL else ((j <= i) & (j > i - W))
        calls.append((qd, kd, vd, mask))
    def run():
        for qd, kd, vd, mask in calls:
            F.scaled_dot_product_attention(qd, kd, vd, attn_mask=mask, scale=w.scale)
    run()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        run()
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1) / reps, len(calls)


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
PER_CONFIG = ["2", "3", "4", "4d", "fig9-decode-128k"]      # measured beside the headline workload in the default run
HEADLINE = "5"                                              # BASELINE.json configs[4]: the largest single-GPU job


def is_decode_shaped(name: str) -> bool:
    return name == "4d" or name.startswith("fig9-decode")


def measure(name: str, steps: int, warmup: int, dev, local_rank: int, world: int, dist, peaks, peaks_src, tiles: int,
            full: bool, cpu_rows_pairs: float = 0.0, dense_mask: bool = False):
    """One workload through the C ABI: `steps` steps enqueued back to back inside one CUDA-event bracket.  Returns the
    measurement record; `full` adds the isolated-step latency, the e2e (host buffers) leg and the oracle timing."""
    import torch
    from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl

    w = get_workload(name)
    k_pool, v_pool = wl.pool_values(w, dev)
    qs = [wl.q_values(w, l, dev) for l in range(w.num_layers)]
    outs = [torch.empty_like(q) for q in qs]
    lses = [torch.empty((w.Hq, w.T[l]), dtype=torch.float32, device=dev) for l in range(w.num_layers)]
    # the batch's K/V rows, resident in HBM (what the QKV projections would have produced); the
    # marshalled request array is prepared once (the same batch is stored every step)
    append_reqs = H.append_requests(w, k_pool, v_pool)
    batch = B.AppendBatch(append_reqs)
    cache = H.create_cache(w, local_rank, tiles_per_item=tiles)
    stream = torch.cuda.current_stream()
    flush_buf = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)
    useful = sum(wl.useful_flops(w, l) for l in range(w.num_layers))
    seg_objs = []
    seg_batches = [B.SegmentBatch(H.segment_reqs(w, l)) for l in range(w.num_layers)]

    def append_all(b):
        """a1: drop the previous batch's streams and segment objects, store this batch (one scatter launch)"""
        for s in seg_objs:
            B.segpa_free_segments(cache, s)
        seg_objs.clear()
        B.segpa_clear_streams(cache)
        B.segpa_append_pages_batch(cache, b, stream=stream)
        return 1

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step():
        """one pass of the hot path, enqueued on `stream` with no host synchronisation; returns the CUDA
        events around each layer's segpa_attention_fwd and the number of our kernels launched"""
        fa, fb = [], []
        n = append_all(batch)
        for l in range(w.num_layers):
            segs = B.segpa_build_segments(cache, l, seg_batches[l], stream=stream)
            seg_objs.append(segs)
            a, b = ev(), ev()
            a.record(stream)
            B.segpa_attention_fwd(cache, segs, qs[l], w.scale, outs[l], lses[l], stream=stream)
            b.record(stream)
            fa.append(a)
            fb.append(b)
            n += B.segpa_last_launch_count(cache)
        return fa, fb, n

    for _ in range(warmup):
        step()
        flush_buf.fill_(1)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    # The K timed steps are enqueued back to back inside ONE CUDA-event bracket (E0 .. E1): the host plans
    # step k+1 (build_segments) while the device runs step k, as a serving loop does.  L2 is flushed on the
    # stream before every step; each flush has its own events.  Two figures come out of the bracket:
    #   ms_per_step_incl_flush = (E1 - E0) / K                        everything the device did, flushes included
    #   ms_per_step            = max((E1 - E0 - flushes) / K, host enqueue time per step)
    # `value` uses the second: the flush is the harness's, not the path's, but the host's planning of step k+1
    # runs under it, so the step is never credited with less than the host needed to enqueue it.
    E0, E1 = ev(), ev()
    flushes, fwd_ev = [], []
    host_s = 0.0
    launches = 0
    wall0 = time.perf_counter()
    E0.record(stream)
    for _ in range(steps):
        f0, f1 = ev(), ev()
        f0.record(stream)
        flush_buf.fill_(1)                      # L2 flush between timed iterations
        f1.record(stream)
        flushes.append((f0, f1))
        h0 = time.perf_counter()
        fa, fb, n = step()
        host_s += time.perf_counter() - h0
        fwd_ev.append((fa, fb))
        launches += n
    E1.record(stream)
    E1.synchronize()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    flush_ms = float(sum(f0.elapsed_time(f1) for f0, f1 in flushes))
    bracket_ms = max_over_ranks(E0.elapsed_time(E1), dist, dev)
    host_ms = max_over_ranks(1e3 * host_s / steps, dist, dev)
    dev_ms = max_over_ranks((E0.elapsed_time(E1) - flush_ms) / steps, dist, dev)
    ms_per_step = max(dev_ms, host_ms)
    value = world * useful / (ms_per_step * 1e-3) / 1e12
    fwd_ms = [sum(a.elapsed_time(b) for a, b in zip(fa, fb)) for fa, fb in fwd_ev]
    fwd_mean = float(np.mean(fwd_ms))
    layer_ms = [float(np.mean([fa[l].elapsed_time(fb[l]) for fa, fb in fwd_ev])) for l in range(w.num_layers)]

    # ---- plan statistics / algorithmic bytes for the roofline
    st0 = None
    alg_bytes = 0
    for l in range(w.num_layers):
        sg = H.build_layer(cache, w, l)
        st = B.segpa_segments_stats(sg)
        B.segpa_free_segments(cache, sg)
        st0 = st0 or st
        cov_rows = sum(s.q_len * w.G for s in w.layer_segments(l))
        alg_bytes += st["visible_kv_tokens"] * w.D * 2 * 2 + cov_rows * w.D * 2 * 2 + cov_rows * 4
    torch.cuda.synchronize()
    # a kernel timed inside a long step (tens of ms back to back: the device sits at its power cap) is held against
    # the sustained bf16 figure, a short one against the burst figure (B200_PROFILING.md); both fractions are printed
    long_step = fwd_mean >= 20.0
    if is_decode_shaped(name):
        roof = {"bound": "hbm", "achieved": alg_bytes / (fwd_mean * 1e-3) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s"}
        roof["frac"] = roof["achieved"] / roof["peak"]
        roof["peak_source"] = peaks_src
    else:
        ach = useful / (fwd_mean * 1e-3) / 1e12
        pk = peaks["bf16_tflops_sustained"] if long_step else peaks["bf16_tflops"]
        roof = {"bound": "tensor", "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": ach / pk,
                "frac_of_burst": ach / peaks["bf16_tflops"], "frac_of_sustained": ach / peaks["bf16_tflops_sustained"],
                "peak_source": peaks_src + (", sustained figure (kernel timed inside a %.0f ms step)" % fwd_mean if long_step else ", burst figure")}
    roof["traffic"], roof["traffic_capture"] = ncu_traffic(w.name)
    roof["kernel"] = "attention_tc_kernel (+ combine_kernel where the plan splits KV) = segpa_attention_fwd, mean over %d steps x %d layers, CUDA events on the launching stream" % (steps, w.num_layers)
    roof["algorithmic_bytes"] = alg_bytes
    roof["useful_flops"] = useful

    rec = {"workload": w.name, "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step,
           "ms_per_step_incl_flush": bracket_ms / steps, "value": value, "fwd_ms": fwd_mean,
           "us_per_layer": 1e3 * fwd_mean / w.num_layers, "useful_tflops": useful / (fwd_mean * 1e-3) / 1e12,
           "roofline": roof, "clocks": clocks, "gpu_launches": int(launches), "wall_s_timed_region": wall,
           "plan": {k: st0[k] for k in ("n_tiles", "n_items", "n_split_tiles", "kv_blocks", "workspace_bytes")},
           "shape": {"Hq": w.Hq, "Hkv": w.Hkv, "D": w.D, "page_size": w.P, "layers": w.num_layers, "q_rows": int(sum(w.T)),
                     "segments": len(w.segments)},
           "timing": {"flush_ms_total": flush_ms, "device_ms_per_step_excl_flush": dev_ms, "host_enqueue_ms_per_step": host_ms,
                      "value_uses": "max(device time excluding the L2 flushes, host enqueue time) per step"}}
    if w.num_layers > 1:
        rec["layer_ms"] = {"min": min(layer_ms), "max": max(layer_ms), "mean": float(np.mean(layer_ms))}

    if full:
        # ---- the same step run alone: flush, device idle, then one step with the host waiting for its end
        # (planning and kernels in series: the latency of a single isolated step, not the throughput)
        iso_ms = []
        for _ in range(max(2, min(steps, 5))):
            flush_buf.fill_(1)
            torch.cuda.synchronize()
            e0, e1 = ev(), ev()
            e0.record(stream)
            step()
            e1.record(stream)
            e1.synchronize()
            iso_ms.append(e0.elapsed_time(e1))
        torch.cuda.synchronize()
        rec["timing"]["isolated_step_ms"] = float(np.mean(iso_ms))

        # ---- e2e, everything through the C ABI with HOST buffers (pinned): the step's K/V rows go up inside
        # segpa_append_pages_batch (src_is_host), Q / out / LSE through segpa_attention_fwd_host (row-chunked:
        # H2D, kernels and D2H overlap)
        h_reqs, keep = [], []
        for (layer, kvh, seq, kr, vr, n, ids) in append_reqs:
            if kr is None:
                h_reqs.append((layer, kvh, seq, None, None, n, ids))
            else:
                a, b = kr.cpu().pin_memory(), vr.cpu().pin_memory()
                keep.append((a, b))
                h_reqs.append((layer, kvh, seq, a, b, n, ids))
        h_batch = B.AppendBatch(h_reqs)
        h_q = [q.cpu().pin_memory() for q in qs]
        h_out = [torch.empty_like(q).pin_memory() for q in h_q]
        h_lse = [torch.empty((w.Hq, w.T[l]), dtype=torch.float32).pin_memory() for l in range(w.num_layers)]
        h2d = sum(a.numel() * 2 * 2 for a, _ in keep) + sum(q.numel() * 2 for q in h_q)
        d2h = sum(o.numel() * 2 for o in h_out) + sum(x.numel() * 4 for x in h_lse)

        def e2e_step():
            append_all(h_batch)
            for l in range(w.num_layers):
                segs = B.segpa_build_segments(cache, l, seg_batches[l], stream=stream)
                seg_objs.append(segs)
                # (several layers: asynchronous calls, so that layer l+1's rows go up while layer l's results come down)
                B.segpa_attention_fwd_host(cache, segs, h_q[l], w.scale, h_out[l], h_lse[l], stream=stream, wait=w.num_layers == 1)
            B.segpa_host_wait(cache)          # every layer's out / lse rows are in host memory
            torch.cuda.synchronize()

        e2e_step()
        # the host-buffer results of the warm-up step against the device entry point (first and last layer, bit for bit;
        # pairs no segment covers are zeros on both sides): an e2e figure from wrong results would be worthless
        for l in sorted({0, w.num_layers - 1}):
            chk = torch.zeros_like(qs[l])
            chk_lse = torch.zeros((w.Hq, w.T[l]), dtype=torch.float32, device=dev)
            B.segpa_attention_fwd(cache, seg_objs[l - w.num_layers], qs[l], w.scale, chk, chk_lse, stream=stream)
            torch.cuda.synchronize()
            if not (torch.equal(chk.cpu(), h_out[l]) and torch.equal(chk_lse.cpu(), h_lse[l])):
                raise RuntimeError("e2e: host-buffer results of layer %d differ from the device entry point" % l)
            del chk, chk_lse
        n_e2e = max(2, min(steps, 5))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        e2e_s = max_over_ranks((time.perf_counter() - t0) / n_e2e, dist, dev)
        pcie = max(h2d, d2h) / (e2e_s) / 1e9
        rec["e2e"] = {"value": world * useful / e2e_s / 1e12, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                      "ms_per_step": 1e3 * e2e_s, "steps": n_e2e,
                      "how": "segpa_append_pages_batch(src_is_host) + (segpa_build_segments + segpa_attention_fwd_host_async) per layer + segpa_host_wait, pinned host buffers, wall clock around whole steps",
                      "larger_direction_gbs": pcie}
        del h_q, h_out, h_lse, keep, h_batch

    if dense_mask:
        try:
            dm, ncalls = dense_mask_ms(w, k_pool, v_pool, qs[0])
            rec["dense_mask_context"] = {"ms_per_layer": dm, "x_slower_than_segpa_fwd": dm / (fwd_mean / w.num_layers),
                                         "how": "torch SDPA, boolean attn_mask, dense gathered K/V, %d calls (one per request x head class), layer 0" % ncalls,
                                         "note": "context for the paper's 4.9-7.6x mask penalty (PAPER.md:19; its shapes are unknown), not a like-for-like number"}
        except Exception as ex:  # library path, context only
            rec["dense_mask_context"] = {"error": repr(ex)[:200]}
    if cpu_rows_pairs > 0:
        rows = oracle_rows_for(w, cpu_rows_pairs)
        tf, dt, cores, pairs, desc = oracle_sample(w, rows, seed=0, k_pool=k_pool.cpu(), v_pool=v_pool.cpu(), q=qs[0].cpu())
        rec["cpu_baseline"] = {"value": tf, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc + "; %.1f s" % dt}
    for s in seg_objs:
        B.segpa_free_segments(cache, s)
    B.segpa_destroy(cache)
    del k_pool, v_pool, qs, outs, lses, batch, append_reqs, flush_buf
    torch.cuda.empty_cache()
    return rec


def oracle_rows_for(w, pairs_budget: float) -> int:
    """Rows of layer 0 whose oracle evaluation costs about `pairs_budget` attended (query, key, q-head) pairs."""
    from paper_2606_06256_b200 import workloads as wl
    per_row = wl.useful_flops(w, 0) / (4.0 * w.D) / max(1, w.T[0])
    return int(min(w.T[0], max(16, pairs_budget / max(per_row, 1.0))))


def run_ours(args):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=dev)
    peaks, peaks_src = load_peaks()
    name = args.config or HEADLINE
    head = measure(name, args.steps, args.warmup, dev, local_rank, world, dist, peaks, peaks_src, args.tiles, full=True,
                   cpu_rows_pairs=(0.0 if (args.no_cpu_baseline or rank != 0 or world != 1) else args.cpu_pairs),
                   dense_mask=(rank == 0 and world == 1 and args.dense_mask == "on"))
    line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": head["ms_per_step"], "ms_per_step_incl_flush": head["ms_per_step_incl_flush"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": dict(head["shape"], workload=head["workload"], l2_flush_between_steps=True,
                           step="append_pages_batch + (build_segments + attention_fwd) per layer", tiles_per_item=args.tiles,
                           replicas=world),
            "fwd_ms_per_step": head["fwd_ms"], "us_per_layer": head["us_per_layer"],
            "pct_of_bf16_peak": 100.0 * head["useful_tflops"] / peaks["bf16_tflops"],
            "plan": head["plan"], "roofline": head["roofline"], "clocks": head["clocks"], "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "wall_s_timed_region": head["wall_s_timed_region"],
            "timing": dict(head["timing"], how="one CUDA-event bracket over the K steps enqueued back to back (host plans step k+1 under the "
                                              "kernels of step k); the on-stream L2 flushes before each step are timed with their own events")}
    for k in ("layer_ms", "dense_mask_context", "cpu_baseline"):
        if k in head:
            line[k] = head[k]
    # the other workloads, each with its own clocks record (default run only: one GPU, no --config)
    if args.config is None and world == 1 and not args.no_per_config:
        per = [{k: head[k] for k in ("workload", "steps", "warmup", "ms_per_step", "ms_per_step_incl_flush", "value", "fwd_ms", "us_per_layer",
                                     "useful_tflops", "roofline", "clocks", "gpu_launches")}]
        for c in PER_CONFIG:
            r = measure(c, min(args.steps, 20), 3, dev, local_rank, world, None, peaks, peaks_src, args.tiles, full=False,
                        dense_mask=(c == "2" and args.dense_mask != "off"))
            ent = {k: r[k] for k in ("workload", "steps", "warmup", "ms_per_step", "ms_per_step_incl_flush", "value", "fwd_ms", "us_per_layer",
                                     "useful_tflops", "roofline", "clocks", "gpu_launches", "timing")}
            if "dense_mask_context" in r:
                ent["dense_mask_context"] = r["dense_mask_context"]
            per.append(ent)
            line["gpu_launches"] += r["gpu_launches"]
        line["per_config"] = per
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_rope(args):
    """`--config rope`: the step before the hot path (RoPEAlign) on its own:
    K of every stream of cfg3 (8 KV heads x 65536 tokens, D 128) rotated in place, one call per stream.
    HBM-bound: algorithmic bytes = tokens x D x 2 B read + the same written."""
    import torch
    from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = wl.config3()
    peaks, peaks_src = load_peaks()
    k_pool, v_pool = wl.pool_values(w, dev)
    cache = H.create_cache(w, 0)
    H.append_workload(cache, w, k_pool, v_pool)
    stream = torch.cuda.current_stream()
    flush_buf = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)
    tokens = sum(s.kv_len for s in w.streams)
    alg_bytes = tokens * w.D * 2 * 2

    # the 12 reused chunks of every head, each moved by its own delta: one batched call, one launch
    chunks = w.notes["chunks"]
    reqs = []
    for s in w.streams:
        t0 = 0
        for ci, n in enumerate(chunks):
            reqs.append((s.layer, s.kv_head, s.seq_id, t0, n, 1000 + 4096 * ci))
            t0 += n
    tokens = sum(r[4] for r in reqs)
    alg_bytes = tokens * w.D * 2 * 2

    batch = B.RopeBatch(reqs)

    def step():
        B.segpa_rope_align_batch(cache, batch, 10000.0, stream=stream)

    for _ in range(max(3, args.warmup)):
        step()
    ms = []
    for _ in range(args.steps):
        flush_buf.fill_(1)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        step()
        e1.record(stream)
        e1.synchronize()
        ms.append(e0.elapsed_time(e1))
    t = float(np.mean(ms))
    gbs = alg_bytes / (t * 1e-3) / 1e9
    B.segpa_destroy(cache)
    print(json.dumps({"metric": "rope_align_gbs", "value": gbs, "unit": "GB/s (K bytes read + written)", "n_gpus": 1,
                      "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": t, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "bf16 in/out, fp32 rotation", "data": "synthetic",
                      "config": {"workload": "rope_align over the reused chunks of cfg3_llama70b_64k (%d heads x %d chunks, %d tokens)" % (len(w.streams), len(chunks), tokens),
                                 "l2_flush_between_steps": True},
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                   "frac": gbs / peaks["hbm_gbs"], "traffic": None, "algorithmic_bytes": alg_bytes,
                                   "peak_source": peaks_src, "kernel": "rope_align_kernel, 1 launch per step (%d chunks)" % len(reqs)},
                      "gpu_launches": args.steps}))


def run_mass(args):
    """`--config mass`: the step after the hot path (attention mass + salient-token selection, PAPER.md:198, 296;
    SURVEY 8(f) NEXT #4) on cfg2.  The contraction is S^T = K Q^T only: 2*D FLOPs per attended (query, key, q-head)."""
    import torch
    from paper_2606_06256_b200 import binding as B, harness as H, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    w = wl.config2()
    peaks, peaks_src = load_peaks()
    k_pool, v_pool = wl.pool_values(w, dev)
    cache = H.create_cache(w, 0)
    H.append_workload(cache, w, k_pool, v_pool)
    segs = H.build_layer(cache, w, 0)
    q = wl.q_values(w, 0, dev)
    out = torch.empty_like(q)
    lse = torch.empty((w.Hq, w.T[0]), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()
    B.segpa_attention_fwd(cache, segs, q, w.scale, out, lse, stream=stream)
    offs = B.segpa_segments_mass_layout(segs)
    mass = torch.zeros((int(offs[-1]),), dtype=torch.float32, device=dev)
    sel = torch.zeros((int(offs[-1]),), dtype=torch.uint8, device=dev)
    cnt = torch.zeros((len(offs) - 1,), dtype=torch.int32, device=dev)
    flush_buf = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=dev)
    flops = wl.useful_flops(w, 0) // 2
    ms_mass, ms_sel = [], []
    for i in range(max(3, args.warmup) + args.steps):
        flush_buf.fill_(1)
        torch.cuda.synchronize()
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        B.segpa_attention_mass(cache, segs, q, w.scale, lse, mass, stream=stream)
        e1.record(stream)
        B.segpa_mass_select(cache, segs, mass, 0.7, sel, cnt, stream=stream)
        e2.record(stream)
        e2.synchronize()
        if i >= max(3, args.warmup):
            ms_mass.append(e0.elapsed_time(e1))
            ms_sel.append(e1.elapsed_time(e2))
    t, ts = float(np.mean(ms_mass)), float(np.mean(ms_sel))
    tf = flops / (t * 1e-3) / 1e12
    B.segpa_destroy(cache)
    print(json.dumps({"metric": "attention_mass_useful_tflops", "value": tf, "unit": "TFLOP/s (useful: 2*D per attended (query, key, q-head) pair)",
                      "n_gpus": 1, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": t, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                      "config": {"workload": "attention mass over " + w.name, "l2_flush_between_steps": True, "select_ms": ts, "tau": 0.7},
                      "roofline": {"bound": "tensor", "achieved": tf, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s", "frac": tf / peaks["bf16_tflops"],
                                   "traffic": None, "useful_flops": flops, "peak_source": peaks_src,
                                   "kernel": "attention_mass_kernel; MUFU co-limited: 1024 ex2 cycles per 512 MMA cycles per tile"},
                      "gpu_launches": 2 * args.steps}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=None,
                    help="workload: 1..5, 4d, fig9-{decode,prefill}-{8,32,128}k, rope, mass.  Default: BASELINE.json configs[4] "
                         "(cfg5, the whole 28-layer stack) as the headline, plus a per_config list over cfg2, cfg3, cfg4, 4d and fig9-decode-128k")
    ap.add_argument("--tiles", type=int, default=2)
    ap.add_argument("--cpu-pairs", type=float, default=1.2e9, help="attended pairs in the cpu_baseline oracle sample (about 15 s of CPU)")
    ap.add_argument("--ref-rows", type=int, default=0, help="rows per step of the --impl reference oracle sample (0: from --ref-pairs)")
    ap.add_argument("--ref-pairs", type=float, default=8e7, help="attended pairs per step of the --impl reference oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="default run: skip the per_config list")
    ap.add_argument("--dense-mask", default="auto", choices=["auto", "on", "off"],
                    help="also time dense attention with an explicit mask (context; auto = for cfg2 in the per_config list)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.config == "rope" and args.impl == "ours":
        run_rope(args)
    elif args.config == "mass" and args.impl == "ours":
        run_mass(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
