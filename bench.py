#!/usr/bin/env python
"""bench.py -- times the fused sparse decode step (all hot-path rows a1..a5) on synthetic, seeded
decode workloads shaped like BASELINE.json's configs, and prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4|C3|C2|C5|C1] [--impl reference]

metric : sparse decode step time in microseconds (lower is better), with the achieved HBM GB/s and
         the fraction of the bytes roofline (summary bytes + selected-KV bytes + Q/O bytes).
value  : device-timed (CUDA events on the launching stream, L2 flushed between steps), inputs resident.
e2e    : the same step through vx_sparse_decode_step_host: pinned HOST q / page table / budgets in,
         HOST out / lse back, copies inside the timed region.
N > 1  : one process per GPU (torchrun), every rank runs its own seeded copy of the workload
         (requests shard with no exchange step: "weak" scaling, no collective on the data path);
         time = max over ranks.
--impl reference : the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sparse_decode_step_us"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json "about 8 TB/s"
FALLBACK_HBM_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="C4", help="workload: C1..C5 (default C4, the MLA config the north star's >= 70 %% target "
                    "names and the one furthest from it; C3 is the other target config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--also", default="C3,C2,C5,C1", help="further configs, each a full record (step, stages, roofline, e2e, "
                    "clocks) under 'also'")
    ap.add_argument("--also-steps", type=int, default=50)
    ap.add_argument("--kv-dtype", default="same", choices=["same", "e4m3", "e5m2"],
                    help="storage of the KV cache and the summaries: the config's dtype (default, the north star) or fp8 codes "
                         "with per-tensor scales (PAPER.md:200, :520; the bytes roofline is recomputed: summary and KV bytes halve)")
    ap.add_argument("--mla-step", default="auto", choices=["auto", "chained", "fused", "flat"],
                    help="schedule of the MLA step (VX_OPT_MLA_STEP); auto = the library's choice")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--summary", default="envelope", choices=["envelope", "centroid"],
                    help="page summary / score flow: Quest envelope (default, the north star) or block top-k centroid")
    ap.add_argument("--agg", default="sum", choices=["sum", "max"],
                    help="head-group aggregation of the envelope score: sum (default, the north star) or max_h (PAPER.md:556)")
    ap.add_argument("--topk-approx", type=float, default=0.0, metavar="RATIO",
                    help="select with vx_topk_pages_approx at this tolerate_ratio (PAPER.md:196; lossy, recall@k >= "
                         "1 - RATIO).  Default 0: the exact selection, the north star's path")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(cfg, stage):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of the stage's kernel, source) from the committed
    `ncu --set full` captures of this round (profiles/r2_traffic.csv: one row per config and kernel, each naming the
    raw export it was read from and the git revision of the library that was profiled), or (None, None)."""
    kernels = {"page_score": ("score_kernel", "score_mla_max_kernel"),
               "sparse_paged_decode": ("decode_gqa_mma_kernel", "decode_mla_kernel", "decode_generic_kernel")}[stage]
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None, None
    import csv
    for row in csv.DictReader(open(path)):
        if row["config"] == cfg and row["kernel"] in kernels:
            return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]), f"profiles/{row['source']} (library at {row['lib_rev']})"
    return None, None


def algorithmic_bytes(w, sel_count=None, summary="envelope"):
    """Bytes roofline of one step: every summary row once, every selected
    page's K and V tokens once, Q in and O out.  Page table / scores / partials are not counted."""
    import torch
    s = w.spec
    esz = 2 if s.dtype == "bf16" else 4                # q and out
    kv_esz = 1 if getattr(s, "kv_dtype", "") else esz   # K, V and the summaries (fp8 KV cache: one byte)
    b = s.page_size
    n = w.seq_lens.cpu().long()
    P = (n + b - 1) // b
    summary = int(P.sum()) * s.num_kv_heads * (1 if summary == "centroid" else 2) * s.qk_dim * kv_esz
    k = torch.minimum(w.budget.cpu().long(), P)
    tokens = (k - 1) * b + (n - (P - 1) * b)          # the partial last page is always selected (n_local >= 1)
    per_tok = (s.qk_dim if s.kv_shared else s.qk_dim + s.v_dim) * kv_esz
    kv = int(tokens.sum()) * s.num_kv_heads * per_tok
    qo = s.batch * s.num_q_heads * (s.qk_dim + s.v_dim) * esz
    return dict(summary=summary, kv=kv, qo=qo, total=summary + kv + qo)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (NVML; ~20 ms period)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None
        self.ready = threading.Event()

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20,
                     "hw_thermal_slowdown": 0x40, "hw_power_brake": 0x80}
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.reasons |= {k for k, bit in names.items() if r & bit}
                self.ready.set()
                time.sleep(0.001)
        except Exception as e:  # NVML unavailable: report that rather than guessing
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")
        self.ready.set()

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


class Runner:
    """One workload resident on one GPU: context, pools, summaries, outputs, L2 flush buffer."""

    def __init__(self, cfg, device, seed_offset=0, summary="envelope", topk_approx=0.0, agg="sum", mla_step="auto",
                 kv_dtype="same"):
        import torch
        import paper_2606_06453_b200 as vx
        from paper_2606_06453_b200.workloads import make_workload, with_fp8
        self.torch, self.vx = torch, vx
        spec = cfg if kv_dtype == "same" else with_fp8(cfg, kv_dtype)
        self.w = w = make_workload(spec, device=device, seed_offset=seed_offset)
        kind = vx.binding.VX_SUMMARY_CENTROID if summary == "centroid" else vx.binding.VX_SUMMARY_ENVELOPE
        self.summary_name = summary
        self.ctx = vx.context_for(w, summary_kind=kind, agg=vx.binding.VX_AGG_MAX if agg == "max" else vx.binding.VX_AGG_SUM)
        if w.spec.kv_shared:
            self.ctx.set_option(vx.VX_OPT_MLA_STEP, {"auto": vx.VX_MLA_STEP_AUTO, "chained": vx.VX_MLA_STEP_CHAINED,
                                                     "fused": vx.VX_MLA_STEP_FUSED, "flat": vx.VX_MLA_STEP_FLAT}[mla_step])
        self.tau = float(topk_approx)
        self.step_flags = vx.VX_STEP_UPDATE_SUMMARY | (vx.VX_STEP_APPROX_TOPK if self.tau > 0 else 0)
        self.ctx.set_topk_approx(self.tau, 20260604)
        self.pool, self.pt = vx.tables_for(w)
        self.summary = vx.alloc_summary(w, kind)
        self.ctx.page_summary_update(self.pool, self.pt, self.summary, first_new_pos=torch.zeros_like(w.seq_lens))
        s = w.spec
        self.out = torch.empty(s.batch, s.num_q_heads, s.v_dim, dtype=w.q.dtype, device=device)
        self.lse = torch.empty(s.batch, s.num_q_heads, dtype=torch.float32, device=device)
        self.scores = torch.empty(s.num_kv_heads, w.total_pages, dtype=torch.float32, device=device)
        self.sel_phys = torch.empty(s.batch, s.num_kv_heads, w.max_budget, dtype=torch.int32, device=device)
        self.sel_logical = torch.empty_like(self.sel_phys)
        self.sel_count = torch.empty(s.batch, s.num_kv_heads, dtype=torch.int32, device=device)
        self.flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2
        self.flush_rd = torch.zeros(64 << 20, dtype=torch.int32, device=device)  # 256 MiB read sweep
        pin = lambda t: t.cpu().contiguous().pin_memory()
        self.h = dict(q=pin(w.q), indptr=pin(w.page_indptr), indices=pin(w.page_indices), seq=pin(w.seq_lens),
                      budget=pin(w.budget), out=torch.empty_like(self.out, device="cpu").pin_memory(),
                      lse=torch.empty_like(self.lse, device="cpu").pin_memory())
        torch.cuda.synchronize()

    # the stages, each through the C ABI
    def step(self):
        self.ctx.sparse_decode_step(self.w.q, self.pool, self.summary, self.pt, self.w.budget, self.w.max_budget,
                                    self.out, self.lse, self.sel_phys, self.sel_logical, self.sel_count,
                                    flags=self.step_flags)

    def step_host(self):
        h = self.h
        self.ctx.sparse_decode_step_host(h["q"], self.pool, self.summary, h["indptr"], h["indices"], h["seq"],
                                         h["budget"], self.w.max_budget, h["out"], h["lse"],
                                         flags=self.step_flags)

    def stage_summary(self):
        self.ctx.page_summary_update(self.pool, self.pt, self.summary, first_new_pos=None)

    def stage_score(self):
        self.ctx.page_score(self.w.q, self.summary, self.pt, self.scores)

    def stage_topk(self):
        self.ctx.topk_pages_approx(self.scores, self.pt, self.w.budget, self.w.max_budget, self.tau, 20260604,
                                   self.sel_phys, self.sel_logical, self.sel_count)   # ratio 0 = vx_topk_pages

    def stage_decode(self):
        self.ctx.sparse_paged_decode(self.w.q, self.pool, self.pt, self.sel_phys, self.sel_logical, self.sel_count,
                                     self.w.max_budget, self.out, self.lse)

    def flush_l2(self):
        """Cold L2 for the next step: a 512 MiB write sweep, then a 256 MiB read sweep so the L2 is left
        full of CLEAN foreign lines (a write-only flush leaves ~126 MB of dirty lines whose write-back
        the timed step would pay for).  Outside the timed events.  DESIGN.md section 8.1."""
        self.flush.zero_()
        self.flush_rd.max()

    def time_device(self, fn, steps, warmup):
        """per-step CUDA-event times (ms) on the current stream, L2 flushed before every step."""
        torch = self.torch
        for _ in range(warmup):
            self.flush_l2()
            fn()
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            self.flush_l2()
            a.record()
            fn()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def time_host(self, fn, steps, warmup):
        """wall-clock per step (ms) of a synchronous host-buffer call, L2 flushed before every step."""
        torch = self.torch
        out = []
        for it in range(warmup + steps):
            self.flush_l2()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            t1 = time.perf_counter()
            if it >= warmup:
                out.append((t1 - t0) * 1e3)
        return out


def oracle_prepare(cfg, n_requests, seed_offset=0, device="cpu", workload=None, summary="envelope", agg="sum"):
    """The oracle (as it stands) on the first n_requests requests of the workload: gathers their pages to the host ONCE and
    returns (run, requests in sample, batch, threads), run() = one timed pass (score + top-k + attention) in seconds."""
    from oracle import vx_oracle as vo
    from paper_2606_06453_b200.workloads import make_workload, subproblem
    from oracle.workload_io import to_oracle
    w = workload if workload is not None else make_workload(cfg, device=device, seed_offset=seed_offset)
    n_requests = min(n_requests, w.spec.batch)
    sub = subproblem(w, range(n_requests))
    q, pool, pt = to_oracle(sub)
    s = sub.spec
    build = vo.page_centroid if summary == "centroid" else vo.page_summary
    summ = build(pool, pt, s.num_kv_heads, s.qk_dim)                    # built outside the timed step
    page = pt.page_size                                                 # (the block size when blocks are finer than the page)

    def run():
        t0 = time.perf_counter()
        vo.decode_step(q, pool, pt, vo.as_np(sub.budget), sub.max_budget, s.num_q_heads, s.num_kv_heads, s.qk_dim,
                       s.v_dim, s.sm_scale, s.n_sink, s.n_local, agg=vo.AGG_MAX if agg == "max" else vo.AGG_SUM, summary=summ,
                       kind=summary)
        return time.perf_counter() - t0

    return run, n_requests, w.spec.batch, vo.num_threads()


def oracle_sample_time(cfg, n_requests, seed_offset=0, device="cpu", workload=None, summary="envelope", agg="sum", passes=3):
    """one untimed warm-up pass, then the MEDIAN of `passes` timed passes -> (seconds, requests in sample, batch, threads)"""
    run, n, batch, threads = oracle_prepare(cfg, n_requests, seed_offset, device, workload, summary, agg)
    run()
    return statistics.median([run() for _ in range(passes)]), n, batch, threads


SAMPLE_REQUESTS = {"C1": 1, "C2": 32, "C3": 8, "C4": 64, "C5": 16}  # cpu_baseline: requests per oracle pass (C1-C4: the whole batch)
PARITY_REQUESTS = {"C1": [0], "C2": [5, 27], "C3": [6], "C4": [7, 50], "C5": [33, 90]}   # post-timing sampled parity check


def config_dict(cfg, w, args, world, is_main=True):
    """what both arms print under "config": the workload the metric is quoted on"""
    s = w.spec
    return {"workload": cfg, "batch_per_gpu": s.batch, "num_q_heads": s.num_q_heads,
            "num_kv_heads": s.num_kv_heads, "qk_dim": s.qk_dim, "page_size": s.page_size,
            "seq_len": list(s.seq_len), "budget_pages": w.max_budget, "summary": args.summary if is_main else "envelope",
            "agg": args.agg if is_main else "sum",
            "topk": "exact" if args.topk_approx <= 0 else f"approx tolerate_ratio={args.topk_approx} (lossy)",
            "mla_step": args.mla_step if s.kv_shared else "n/a",
            "kv_dtype": getattr(s, "kv_dtype", "") or s.dtype,
            "l2": "flushed before every step (512 MiB write sweep + 256 MiB read sweep)", "parallelism": f"dp{world}"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_06453_b200.workloads import make_workload, with_fp8
    nreq = SAMPLE_REQUESTS.get(args.config, 1)
    spec = args.config if args.kv_dtype == "same" or args.config == "C1" else with_fp8(args.config, args.kv_dtype)
    w = make_workload(spec, device=_gen_device())     # inputs only; the oracle runs on the host cores
    run, n, batch, threads = oracle_prepare(args.config, nreq, workload=w, summary=args.summary, agg=args.agg)
    t_first = run()                                   # (untimed: also sizes the run)
    budget_s = 150.0                                  # the whole --steps K --warmup W run ends within a few minutes
    per = max(t_first, 1e-3)
    warmup = max(0, min(args.warmup, int(0.2 * budget_s / per)))
    steps = max(1, min(args.steps, int(0.8 * budget_s / per)))
    for _ in range(max(0, warmup - 1)):
        run()
    times = [run() for _ in range(steps)]
    us = statistics.mean(times) / n * batch * 1e6        # scaled from the sample to the whole batch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": "us", "n_gpus": args.gpus, "steps": steps,
            "warmup": max(warmup, 1), "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(args.config, w, args, world),
            "cpu_baseline": {"value": us, "unit": "us", "cores": threads, "kind": "oracle",
                             "sample": f"first {n} of {batch} requests per step (score + top-k + attention)"
                                       + ("" if n == batch else f", scaled by {batch}/{n}") + "; host run, config.l2 does not apply"
                                       + ("" if steps == args.steps else f"; {steps} of the {args.steps} steps asked for fit the time budget")},
            "e2e": {"value": us, "unit": "us", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def _gen_device():
    import torch
    return "cuda:0" if torch.cuda.is_available() else "cpu"


def spawn_ranks(args):
    """`python bench.py --gpus N` without torchrun in front: start the N ranks ourselves (one process per GPU)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def measure(cfg, args, device, local, rank, world, steps, warmup, peak, peak_src, seed_offset):
    """One full record for one workload: K device-timed fused steps (max over ranks), the end-to-end leg, and on rank 0
    the per-stage times, the dominant kernel's roofline, the oracle beside it and a sampled parity check."""
    import torch
    import torch.distributed as dist
    is_main = cfg == args.config
    r = Runner(cfg, device, seed_offset=seed_offset, summary=args.summary if is_main else "envelope",
               topk_approx=args.topk_approx, agg=args.agg if is_main else "sum", mla_step=args.mla_step,
               kv_dtype=args.kv_dtype if cfg != "C1" else "same")
    summary_kind = args.summary if is_main else "envelope"
    w, s = r.w, r.w.spec
    bytes_ = algorithmic_bytes(w, summary=summary_kind)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world > 1:
            t = torch.tensor([x], device=device, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return x

    # ---- the timed region: K fused steps, device-timed, max over ranks --------------------------
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    sampler.ready.wait(timeout=10)          # NVML is up and the first sample is in before the timed region
    times = r.time_device(r.step, steps, warmup)
    launches_per_step = r.ctx.last_launch_count
    barrier()
    clocks = sampler.result()
    ms = max_over_ranks(statistics.mean(times))
    # ---- end to end through the host-buffer entry point ------------------------------------------
    e2e_ms = max_over_ranks(statistics.mean(r.time_host(r.step_host, min(steps, 30), 3)))
    esz = 2 if s.dtype == "bf16" else 4
    h2d = s.batch * s.num_q_heads * s.qk_dim * esz + 4 * (s.batch + 1 + w.total_pages + 2 * s.batch)
    d2h = s.batch * s.num_q_heads * s.v_dim * esz + 4 * s.batch * s.num_q_heads
    rec = None
    if rank == 0:
        # ---- per-stage times (each C-ABI call alone) and the dominant kernel's roofline -------------------
        r.step()
        stage = {}
        for name, fn in (("summary_append", r.stage_summary), ("page_score", r.stage_score),
                         ("topk_pages", r.stage_topk), ("sparse_paged_decode", r.stage_decode)):
            stage[name] = statistics.mean(r.time_device(fn, min(steps, 30), 3)) * 1e3      # us
        stage_bytes = {"page_score": bytes_["summary"], "sparse_paged_decode": bytes_["kv"] + bytes_["qo"]}
        dom = max(stage_bytes, key=lambda k: stage[k])
        achieved = stage_bytes[dom] / (stage[dom] * 1e-6) / 1e9
        traffic, traffic_src = ncu_traffic(cfg, dom) if not getattr(s, "kv_dtype", "") else (None, None)
        roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "algorithmic_bytes": stage_bytes[dom], "us": stage[dom]}
        step_gbs = bytes_["total"] / (ms * 1e-3) / 1e9
        cpu = None
        if not args.no_cpu_baseline:
            t, n, batch, threads = oracle_sample_time(cfg, SAMPLE_REQUESTS.get(cfg, 1), workload=w, summary=summary_kind,
                                                      agg=args.agg if is_main else "sum")
            cpu = {"value": t / n * batch * 1e6, "unit": "us", "cores": threads, "kind": "oracle",
                   "sample": f"first {n} of {batch} requests (score + top-k + attention), one warm-up pass then the median of "
                             f"3 passes, scaled by {batch}/{n}"}
        # ---- sampled parity of the very outputs the timed step produced (outside every timed region) ----------
        parity = None
        if not args.no_cpu_baseline and summary_kind == "envelope" and args.agg == "sum" and args.topk_approx <= 0:
            from oracle.workload_io import parity_sample
            r.step()
            torch.cuda.synchronize()
            parity = parity_sample(w, PARITY_REQUESTS.get(cfg, [0]), r.sel_logical, r.sel_count, r.out, r.lse)
        rec = {"value": ms * 1e3, "unit": "us", "steps": steps, "warmup": warmup, "ms_per_step": ms, "dtype": s.dtype,
               "config": config_dict(cfg, w, args, world, is_main),
               "hbm_gbs": step_gbs, "roofline_frac": step_gbs / peak, "roofline_frac_nominal_8TBs": step_gbs / NOMINAL_HBM_GBS,
               "step_bytes": bytes_, "stage_us": stage, "roofline": roofline, "cpu_baseline": cpu, "parity": parity,
               "e2e": {"value": e2e_ms * 1e3, "unit": "us", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
               "gpu_launches": launches_per_step * steps, "launches_per_step": launches_per_step, "clocks": clocks}
    del r
    torch.cuda.empty_cache()
    return rec


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))
    import __graft_entry__
    if rank == 0:
        __graft_entry__.build()
    if world > 1:
        dist.barrier()
    peak, peak_src = measured_peak()
    main_rec = measure(args.config, args, device, local, rank, world, args.steps, max(args.warmup, 3), peak, peak_src, rank)
    also = {}
    names = [c for c in args.also.split(",") if c and c != args.config]
    if world == 1 and "WORLD_SIZE" not in os.environ:
        # One process per workload: a step's time moves by ~1 us with where the driver places the 4-5 GB pool, and that
        # depends on what the process allocated and freed before (C3 timed after C4 in one process: +0.7..1.0 us on every
        # box tried, C4 after C3: -0.5 us).  A fresh process per record gives every workload the main record's conditions.
        import subprocess
        for name in names:
            cmd = [sys.executable, os.path.abspath(__file__), "--config", name, "--also", "", "--steps", str(args.also_steps),
                   "--warmup", str(max(args.warmup, 3)), "--kv-dtype", args.kv_dtype, "--mla-step", args.mla_step,
                   "--topk-approx", str(args.topk_approx)] + (["--no-cpu-baseline"] if args.no_cpu_baseline else [])
            out = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
            lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
            if out.returncode != 0 or not lines:
                raise SystemExit(f"bench.py: the record of {name} failed (exit {out.returncode}): {out.stderr[-2000:]}")
            rec = json.loads(lines[-1])
            for k in ("also", "metric", "n_gpus", "higher_is_better", "scaling", "vs_baseline", "data", "also_isolation"):
                rec.pop(k, None)
            also[name] = rec
    else:
        for name in names:
            rec = measure(name, args, device, local, rank, world, args.also_steps, max(args.warmup, 3), peak, peak_src, rank)
            if rec is not None:
                also[name] = rec
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        line = {"metric": METRIC, "n_gpus": world, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
                "data": "synthetic"}
        line.update(main_rec)
        line["also"] = also
        line["also_isolation"] = "own process per workload" if (world == 1 and "WORLD_SIZE" not in os.environ) else "in process"
        print(json.dumps(line))


if __name__ == "__main__":
    main()
