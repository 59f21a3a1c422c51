"""Per-CTA phase timelines of the four hot kernels -- a debugging aid, not part of the method.

    python -m paper_2606_06453_b200.trace [--config C3] [--kernel score|topk|decode] [--mode alone|step] [--iters 3]

Builds libvortex_b200_trace.so (`build.py --trace`: the same sources with -DVX_TRACE, every stamp a
`mov.u64 %globaltimer` by one thread of the CTA), runs the kernel on the seeded workload with L2 flushed as in
bench.py -- through its own C-ABI call (`alone`) or inside vx_sparse_decode_step (`step`) -- and prints, per
phase, min / p10 / median / p90 / max over the CTAs in microseconds since the first CTA's entry (top-k in a step:
since the preceding kernel finished, i.e. since griddepcontrol.wait returned).  Times under tracing are a few
hundred ns longer than the product's; they are never bench values.
"""
from __future__ import annotations

import argparse
import os
import sys

SLOTS = {
    "score": {0: "entry", 1: "prod: schedule ready", 2: "prod: first group issued", 3: "prod: ring filled",
              4: "prod: all issued", 5: "cons: first rebuild begin", 6: "cons: first rebuild end",
              7: "cons: last mid-stream rebuild begin", 8: "cons: last mid-stream rebuild end",
              9: "cons: first stage landed", 11: "cons: done"},
    "topk": {0: "entry", 1: "before griddepcontrol.wait", 2: "wait returned", 3: "keys + block min/max",
             4: "histogram done", 5: "threshold bin found", 6: "threshold known", 7: "emission counts",
             8: "ids staged", 9: "exit"},
    "decode_gqa": {0: "entry", 1: "Q loaded", 2: "wait returned", 3: "warp 0: ring filled (issue)",
                   4: "warp 0: page 0 landed", 5: "warp 0: last page landed", 6: "warp 0: loop done",
                   7: "all warps done", 8: "partial stored", 9: "merge begin (last split)", 10: "merge end",
                   11: "exit"},
    "decode_mla": {0: "entry", 1: "barriers + TMEM ready", 2: "Q in TMEM", 3: "wait returned",
                   4: "prod: page 0 issued", 5: "QK: page 0 landed", 6: "QK: last page landed",
                   7: "PV: last issued", 8: "epilogue stored", 9: "cluster barrier passed", 10: "merge done",
                   11: "exit"},
    # the fused MLA step (decode_mla_kernel<FUSED>): `--kernel decode --mode step` on an MLA config
    "step_mla": {0: "entry", 1: "barriers + TMEM ready", 12: "prod: first summary rows issued",
                 13: "cons: first summary stage landed", 14: "scores complete (cluster barrier passed)",
                 2: "selection done", 3: "block table written, decode barriers ready", 4: "prod: page 0 issued",
                 5: "QK: page 0 landed", 6: "QK: last page landed", 7: "PV: last issued", 8: "epilogue stored",
                 9: "cluster barrier passed", 10: "merge done", 11: "exit"},
}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="C3")
    ap.add_argument("--kernel", default="score", choices=["score", "topk", "decode"])
    ap.add_argument("--mode", default="alone", choices=["alone", "step"])
    ap.add_argument("--iters", type=int, default=3)
    args = ap.parse_args()

    from paper_2606_06453_b200 import build as vx_build
    os.environ["VX_B200_LIBRARY"] = vx_build.build(trace=True)
    import numpy as np
    import torch
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200 import binding
    from paper_2606_06453_b200.workloads import make_workload

    dev = "cuda:0"
    w = make_workload(args.config, device=dev)
    s = w.spec
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    B, Hkv = s.batch, s.num_kv_heads
    out = torch.empty(B, s.num_q_heads, s.v_dim, dtype=w.q.dtype, device=dev)
    lse = torch.empty(B, s.num_q_heads, dtype=torch.float32, device=dev)
    sp = torch.empty(B, Hkv, w.max_budget, dtype=torch.int32, device=dev)
    sl, sc = torch.empty_like(sp), torch.empty(B, Hkv, dtype=torch.int32, device=dev)
    scores = torch.empty(Hkv, w.total_pages, dtype=torch.float32, device=dev)
    step = lambda: ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc)
    step()
    fused_step = ctx.last_launch_count == 1       # AUTO takes the one-kernel MLA step for small batches only
    ctx.page_score(w.q, summary, pt, scores)
    torch.cuda.synchronize()
    alone = {"score": lambda: ctx.page_score(w.q, summary, pt, scores),
             "topk": lambda: ctx.topk_pages(scores, pt, w.budget, w.max_budget, sp, sl, sc),
             "decode": lambda: ctx.sparse_paged_decode(w.q, pool, pt, sp, sl, sc, w.max_budget, out, lse)}[args.kernel]
    kind = {"score": binding.VX_TRACE_SCORE, "topk": binding.VX_TRACE_TOPK, "decode": binding.VX_TRACE_DECODE}[args.kernel]
    names = SLOTS[args.kernel if args.kernel != "decode" else ("decode_mla" if s.kv_shared else "decode_gqa")]
    if args.kernel == "decode" and args.mode == "step" and s.kv_shared and fused_step:
        names = SLOTS["step_mla"]                  # (the one-kernel MLA step stamps its own phases)
    buf = torch.zeros(8192, 16, dtype=torch.int64, device=dev)
    ctx.trace_attach(buf, kind)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    sweep = torch.zeros(64 << 20, dtype=torch.int32, device=dev)
    last = max(names)
    zero_slot = 2 if (args.kernel == "topk" and args.mode == "step") else 0
    for it in range(args.iters):
        buf.zero_(); flush.zero_(); sweep.max(); torch.cuda.synchronize()
        (alone if args.mode == "alone" else step)()
        torch.cuda.synchronize()
        b = buf.cpu().numpy()
        b = b[b[:, 0] > 0]
        t0 = b[:, zero_slot].min()
        print(f"--- {args.config} {args.kernel} ({args.mode}) launch {it}: {len(b)} CTAs on {len(set(b[:, 15].tolist()))} SMs, "
              f"span {(b[:, last].max() - b[:, 0].min()) / 1e3:.1f} us")
        for k, n in names.items():
            col = b[:, k]
            ok = col > 0
            if not ok.any():
                continue
            v = (col[ok] - t0) / 1e3
            print(f"{n:44s} n {ok.sum():4d}  min {v.min():6.1f}  p10 {np.percentile(v, 10):6.1f}  med {np.median(v):6.1f}"
                  f"  p90 {np.percentile(v, 90):6.1f}  max {v.max():6.1f}")
        keys = [k for k in names if (b[:, k] > 0).all()]
        print("    per-CTA durations between consecutive stamps:")
        for k0, k1 in zip(keys[:-1], keys[1:]):
            d = (b[:, k1] - b[:, k0]) / 1e3
            print(f"    {names[k0][:30]:30s} -> {names[k1][:30]:30s} min {d.min():6.1f}  med {np.median(d):6.1f}  max {d.max():6.1f}")
        if names is SLOTS["step_mla"]:
            # aggregate HBM rate over time, assuming every CTA streams its summary share evenly between stamps 13 and 14
            # and its pages evenly between stamps 4 and 6 (grid = (splits, 1, batch): CTA index = request * splits + split)
            splits = len(b) // B
            Pn = ((w.seq_lens.cpu().numpy() + s.page_size - 1) // s.page_size)
            kk = np.minimum(w.budget.cpu().numpy(), Pn)
            edges = np.arange(0.0, (b[:, last].max() - t0) / 1e3 + 2.0, 2.0)
            rate = np.zeros(len(edges) - 1)
            row_bytes = 2 * s.qk_dim * 2
            for c in range(len(b)):
                req, sp_ = c // splits, c % splits
                rows = Pn[req] * (sp_ + 1) // splits - Pn[req] * sp_ // splits
                per = -(-kk[req] // splits)
                pages = max(0, min(kk[req], (sp_ + 1) * per) - min(kk[req], sp_ * per))
                for (k0, k1, nbytes) in ((12, 14, rows * row_bytes), (4, 6, pages * s.page_size * s.qk_dim * 2)):
                    a, e = (b[c, k0] - t0) / 1e3, (b[c, k1] - t0) / 1e3
                    if e <= a:
                        continue
                    lo, hi = np.maximum(edges[:-1], a), np.minimum(edges[1:], e)
                    rate += np.clip(hi - lo, 0, None) / (e - a) * nbytes
            print("    aggregate stream rate, TB/s per 2 us bin (summary rows between stamps 12-14, pages between 4-6):")
            print("    " + " ".join(f"{x / 2e-6 / 1e12:4.1f}" for x in rate))
    ctx.trace_attach(None, 0)


if __name__ == "__main__":
    sys.exit(main())
