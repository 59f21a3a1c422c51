"""Top-k microbenchmark on the score distributions of the paper's App. D.2/D.3 (bimodal,
normal, lognormal, uniform): times vx_topk_pages alone on synthetic page scores and checks every result against
torch.topk (set equality; ties are measure-zero for these draws).

The paper reports its radix_topk as "highly sensitive to the score distribution" (:194); the select here bins
the LIVE key range of each problem, so the four distributions should cost the same.

With --ratios the approximate selection (vx_topk_pages_approx, PAPER.md:196 stochastic early termination) is timed
beside it at each tolerate_ratio, with its mean / min recall@k against the exact set (PAPER.md:497 reports latency at
recall@k > 0.97).  With --remap the two remapped variants of App. D.2 (:485 "radix topk with remap", "approx_radix_topk +
remap") are timed as well: a knot table fitted offline (remap_profile.profile_knots) to OTHER draws of the same
distribution is installed with vx_set_topk_remap, then tolerate_ratio 0 (the exact selection through the remapped first
pass, checked against the exact set) and each ratio are timed again.

    python -m paper_2606_06453_b200.topk_microbench [--batch 32] [--heads 8] [--iters 50] [--ratios 0.05,0.1,0.25] [--remap]
"""
from __future__ import annotations

import argparse
import json

import torch

from . import binding as vx


def draw(dist: str, shape, seed, device):
    """the App. D stand-in distributions: workloads.appd_scores (the one generator the tests use too), moved to the GPU"""
    from .workloads import appd_scores
    return appd_scores(dist, shape, seed).to(device)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--batch", type=int, default=32)
    ap.add_argument("--heads", type=int, default=8)
    ap.add_argument("--iters", type=int, default=50)
    ap.add_argument("--ratios", default="0.05,0.1,0.25", help="tolerate_ratio values for vx_topk_pages_approx ('' = none)")
    ap.add_argument("--remap", action="store_true", help="also time the selection with an offline-profiled remap table installed")
    ap.add_argument("--knots", type=int, default=33)
    args = ap.parse_args()
    dev = "cuda:0"
    gen = torch.Generator(device=dev).manual_seed(77)
    B, H = args.batch, args.heads
    rows = []
    for P in (2048, 8192, 32768):
        for k in (32, 128, 256):
            T = B * P
            ctx = vx.Context(dtype=torch.bfloat16, num_q_heads=4 * H, num_kv_heads=H, qk_dim=128, v_dim=128, page_size=16,
                             sm_scale=1.0, n_sink=1, n_local=2, max_batch=B, max_total_pages=T, max_pages_per_req=P,
                             max_budget=k, device=dev)
            indptr = (torch.arange(B + 1, dtype=torch.int32, device=dev) * P)
            indices = torch.randperm(T, generator=gen, device=dev).to(torch.int32)
            seq = torch.full((B,), P * 16, dtype=torch.int32, device=dev)
            pt = vx.PageTable(indptr, indices, seq, T, P)
            budget = torch.full((B,), k, dtype=torch.int32, device=dev)
            sp = torch.empty(B, H, k, dtype=torch.int32, device=dev)
            sl = torch.empty_like(sp)
            sc = torch.empty(B, H, dtype=torch.int32, device=dev)
            for dist in ("bimodal", "normal", "lognormal", "uniform"):
                scores = draw(dist, (H, T), 7700 + P + k, dev)
                ctx.topk_pages(scores, pt, budget, k, sp, sl, sc)
                torch.cuda.synchronize()
                # exactness: forced pages + the k - 3 best of the rest, as a set per problem
                s3 = scores.view(H, B, P).permute(1, 0, 2).clone()
                s3[:, :, 0] = float("inf"); s3[:, :, P - 2:] = float("inf")
                want = torch.topk(s3, k, dim=-1).indices.sort(-1).values
                assert torch.equal(sl.long(), want), (P, k, dist)
                # device time: `iters` back-to-back launches replayed as ONE CUDA graph (the C ABI is capturable:
                # no host sync, no device->host reads), so the host's per-call cost does not starve the GPU
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph):
                    for _ in range(args.iters):
                        ctx.topk_pages(scores, pt, budget, k, sp, sl, sc)
                graph.replay()
                torch.cuda.synchronize()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(); graph.replay(); b.record()
                torch.cuda.synchronize()
                us = a.elapsed_time(b) * 1e3 / args.iters
                assert torch.equal(sl.long(), want), (P, k, dist, "after graph replay")
                row = dict(pages=P, k=k, dist=dist, problems=B * H, us=round(us, 2))
                taus = [float(x) for x in args.ratios.split(",") if x] if P <= 8192 else []

                def time_approx(tau, name):
                    ctx.topk_pages_approx(scores, pt, budget, k, tau, 7, sp, sl, sc)
                    torch.cuda.synchronize()
                    hit = (sl.long().unsqueeze(-1) == want.unsqueeze(-2)).any(-1).float().sum(-1) / k   # [B, H] recall@k
                    if tau == 0.0:
                        assert torch.equal(sl.long(), want), (P, k, dist, name)       # ratio 0 stays exact under any table
                    g2 = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g2):
                        for _ in range(args.iters):
                            ctx.topk_pages_approx(scores, pt, budget, k, tau, 7, sp, sl, sc)
                    g2.replay()
                    torch.cuda.synchronize()
                    a.record(); g2.replay(); b.record()
                    torch.cuda.synchronize()
                    row[name] = dict(us=round(a.elapsed_time(b) * 1e3 / args.iters, 2),
                                     recall_mean=round(hit.mean().item(), 4), recall_min=round(hit.min().item(), 4))

                for tau in taus:
                    time_approx(tau, f"approx_{tau}")
                if args.remap and P <= 8192:
                    from .remap_profile import profile_knots
                    ctx.set_topk_remap(profile_knots(draw(dist, (8, P), 990000 + P + k, "cpu").numpy(), args.knots))
                    for tau in [0.0] + taus:
                        time_approx(tau, f"remap_{tau}")
                    ctx.set_topk_remap(None)
                rows.append(row)
                print(json.dumps(rows[-1]))
            ctx.close()
    by = {}
    for r in rows:
        by.setdefault((r["pages"], r["k"]), []).append(r["us"])
    worst = max(max(v) / min(v) for v in by.values())
    print(json.dumps({"max_spread_across_distributions": round(worst, 3)}))


if __name__ == "__main__":
    main()
