"""Offline profiling of the top-k remap (App. D.2: "a monotonic transformation x' = f(x) that preserves
ordering while reshaping the value distribution ... selected offline through profiling and fused into the histogram pass").

f is a knot table for `Context.set_topk_remap` (include/vortex_b200.h: vx_set_topk_remap; reading G29):
n values in [0, 1], non-decreasing, f piecewise linear between them on the score normalised by the request's own
min / max.  `profile_knots` fits the table to sample score rows (one row per (request, KV head) problem, e.g. captured
from `Context.page_score` on representative traffic): the empirical distribution function of the normalised scores, so
that the first radix pass spreads the pages evenly over its bins -- mixed with the identity by `blend` in [0, 1], because
a selection of the k largest wants the TOP of the range resolved finely, not the bulk.

    python -m paper_2606_06453_b200.remap_profile --dist lognormal --pages 8192 --knots 33
prints the table fitted to one of the App. D score distributions (workloads.appd_scores).
"""
from __future__ import annotations

import argparse

import numpy as np

MAX_KNOTS = 65


def profile_knots(rows, n_knots: int = 33, blend: float = 1.0) -> np.ndarray:
    """rows: iterable of 1-D score arrays (one per problem).  Returns n_knots float32 values, 0 = f(0) <= ... <= f(1) = 1."""
    if not 2 <= n_knots <= MAX_KNOTS:
        raise ValueError(f"n_knots must be in [2, {MAX_KNOTS}]")
    if not 0.0 <= blend <= 1.0:
        raise ValueError("blend must be in [0, 1]")
    grid = np.linspace(0.0, 1.0, n_knots)
    cdf = np.zeros(n_knots, dtype=np.float64)
    total = 0
    for r in rows:
        x = np.asarray(r, dtype=np.float64).ravel()
        x = x[np.isfinite(x)]
        if x.size < 2 or x.max() <= x.min():
            continue
        t = np.sort((x - x.min()) / (x.max() - x.min()))
        cdf += np.searchsorted(t, grid, side="right")
        total += x.size
    if total == 0:
        return grid.astype(np.float32)
    f = blend * (cdf / total) + (1.0 - blend) * grid
    f[0], f[-1] = 0.0, 1.0
    f = np.clip(np.maximum.accumulate(f), 0.0, 1.0)
    return f.astype(np.float32)


def main() -> int:
    from .workloads import APPD_DISTRIBUTIONS, appd_scores
    ap = argparse.ArgumentParser()
    ap.add_argument("--dist", default="lognormal", choices=list(APPD_DISTRIBUTIONS))
    ap.add_argument("--pages", type=int, default=8192)
    ap.add_argument("--problems", type=int, default=64)
    ap.add_argument("--knots", type=int, default=33)
    ap.add_argument("--blend", type=float, default=1.0)
    args = ap.parse_args()
    sc = appd_scores(args.dist, (args.problems, args.pages), seed=1).numpy()
    print(" ".join(f"{v:.6f}" for v in profile_knots(sc, args.knots, args.blend)))
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
