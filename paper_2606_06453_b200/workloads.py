"""Seeded synthetic decode workloads (BASELINE.json configs C1..C5 and reduced variants).

This module holds NO arithmetic of the method (no summary, score, selection or
attention): it only draws random tensors, page tables and budgets.  It is the one
module the tests hand to both the CUDA path and the oracle.  Recipe: DESIGN.md
"Input recipe"; shapes follow the paper's decode workloads (PAPER.md:280 first + last
blocks forced, :300 block 16 / ~125 blocks, :262 MLA on one B200), the paper's own
datasets and weights are not reproduced.

Pool layout: K, V = [N_pool, Hkv, page, d] (one contiguous
page*d chunk per (page, head)); MLA latent pool = [N_pool, 1, page, 576], V aliases
K[..., :512].
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import torch


@dataclass(frozen=True)
class Spec:
    name: str
    dtype: str                 # "bf16" | "f32"
    batch: int
    num_q_heads: int
    num_kv_heads: int
    qk_dim: int
    v_dim: int
    page_size: int
    seq_len: tuple             # (lo, hi) inclusive uniform, or (n, n) fixed
    budget: int                # pages incl. forced; 0 -> fraction policy below
    budget_frac: float = 0.0   # k_i = max(budget_min, floor(frac * P_i))   (PAPER.md:516 policy form)
    budget_min: int = 16
    n_sink: int = 1
    n_local: int = 2
    kv_shared: bool = False    # MLA: V = K[..., :v_dim]
    outlier_channels: int = 0  # K channels per KV head scaled x8
    planted_frac: float = 0.0  # fraction of middle pages shifted toward the query direction
    planted_alpha: float = 4.0
    pool_slack: int = 64       # unused physical pages in the pool
    pool_pages: int = 0        # fixed pool size (C1: 128), 0 -> total + slack
    cfg_id: int = 0            # seeds: 1000+id data, 2000+id permutation, 3000+id lengths, 4000+id planted
    block_size: int = 0        # selection block finer than the page: 0 = the page; must divide page_size.
                               # budget, n_sink and n_local then count BLOCKS
    kv_dtype: str = ""         # "" = pools in `dtype`; "e4m3" / "e5m2" = fp8 KV cache: uint8 code pools

    @property
    def sm_scale(self) -> float:
        return float(self.qk_dim) ** -0.5


SPECS = {
    # BASELINE.json configs[0..4]
    "C1": Spec("C1", "f32", 1, 4, 1, 64, 64, 16, (1024, 1024), 8, n_sink=1, n_local=1,
               pool_pages=128, cfg_id=1),
    "C2": Spec("C2", "bf16", 32, 32, 8, 128, 128, 16, (32768, 32768), 128, n_local=2,
               outlier_channels=4, cfg_id=2),
    "C3": Spec("C3", "bf16", 8, 32, 8, 128, 128, 16, (131072, 131072), 256, n_local=4,
               planted_frac=0.01, cfg_id=3),
    "C4": Spec("C4", "bf16", 64, 32, 1, 576, 512, 64, (16384, 65536), 32, n_local=1,
               kv_shared=True, cfg_id=4),
    "C5": Spec("C5", "bf16", 128, 48, 8, 128, 128, 16, (4096, 65536), 0, budget_frac=0.10,
               n_local=2, outlier_channels=4, cfg_id=5),
}
# reduced variants: same structure, sizes the oracle finishes in seconds; ragged tails on purpose
SPECS["C2-small"] = replace(SPECS["C2"], name="C2-small", batch=3, seq_len=(3000, 4100), budget=32)
SPECS["C3-small"] = replace(SPECS["C3"], name="C3-small", batch=2, seq_len=(16384, 16384), budget=64,
                            planted_frac=0.02)
SPECS["C4-small"] = replace(SPECS["C4"], name="C4-small", batch=3, seq_len=(1000, 5000), budget=8)
SPECS["C5-small"] = replace(SPECS["C5"], name="C5-small", batch=6, seq_len=(600, 6000))


def with_fp8(spec: "Spec | str", fmt: str = "e4m3") -> Spec:
    """the same workload with an fp8 KV cache: the pools are drawn as before, then stored as fp8 codes with one scale
    per pool tensor (scale = max |x| / largest fp8 value, so nothing saturates)"""
    spec = SPECS[spec] if isinstance(spec, str) else spec
    assert fmt in ("e4m3", "e5m2") and spec.dtype == "bf16"
    return replace(spec, name=f"{spec.name}-{fmt}", kv_dtype=fmt)


@dataclass
class Workload:
    spec: Spec
    q: torch.Tensor             # [B, Hq, d]
    k_pool: torch.Tensor        # [N_pool, Hkv, page, d]
    v_pool: torch.Tensor | None  # same shape with v_dim, None when kv_shared
    page_indptr: torch.Tensor   # int32 [B+1]
    page_indices: torch.Tensor  # int32 [T]
    seq_lens: torch.Tensor      # int32 [B]
    budget: torch.Tensor        # int32 [B]
    max_budget: int
    total_pages: int
    max_pages_per_req: int
    planted: list = field(default_factory=list)  # per request: logical ids of planted pages
    k_scale: float = 1.0        # fp8 pools: a code c stands for scale * decode(c)
    v_scale: float = 1.0

    @property
    def num_pool_pages(self) -> int:
        return self.k_pool.shape[0]

    @property
    def strides(self):
        """(stride_page, stride_token, stride_head) in elements."""
        s = self.k_pool.stride()
        return s[0], s[2], s[1]

    def to(self, device) -> "Workload":
        mv = lambda t: None if t is None else t.to(device)
        return replace(self, q=mv(self.q), k_pool=mv(self.k_pool), v_pool=mv(self.v_pool),
                       page_indptr=mv(self.page_indptr), page_indices=mv(self.page_indices),
                       seq_lens=mv(self.seq_lens), budget=mv(self.budget))


def _torch_dtype(name: str):
    return {"bf16": torch.bfloat16, "f32": torch.float32}[name]


def make_workload(spec: Spec | str, device="cpu", seed_offset: int = 0) -> Workload:
    """Draw one decode step's inputs.  Deterministic for a given (spec, device type, seed_offset)."""
    if isinstance(spec, str):
        spec = SPECS[spec]
    dev = torch.device(device)
    dt = _torch_dtype(spec.dtype)
    cpu_gen = lambda s: torch.Generator().manual_seed(s + seed_offset)
    g_data = torch.Generator(device=dev).manual_seed(1000 + spec.cfg_id + seed_offset)

    # lengths, page counts, budgets (host side: they size everything else)
    lo, hi = spec.seq_len
    if lo == hi:
        seq = torch.full((spec.batch,), lo, dtype=torch.int64)
    else:
        seq = torch.randint(lo, hi + 1, (spec.batch,), generator=cpu_gen(3000 + spec.cfg_id))
    pages = (seq + spec.page_size - 1) // spec.page_size
    indptr = torch.zeros(spec.batch + 1, dtype=torch.int64)
    indptr[1:] = torch.cumsum(pages, 0)
    total = int(indptr[-1])
    units = pages if not spec.block_size else (seq + spec.block_size - 1) // spec.block_size     # what the budget counts
    if spec.budget > 0:
        budget = torch.full((spec.batch,), spec.budget, dtype=torch.int64)
    else:
        budget = torch.clamp((units.double() * spec.budget_frac).floor().long(), min=spec.budget_min)
    max_budget = int(budget.max())

    # shuffled shared pool: a global seeded permutation dealt to requests in order
    n_pool = spec.pool_pages if spec.pool_pages else total + spec.pool_slack
    assert n_pool >= total
    perm = torch.randperm(n_pool, generator=cpu_gen(2000 + spec.cfg_id))
    indices = perm[:total].to(torch.int32)

    q = torch.randn(spec.batch, spec.num_q_heads, spec.qk_dim, generator=g_data, device=dev,
                    dtype=torch.float32).to(dt)
    kshape = (n_pool, spec.num_kv_heads, spec.page_size, spec.qk_dim)
    k_pool = torch.empty(kshape, dtype=dt, device=dev)
    v_pool = None if spec.kv_shared else torch.empty(
        (n_pool, spec.num_kv_heads, spec.page_size, spec.v_dim), dtype=dt, device=dev)
    step = max(1, (1 << 28) // (spec.num_kv_heads * spec.page_size * spec.qk_dim))  # <=1 GiB fp32 temporaries
    for p0 in range(0, n_pool, step):
        p1 = min(n_pool, p0 + step)
        k_pool[p0:p1] = torch.randn((p1 - p0,) + kshape[1:], generator=g_data, device=dev,
                                    dtype=torch.float32).to(dt)
        if v_pool is not None:
            v_pool[p0:p1] = torch.randn((p1 - p0,) + tuple(v_pool.shape[1:]), generator=g_data,
                                        device=dev, dtype=torch.float32).to(dt)

    if spec.outlier_channels:
        gch = cpu_gen(1500 + spec.cfg_id)
        for h in range(spec.num_kv_heads):
            ch = torch.randperm(spec.qk_dim, generator=gch)[: spec.outlier_channels].to(dev)
            k_pool[:, h, :, ch] = (k_pool[:, h, :, ch].float() * 8.0).to(dt)

    planted = []
    if spec.planted_frac > 0:
        gpl = cpu_gen(4000 + spec.cfg_id)
        grp = spec.num_q_heads // spec.num_kv_heads
        qsum = q.float().view(spec.batch, spec.num_kv_heads, grp, spec.qk_dim).sum(2)
        qhat = qsum / qsum.norm(dim=-1, keepdim=True)          # direction only: data recipe, not a score
        for i in range(spec.batch):
            P = int(pages[i])
            lo_p, hi_p = spec.n_sink, P - spec.n_local          # non-forced pages
            n_pl = max(1, int(round(spec.planted_frac * P)))
            pick = (torch.randperm(hi_p - lo_p, generator=gpl)[:n_pl] + lo_p).sort().values
            planted.append(pick.tolist())
            phys = indices[int(indptr[i]) + pick].long().to(dev)
            blk = k_pool[phys].float() + spec.planted_alpha * qhat[i].view(1, spec.num_kv_heads, 1, -1)
            k_pool[phys] = blk.to(dt)

    k_scale = v_scale = 1.0
    if spec.kv_dtype:
        k_pool, k_scale = _to_fp8_codes(k_pool, spec.kv_dtype)
        if v_pool is not None:
            v_pool, v_scale = _to_fp8_codes(v_pool, spec.kv_dtype)
        else:
            v_scale = k_scale

    return Workload(spec=spec, q=q, k_pool=k_pool, v_pool=v_pool,
                    page_indptr=indptr.to(torch.int32).to(dev), page_indices=indices.to(dev),
                    seq_lens=seq.to(torch.int32).to(dev), budget=budget.to(torch.int32).to(dev),
                    max_budget=max_budget, total_pages=total, max_pages_per_req=int(pages.max()),
                    planted=planted, k_scale=k_scale, v_scale=v_scale)


_FP8 = {"e4m3": (torch.float8_e4m3fn, 448.0), "e5m2": (torch.float8_e5m2, 57344.0)}


def _to_fp8_codes(pool: torch.Tensor, fmt: str):
    """(uint8 codes of the pool stored as fp8, fp32 scale): storage conversion of the drawn data, not the method"""
    tdt, fmax = _FP8[fmt]
    scale = float(torch.tensor(float(pool.abs().max()) / fmax, dtype=torch.float32))
    codes = torch.empty(pool.shape, dtype=torch.uint8, device=pool.device)
    step = max(1, (1 << 27) // max(1, pool[0].numel()))
    for p0 in range(0, pool.shape[0], step):
        codes[p0:p0 + step] = (pool[p0:p0 + step].float() / scale).to(tdt).view(torch.uint8)
    return codes, scale


def subproblem(w: Workload, requests) -> Workload:
    """The same inputs restricted to some requests, on the CPU, with a compact pool
    (only those requests' pages, renumbered).  Pure gathering: lets the oracle check a
    sample of a full-size workload without holding the whole pool on the host."""
    requests = [int(r) for r in requests]
    indptr = w.page_indptr.cpu().long()
    rows = [torch.arange(int(indptr[r]), int(indptr[r + 1])) for r in requests]
    counts = torch.tensor([len(r) for r in rows])
    rows = torch.cat(rows)
    phys = w.page_indices.cpu().long()[rows]
    dev = w.k_pool.device
    k = w.k_pool[phys.to(dev)].cpu()
    v = None if w.v_pool is None else w.v_pool[phys.to(dev)].cpu()
    new_indptr = torch.zeros(len(requests) + 1, dtype=torch.int32)
    new_indptr[1:] = torch.cumsum(counts, 0).to(torch.int32)
    sel = torch.tensor(requests)
    budget = w.budget.cpu()[sel]
    return Workload(spec=replace(w.spec, batch=len(requests)), q=w.q.cpu()[sel].contiguous(),
                    k_pool=k, v_pool=v, page_indptr=new_indptr,
                    page_indices=torch.arange(len(rows), dtype=torch.int32),
                    seq_lens=w.seq_lens.cpu()[sel].contiguous(), budget=budget.contiguous(),
                    max_budget=w.max_budget, total_pages=len(rows),
                    max_pages_per_req=int(counts.max()),
                    planted=[w.planted[r] for r in requests] if w.planted else [], k_scale=w.k_scale, v_scale=w.v_scale)


APPD_DISTRIBUTIONS = ("bimodal", "normal", "lognormal", "uniform")


def appd_scores(dist: str, shape, seed: int) -> torch.Tensor:
    """Seeded fp32 page scores with the value distributions of the paper's top-k study (PAPER.md:485, :497:
    bimodal, normal, lognormal, uniform; its parameters are not printed -- these are stand-ins).  CPU tensor;
    inputs only, no arithmetic of the method."""
    gen = torch.Generator(device="cpu").manual_seed(seed)
    if dist == "normal":
        return torch.randn(shape, generator=gen) * 32.0 + 900.0
    if dist == "uniform":
        return torch.rand(shape, generator=gen) * 100.0
    if dist == "lognormal":
        return torch.exp(torch.randn(shape, generator=gen) * 1.5)
    if dist == "bimodal":
        pick = torch.rand(shape, generator=gen) < 0.1
        return torch.where(pick, torch.randn(shape, generator=gen) * 2.0 + 40.0,
                           torch.randn(shape, generator=gen) * 2.0 - 10.0)
    raise ValueError(dist)
