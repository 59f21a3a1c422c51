"""Edge cases of the fused step across the storage / granularity variants (-m gpu): requests of a few tokens (one partial
page; fewer pages than the budget; fewer pages than the forced counts), n_local = 0 (the newest page is not forced, so the
summary kernel must run before the score kernel), budgets that are all forced pages -- for bf16 pools, an fp8 KV cache,
blocks finer than the page, and both together, GQA and MLA.  Each against the fp64 oracle by the parity comparators."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from oracle.workload_io import oracle_step
from tests.parity import check_attention, check_selection, oracle_attention_on

pytestmark = pytest.mark.gpu

VARIANTS = {"bf16": {}, "fp8": dict(fp8="e4m3"), "blocks": dict(page=32, block=16), "fp8+blocks": dict(fp8="e5m2", page=64, block=16)}
SHAPES = {
    "tiny-requests": dict(batch=7, seq_len=(1, 90), budget=4, n_sink=1, n_local=2),
    "no-local": dict(batch=4, seq_len=(200, 1500), budget=9, n_sink=1, n_local=0),
    "forced-only": dict(batch=3, seq_len=(300, 900), budget=3, n_sink=1, n_local=2),
    "no-forced": dict(batch=3, seq_len=(64, 700), budget=6, n_sink=0, n_local=0),
}


@pytest.mark.parametrize("base", ["C2-small", "C4-small"])
@pytest.mark.parametrize("variant", list(VARIANTS))
@pytest.mark.parametrize("shape", list(SHAPES))
def test_edge_cases(base, variant, shape):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import SPECS, make_workload, with_fp8
    v = dict(VARIANTS[variant])
    fp8 = v.pop("fp8", None)
    spec = replace(SPECS[base], name=f"{base}-{variant}-{shape}", cfg_id=70 + list(SHAPES).index(shape), **SHAPES[shape])
    if "page" in v:
        if base == "C4-small" and v["page"] != 64:
            v = dict(page=64, block=16)
        spec = replace(spec, page_size=v["page"], block_size=v["block"])
    if fp8:
        spec = with_fp8(spec, fp8)
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    dev = w.q.device
    ctx = vx.context_for(w)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    first = (w.seq_lens - 1).clamp(min=0)                                # everything but the newest token's unit is summarised ...
    unit = s.block_size or s.page_size
    ctx.page_summary_update(pool, pt, summary, first_new_pos=(first // unit) * unit)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))   # (bulk build: the reference state)
    clean = summary.clone()
    out = torch.full((s.batch, s.num_q_heads, s.v_dim), float("nan"), dtype=w.q.dtype, device=dev)
    lse = torch.full((s.batch, s.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    sp = torch.full((s.batch, s.num_kv_heads, w.max_budget), -7, dtype=torch.int32, device=dev)
    sl, sc = torch.full_like(sp, -7), torch.full((s.batch, s.num_kv_heads), -7, dtype=torch.int32, device=dev)
    ctx.sparse_decode_step(w.q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc, flags=vx.VX_STEP_UPDATE_SUMMARY)
    torch.cuda.synchronize()
    assert torch.equal(summary, clean), "the append update leaves a bulk-built pool unchanged"
    ref = oracle_step(w)
    check_selection(w, sl.cpu().numpy(), sp.cpu().numpy(), sc.cpu().numpy(), ref, label=spec.name)
    o_ref, l_ref = oracle_attention_on(w, sl.cpu().numpy(), sc.cpu().numpy())
    check_attention(s.dtype, out.float().cpu().numpy(), lse.cpu().numpy(), o_ref, l_ref)
    nu = -(-w.seq_lens.cpu().numpy() // unit)
    assert np.array_equal(sc.cpu().numpy(), np.minimum(w.budget.cpu().numpy(), nu)[:, None].repeat(s.num_kv_heads, 1))
    ctx.close()
