"""vx_sparse_decode_step under CUDA graph capture (-m gpu).  include/vortex_b200.h promises that the device entry points
enqueue work only -- no synchronisation, no host read of device memory, no allocation -- so a step can be captured once
and replayed (SURVEY.md 8(b) "CUDA-graph-capturable").  Every schedule of the step is captured, replayed twice on NEW
queries written into the captured buffers, and compared bit for bit with the eager call: that also shows that the
kernels leave their workspace counters (split arrivals, the flat MLA kernel's sync words) as they found them."""
from dataclasses import replace

import pytest
import torch

pytestmark = pytest.mark.gpu


def _cases():
    from paper_2606_06453_b200.workloads import SPECS, with_fp8
    import paper_2606_06453_b200 as vx
    mla = replace(SPECS["C4"], name="graph-mla", batch=6, seq_len=(700, 9000), budget=12, cfg_id=61)
    return {
        "gqa-chained": (SPECS["C2-small"], None),
        "gqa-ragged": (SPECS["C5-small"], None),
        "gqa-fp8": (with_fp8("C2-small"), None),
        "gqa-blocks": (replace(SPECS["C2-small"], name="graph-blocks", page_size=32, block_size=16), None),
        "mla-chained": (mla, vx.VX_MLA_STEP_CHAINED),
        "mla-fused": (mla, vx.VX_MLA_STEP_FUSED),
        "mla-flat": (mla, vx.VX_MLA_STEP_FLAT),
        "fp32-generic": (SPECS["C1"], None),
    }


@pytest.mark.parametrize("case", ["gqa-chained", "gqa-ragged", "gqa-fp8", "gqa-blocks", "mla-chained", "mla-fused", "mla-flat",
                                  "fp32-generic"])
def test_step_replays_from_a_cuda_graph(case):
    import paper_2606_06453_b200 as vx
    from paper_2606_06453_b200.workloads import make_workload
    spec, mla_step = _cases()[case]
    w = make_workload(spec, device="cuda:0")
    s = w.spec
    dev = w.q.device
    ctx = vx.context_for(w)
    if mla_step is not None:
        ctx.set_option(vx.VX_OPT_MLA_STEP, mla_step)
    pool, pt = vx.tables_for(w)
    summary = vx.alloc_summary(w)
    ctx.page_summary_update(pool, pt, summary, first_new_pos=torch.zeros_like(w.seq_lens))
    q = w.q.clone()
    out = torch.empty(s.batch, s.num_q_heads, s.v_dim, dtype=q.dtype, device=dev)
    lse = torch.empty(s.batch, s.num_q_heads, dtype=torch.float32, device=dev)
    sp = torch.empty(s.batch, s.num_kv_heads, w.max_budget, dtype=torch.int32, device=dev)
    sl, sc = torch.empty_like(sp), torch.empty(s.batch, s.num_kv_heads, dtype=torch.int32, device=dev)

    def step():
        ctx.sparse_decode_step(q, pool, summary, pt, w.budget, w.max_budget, out, lse, sp, sl, sc, flags=vx.VX_STEP_UPDATE_SUMMARY)

    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                   # warm-up outside the capture (one-time per-kernel attribute calls)
        step()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        step()
    gen = torch.Generator(device=dev).manual_seed(99)
    for it in range(2):
        q.copy_(torch.randn(q.shape, generator=gen, device=dev, dtype=torch.float32).to(q.dtype))
        for t in (out, lse):
            t.fill_(float("nan"))
        for t in (sp, sl, sc):
            t.fill_(-7)
        graph.replay()
        torch.cuda.synchronize()
        got = [t.clone() for t in (out, lse, sp, sl, sc)]
        step()                                      # the same inputs, eagerly
        torch.cuda.synchronize()
        for a, b, name in zip(got, (out, lse, sp, sl, sc), ("out", "lse", "sel_phys", "sel_logical", "sel_count")):
            same = torch.equal(a.view(torch.uint8) if a.dtype == torch.bfloat16 else a, b.view(torch.uint8) if b.dtype == torch.bfloat16 else b)
            assert same, f"{case}: replay {it} differs from the eager step in {name}"
        assert bool(torch.isfinite(out.float()).all()) and int(sc.min()) >= 0
    ctx.close()
