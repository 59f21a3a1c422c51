"""Host-side checks that run without a GPU: the C-ABI library builds, loads and exports every
symbol include/vortex_b200.h declares; geometry validation and workspace sizing (no compute calls)."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def vx():
    from paper_2606_06453_b200 import build
    build.build()
    import paper_2606_06453_b200 as vx
    vx.load_library()
    return vx


def declared_functions():
    names = set()
    for header in sorted(os.listdir(os.path.join(ROOT, "include"))):      # every include/*.h
        text = open(os.path.join(ROOT, "include", header)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(vx_[a-z_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported(vx):
    names = declared_functions()
    assert {"vx_page_summary_update", "vx_page_score", "vx_topk_pages", "vx_sparse_paged_decode",
            "vx_sparse_decode_step"} <= set(names)
    lib = vx.load_library()
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(vx.EXPORTS) == names


def geom(vx, **kw):
    from paper_2606_06453_b200.binding import VxGeom
    base = dict(dtype=0, num_q_heads=32, num_kv_heads=8, qk_dim=128, v_dim=128, page_size=16, kv_shared=0,
                sm_scale=0.088, n_sink=1, n_local=2, agg=0, summary_kind=0, kv_format=0, block_size=0)
    base.update(kw)
    return VxGeom(*[base[f[0]] for f in VxGeom._fields_])


def test_workspace_bytes_and_geometry_validation(vx):
    lib = vx.load_library()
    ws = lambda g, *m: lib.vx_workspace_bytes(C.byref(g), *m)
    small = ws(geom(vx), 4, 1000, 500, 64)
    big = ws(geom(vx), 32, 65536, 2048, 128)
    assert 0 < small < big
    # scores [Hkv, T] fp32 + partials [B, Hq, 32, dv] fp32 dominate
    assert big >= 8 * 65536 * 4 + 32 * 32 * 32 * 128 * 4
    assert ws(geom(vx, num_q_heads=30), 4, 1000, 500, 64) == 0          # Hq % Hkv != 0
    assert ws(geom(vx, qk_dim=80, v_dim=80), 4, 1000, 500, 64) == 0     # unsupported width
    assert ws(geom(vx, agg=1), 4, 1000, 500, 64) > 0                    # max_h aggregation: GQA groups of <= 8 heads
    assert ws(geom(vx, agg=2), 4, 1000, 500, 64) == 0                   # unknown aggregation
    assert ws(geom(vx, dtype=0, num_q_heads=32, num_kv_heads=1, qk_dim=576, v_dim=512, page_size=64,
                   kv_shared=1), 64, 50000, 1024, 32) > 0              # MLA geometry
    assert ws(geom(vx, dtype=0, num_q_heads=32, num_kv_heads=1, qk_dim=576, v_dim=512, page_size=64,
                   kv_shared=1, agg=1), 64, 50000, 1024, 32) > 0       # max_h over the 32-head MLA group: tensor-core scoring
    assert ws(geom(vx, dtype=0, num_q_heads=8, num_kv_heads=1, qk_dim=576, v_dim=512, page_size=64,
                   kv_shared=1, agg=1), 64, 50000, 1024, 32) == 0      # ... which takes 16 or 32 heads only
    assert ws(geom(vx, dtype=1, num_q_heads=4, num_kv_heads=1, qk_dim=64, v_dim=64), 1, 64, 64, 8) > 0


def test_create_fails_loudly_without_a_gpu(vx):
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = vx.load_library()
    h = C.c_void_p()
    g = geom(vx)
    buf = (C.c_char * 4096)()
    st = lib.vx_create(C.byref(h), C.byref(g), 0, C.c_void_p((C.addressof(buf) + 255) // 256 * 256), 1 << 40,
                       1, 16, 16, 8)
    assert st == 4 and not h.value and b"cuda" in lib.vx_last_error(None).lower()
    with pytest.raises(vx.VortexError):
        vx.Context(dtype=torch.bfloat16, num_q_heads=32, num_kv_heads=8, qk_dim=128, v_dim=128, page_size=16,
                   sm_scale=0.1, n_sink=1, n_local=2, max_batch=1, max_total_pages=16, max_pages_per_req=16,
                   max_budget=8, device="cpu")


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_06453_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                for line in open(os.path.join(dirpath, f)).read().splitlines():
                    uses = any(w in line for w in ("import", "#include", "CDLL", "dlopen", "subprocess"))
                    assert not (uses and "oracle" in line), (f, line)
