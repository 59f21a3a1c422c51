"""Head-union block table -- TEST INFRASTRUCTURE ONLY (only tests/, smoke() and bench.py's oracle legs may import it;
it does not import paper_2606_06453_b200 and shares no code with the CUDA path).

PAPER.md:538 (Table 1): "TopK, Union -- block-table selection and its deduplicated union (trtllm backend)"; :200: the
sparse block table is handed to a paged decode backend, and a backend that takes one table per request needs the
pages any of the request's KV heads selected.  The definition is the plain set union, written with Python sets:

    union[i] = sorted( U_kvh { sel_logical[i, kvh, r] : r < sel_count[i, kvh] } ),   phys = page table lookup.

Reading G24: ascending logical order (as the selection itself, G10), entries outside
[0, P_i) ignored, outputs padded with -1.

Pins (tests/test_oracle_union.py): hand-worked cases; identical heads -> that head's set; disjoint heads -> the
concatenation's size; |union| between max_h |sel_h| and min(P, sum_h |sel_h|); idempotent; permutation of the heads
and of each head's entries changes nothing; every forced page of the selection is in it.
"""
from __future__ import annotations

import numpy as np


def union_pages(sel_logical: np.ndarray, sel_count: np.ndarray, page_indptr, page_indices, seq_lens, page_size: int,
                max_union: int):
    """sel_logical [B, Hkv, max_budget], sel_count [B, Hkv] -> (union_logical, union_phys [B, max_union] pad -1,
    union_count [B])."""
    B, H, _ = sel_logical.shape
    ul = np.full((B, max_union), -1, dtype=np.int32)
    up = np.full((B, max_union), -1, dtype=np.int32)
    uc = np.zeros(B, dtype=np.int32)
    for i in range(B):
        P = (int(seq_lens[i]) + page_size - 1) // page_size
        pages = set()
        for h in range(H):
            for r in range(int(sel_count[i, h])):
                j = int(sel_logical[i, h, r])
                if 0 <= j < P:
                    pages.add(j)
        ordered = sorted(pages)
        assert len(ordered) <= max_union, "max_union below the union's size"
        for pos, j in enumerate(ordered):
            ul[i, pos] = j
            up[i, pos] = int(page_indices[int(page_indptr[i]) + j])
        uc[i] = len(ordered)
    return ul, up, uc
