"""CPU oracle for libfasttg.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares nothing with
``paper_2607_05095_b200`` (no imports in either direction).  See ``tg_oracle.c`` for what it
computes and which passages of PAPER.md each function follows, and ``tests/test_oracle_*.py``
for the pins.  Parity status: every function below and in ``cache_oracle`` is pinned (none is "parity unpinned").
"""
from .oracle import (build, num_threads, set_num_threads, block_build, sddmm, edge_softmax_fwd, edge_softmax_bwd,  # noqa: F401
                     aggregate_fwd, aggregate_bwd, attn_fwd, attn_bwd, attn_edge_fwd, attn_edge_bwd, OracleBlock)
