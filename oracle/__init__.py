"""CPU oracle for FP8 attention with the paper's P-cast semantics.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It shares
no code with paper_2606_06521_b200 (the CUDA path) and never imports it.
"""
from .oracle import (  # noqa: F401
    DT_F32, DT_BF16, DT_E4M3, DT_BF16Q_E4M3KV,
    OracleResult, attention_fwd, dp, e4m3_table, e4m3_value, quantize_e4m3, round_e4m3,
)
