"""fp64 CPU oracle for SegPagedAttention -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2606_06256_b200/csrc and never imports the
CUDA binding; the product path never imports it.
"""
from .binding import OracleResult, build, num_threads, oracle_attention, set_num_threads  # noqa: F401
from .rope_oracle import rope_align, rope_rotate  # noqa: F401
