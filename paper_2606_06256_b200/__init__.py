"""SegPagedAttention for B200 (sm_100a): a C-ABI library (libsegpa.so, include/segpa.h) with a thin
ctypes binding.  `from paper_2606_06256_b200 import binding` loads the library and fails loudly if
it is not built; `workloads` (seeded inputs) and `harness` (workload -> ABI calls) import lazily."""
__all__ = ["binding", "workloads", "harness"]
