"""Seeded synthetic inputs for the PersistentKV paged-decode hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_26666_b200/``).  It holds none of the method's arithmetic: it
only draws sequence lengths, builds block tables and fills tensors with
random numbers.  Everything is a pure function of an integer seed.

Recipe (§3.7 page-table generation,
PAPER.md:114-118 §3.8 trace families, BASELINE.json ``configs`` for the
concrete lengths):

* RNG = ``numpy.random.Generator(PCG64(seed))``; draw order: lengths, then the
  page permutation.
* every row reserves ``ceil((N_i + steps) / P)`` logical pages, ``L`` = their
  sum, the physical universe has ``ceil(L / (1 - rho))`` page ids, a seeded
  permutation of the universe hands each row a consecutive slice
  (PAPER.md:112).
* unused block-table entries hold ``PAD_PAGE`` (0x7fffffff) so that a kernel
  that dereferences them faults instead of silently reading a valid page.
* q, K, V ~ N(0,1) rounded to FP16; the whole pool is filled, holes included.
"""
from .serving import ServingStep, ServingTrace  # noqa: F401
from .workloads import (  # noqa: F401
    PAD_PAGE,
    Workload,
    make_page_table,
    make_workload,
    config1,
    config2,
    config3,
    config4,
    config4_b4,
    config5,
    bimodal_lengths,
    zipf_lengths,
    uniform_lengths,
    trace_lengths,
    trace,
    PROMPT_CYCLE,
    fill_normal_f16,
    fill_pool_torch,
    TUNE_SEED,
    REPORT_SEEDS,
)
