"""CPU oracle for the POLFED hot path -- TEST INFRASTRUCTURE ONLY.

Plain, slow, fp64, written from PAPER.md (arxiv/paper_2605_10191).  Independent of
the CUDA library: no shared code, headers, tables or helpers.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import it; the product package never does.

Pin status (tests/test_oracle_*.py):
  basis, CSR assembly, SpMM, coefficients, Clenshaw, order rule, Gaussian/KPM DOS,
  scalar and block Lanczos, eigenpairs at D <= 12 870: pinned.
  polfed_eigs convergence schedule and completeness at D >= 2^20: parity unpinned
  (readings R9-R11, R21).
"""
from . import cheb, core, lanczos  # noqa: F401
