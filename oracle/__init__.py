"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, double-precision CPU implementation of what the hot path computes
(arxiv/paper_2602_15605, Eqs. 3, 4, A1-A4), by a route that shares nothing
with the CUDA path: Wigner-3j symbols from the Schulten-Gordon three-term recursion
(`sg_oracle.c`), sums written out literally.  `tables.py` holds the definition of the
lookup-table entries (Eq. 11) in exact integer arithmetic.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It imports nothing from
`paper_2602_15605_b200` and the product imports nothing from here.
"""
from .coupling import (  # noqa: F401
    build,
    lib,
    three_j_family,
    l3_range,
    coupling_pairs,
    coupling_rows,
    coupling_full,
    coupling_band,
    coupling_binned,
    coupling_binned_multi,
    spin1_pairs,
    spin1_full,
    num_threads,
    set_num_threads,
)
from .tables import g_exact_fraction, g_table_float, table_entries_float  # noqa: F401
