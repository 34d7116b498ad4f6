"""oracle — TEST INFRASTRUCTURE, NOT PRODUCT.

Plain fp64 CPU statement of the JefiPIC hot path (arXiv 2209.07944), written from PAPER.md.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; the product (``paper_2209_07944_b200``) never does, and this package never
imports the product.
"""
from .jefi_oracle import (  # noqa: F401
    OracleConfig,
    OracleJefi,
    build_oracle,
    delay,
    RULE_NEAREST,
    RULE_LINEAR,
    delay_table,
    num_dt,
    num_threads,
    set_num_threads,
    field,
    deposit,
    interp,
    push,
    cell_index,
)
