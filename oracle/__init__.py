"""CPU oracle for the LdG/FIRE hot path (arXiv:1911.07045).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_1911_07045_b200/`` may import
this package; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs use it.  See ``lq_oracle.c`` for the
citations and the list of pins.
"""
from .lq_oracle import (  # noqa: F401
    Oracle,
    analyze,
    build_oracle,
    oracle_lib_path,
    q0_of,
    S0_of,
    num_threads,
    set_num_threads,
)
