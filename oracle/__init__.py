"""CPU oracle for the implicit-depletant HPMC trial move (arXiv 1508.07077).

TEST INFRASTRUCTURE ONLY.  Importable from ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` leg; never from the product package
``paper_1508_07077_b200``.  See ``hpmc_oracle.cpp`` for what is computed and which passage
of PAPER.md each step follows.
"""
from .binding import (  # noqa: F401
    Oracle,
    OracleParams,
    COUNTER_NAMES,
    build,
    lib,
)
