"""fp64 CPU oracle for the PRISM / multislice hot path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` leg may import this package.  It shares no code with
``paper_1706_08563_b200`` (the CUDA product) and never imports it.
"""
from .oracle import *  # noqa: F401,F403
