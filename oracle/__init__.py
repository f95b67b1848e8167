"""CPU oracle for the cubic-FP closure hot path (arxiv/paper_2606_15622).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with ``paper_2606_15622_b200`` (the CUDA
path) and neither imports the other.  The arithmetic lives in ``fp_oracle.c`` (plain C, fp64); this module is a
ctypes/numpy marshalling layer plus the composition of one ``fp_step`` in the order of PAPER.md Algorithm 1/2
(:205-225, :250-270).
"""
from .oracle import *  # noqa: F401,F403
