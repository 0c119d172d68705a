"""fp64 CPU oracle for arXiv 1401.4350's force path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_1401_4350_b200/ (the CUDA path) and never imports it.
See oracle/md_oracle.c for what is computed and the paper passages it follows.
"""
from .md_oracle import (Oracle, build, make_pot)  # noqa: F401
