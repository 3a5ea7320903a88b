"""CPU oracle for the thin-disk direct force sum (arXiv 2001.02765).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_2001_02765_b200 and shares no code with it.
"""
from .reference import force, cell_kernels, build  # noqa: F401
