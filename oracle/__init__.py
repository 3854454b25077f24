"""Oracle package: TEST INFRASTRUCTURE ONLY (see crt_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It never imports the CUDA package.
"""
from .oracle import *  # noqa: F401,F403
