"""CPU oracle of the OS+D pulse-profile model (arxiv/paper_2510_07764).  TEST INFRASTRUCTURE:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It shares nothing with paper_2510_07764_b200 (the CUDA product path)."""
from .ppm_oracle import *  # noqa: F401,F403
