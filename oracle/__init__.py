"""TEST INFRASTRUCTURE, NOT THE PRODUCT: the CPU oracle of the Hermite-6 hot path.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports the CUDA package's binding and shares no code with it.
"""
from .hermite6 import OracleSystem, build, lib  # noqa: F401
