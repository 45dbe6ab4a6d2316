"""CPU oracle of the Chebyshev-filter hot path.  TEST INFRASTRUCTURE ONLY: importable from tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg, never from the product."""
