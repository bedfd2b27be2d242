"""CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_1910_12578_b200/.
See oracle/orc.c for the arithmetic and oracle/orc.py for the ctypes wrapper.
"""
