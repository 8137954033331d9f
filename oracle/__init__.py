"""CPU oracle for the CUDACPP hot path -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg import this package.
"""
