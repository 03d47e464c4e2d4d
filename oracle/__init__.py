"""ORACLE -- test infrastructure, not the product.

A plain, slow, obviously-correct fp64 CPU implementation (numpy + LAPACK's dsytrf as a library step) of what
the CUDA hot path computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import it.  It shares no code with paper_2606_26341_b200/ and imports nothing from it.
"""
