"""CPU oracle for PDBO -- TEST INFRASTRUCTURE ONLY (see oracle/pdbo_oracle.c header).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
"""
