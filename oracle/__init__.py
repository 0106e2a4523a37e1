"""fp64 CPU oracle of the regular-force path -- TEST INFRASTRUCTURE (see oracle.c).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs.
"""
