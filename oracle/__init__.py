"""CPU oracle of the hot path (TEST INFRASTRUCTURE — see ocnref.cpp header).

Importable only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
"""
