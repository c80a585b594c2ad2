"""CPU oracle for the TNLM hot path.  TEST INFRASTRUCTURE ONLY (see tnlm_oracle.c header).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs.  Never imported by paper_1201_2450_b200.
"""
