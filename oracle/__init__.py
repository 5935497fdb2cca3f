"""ORACLE -- test infrastructure only (see magnus_oracle.cpp's header).

Importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs only.  Never imported by paper_1709_06483_b200.
"""
