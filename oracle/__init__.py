"""ORACLE package: test infrastructure only (see spf_oracle.c header).

Importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs -- never from paper_2109_05339_b200/.
"""
