"""CPU oracle for the XY Swendsen-Wang sweep (test infrastructure only).

Importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs -- never from paper_1210_6116_b200/.
"""
