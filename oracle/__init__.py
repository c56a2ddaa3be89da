"""ORACLE package -- test infrastructure only (see nbody_oracle.py header).

Importers allowed: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline and
`--impl reference` legs.  Nothing under paper_0707_0438_b200/ imports this.
"""
