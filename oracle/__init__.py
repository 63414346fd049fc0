"""CPU oracle for the NEURON-Fabric low-bit bucket-aggregation path.

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs. The product package never imports this.
"""
