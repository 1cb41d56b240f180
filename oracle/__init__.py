"""CPU oracle of the Valencia GRMHD right-hand side -- TEST INFRASTRUCTURE ONLY.

Importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs; the product package (paper_2210_17509_b200) never imports it.
"""
