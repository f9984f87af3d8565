"""CPU oracle of the columnar HEP kernels (arXiv:1906.06242).  TEST INFRASTRUCTURE ONLY.

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs.  Shares no code with paper_1906_06242_b200/ (the CUDA path); neither imports the other.
"""
