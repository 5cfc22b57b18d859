"""CPU fp64 oracle for Design-CP's pair-bias attention layer -- TEST INFRASTRUCTURE.

Importable only from tests/, __graft_entry__.smoke() and bench.py's CPU legs.  The product
(`paper_2607_05439_b200`) never imports this package and fails loudly without its CUDA library.
"""
