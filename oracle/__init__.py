"""fp64 CPU oracle of the MAPL boundary codec -- TEST INFRASTRUCTURE (see mapl_oracle.c header).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs.
Shares no code with paper_2606_05484_b200/csrc and imports nothing from the CUDA binding.
"""
