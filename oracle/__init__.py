"""fp64 CPU oracle of the Block-GTQ hot path -- TEST INFRASTRUCTURE, not the product.

Allowed importers: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline and
--impl reference legs.  Imports nothing from paper_2606_24033_b200/.
"""
