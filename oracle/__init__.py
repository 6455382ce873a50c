"""CPU oracle of the OSB-PD explicit step -- TEST INFRASTRUCTURE, not the product.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package."""
