"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain CPU restatement, written from PAPER.md, of what the CUDA path in paper_2607_02640_b200/
computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import it.  It never imports the product and the product never imports it.
"""
