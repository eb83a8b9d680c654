"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

Serial fp64 CPU oracle for the HPMC checkerboard sweep (arXiv:1509.04692), written from the
paper.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package; nothing under paper_1509_04692_b200/ does, and this package
imports nothing from there.
"""
