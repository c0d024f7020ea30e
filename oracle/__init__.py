"""CPU oracle for the SK hot path (arXiv 1808.10365) — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  Nothing here imports paper_1808_10365_b200 and nothing there imports this.
"""
