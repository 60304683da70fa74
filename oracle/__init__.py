"""CPU oracle of the triangle multiplicative update -- test infrastructure, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package; paper_2603_14806_b200 never does.
"""
