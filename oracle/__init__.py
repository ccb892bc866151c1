"""CPU oracle (test infrastructure, not the product). See oracle/dgo.c for what it computes and cites.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from paper_2509_25347_b200.
"""
