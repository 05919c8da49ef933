"""CPU oracle (fp64) for the cluster-pair non-bonded step.  TEST INFRASTRUCTURE ONLY:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It imports nothing from paper_2006_09167_b200."""
