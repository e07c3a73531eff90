"""oracle/ — TEST INFRASTRUCTURE, not the product.

A plain fp64 CPU evaluator of the Beagle scoring path written from the paper (beagle_oracle.c),
its ctypes binding (binding.py) and an independent recursive evaluator (infix_check.py) used only
to pin the oracle by brute force. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package. Nothing here imports the CUDA package.
"""
