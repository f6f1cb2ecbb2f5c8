"""CPU oracle of the non-hydrostatic step (test infrastructure, NOT the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  Nothing here imports the CUDA package, and vice versa.
"""
