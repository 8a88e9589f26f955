"""CPU oracle of the arXiv 1311.3004 finite-volume step -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
"""
from .oracle import Oracle, OrcSource, riemann, flux, mc_phi, sweep_line  # noqa: F401
