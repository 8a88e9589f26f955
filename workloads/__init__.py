"""Seeded synthetic inputs for the arXiv 1311.3004 finite-volume step.

This module serves BOTH the CPU oracle (through tests/) and the CUDA path (tests/, bench.py): it only describes
problems -- grid, medium, boundary descriptors, initial fields, step count -- and holds none of the method's
arithmetic (no Riemann solve, no limiter, no update).  It imports neither oracle/ nor paper_1311_3004_b200/.

The paper uses no public data set; its workloads are analytic initial / boundary data (PAPER.md:326-333,
403-432).  Everything here is generated from closed forms and a splitmix64 counter stream.
"""
from .configs import (Workload, MEDIUM_WATER, LAMBDA_1MHZ, c1_piston, c1t_taylor, c2_pulse, c3_random, c4_hifu,
                      c5_sweep, taylor_reference, TAYLOR_STEEP, BY_NAME, EXTRAP, PERIODIC, REFLECT, SOURCE, SINE,
                      PACKET, TANH)  # noqa: F401
from .rng import splitmix64_uniform  # noqa: F401
