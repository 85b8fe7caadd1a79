"""CPU oracle for the FDTD/TDSE hot path (arXiv 2401.07416) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It never imports paper_2401_07416_b200 and shares no code with it.
The arithmetic lives in plain C (tdse_oracle.c, tdse_oracle_step.inc); this module compiles
that file with gcc and marshals numpy arrays through ctypes.
"""
from .driver import (build, lib, OracleRun, potential, mask, wavepacket, stagger,
                     coefficients, max_threads, set_threads, paper_time_step, paper_wavelength,
                     dissimilarity, potential_cell)

__all__ = ["build", "lib", "OracleRun", "potential", "mask", "wavepacket", "stagger",
           "coefficients", "max_threads", "set_threads", "paper_time_step", "paper_wavelength",
           "dissimilarity", "potential_cell"]
