"""CPU oracle for the AERA E-field unfolding path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_1507_07733_b200) never does.
The arithmetic lives in aera_oracle.c (plain C, double precision, naive DFT sums);
this file only marshals numpy arrays into it through ctypes.
"""
from .aera_oracle import (  # noqa: F401
    band, dft_band, fold_station, num_threads, pattern_eval, peak, scan, solve2x2,
    analytic_from_band, twiddles, unfold_batch, unfold_station_spectra,
)
