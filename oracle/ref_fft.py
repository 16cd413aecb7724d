"""FFT form of the CPU oracle of the projection step: the same definition as oracle/afid_ref.c with the two DFTs
taken by a library FFT (scipy.fft, pocketfft, fp64) -- a library primitive as a step.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/ref.py).  It exists for one purpose: bench.py times it
next to the naive-DFT oracle as `cpu_baseline_fft`, so that the line also carries a CPU number for the O(n log n)
algorithm the paper's CPU code runs (FFTW + Thomas) and not only for the O(n^2) accuracy oracle.
Pinned to ref.project (long double, naive DFT) in tests/test_oracle_pins.py.  Everything but the two transforms is
the C oracle's own routine:
  1     d = D(u, v, w)                                    afid_ref_divergence
  3, 5  H(ky, q) = sum_{j,k} d(j, k) exp(-2 pi i (ky j / ny + q k / nz)),  q = 0..nz/2      scipy.fft.rfft2
  7     x-systems per (ky, q), long double Thomas         afid_ref_solve_half
  9, 11 phi = inverse of 3, 5 with the factor 1/(ny nz)   scipy.fft.irfft2
  correction u -= G phi                                   afid_ref_correct
"""
import numpy as np
import scipy.fft

from . import ref


def project_fft(xc, Ly, Lz, u, v, w, workers=-1):
    """u, v, w: C-contiguous float64 arrays, UPDATED IN PLACE.  Returns p."""
    xc = np.ascontiguousarray(xc, dtype=np.float64)
    nx, ny, nz = v.shape
    assert nz % 2 == 0 and u.shape == (nx + 1, ny, nz) and w.shape == v.shape
    d = ref.divergence(xc, Ly, Lz, u, v, w)
    H = np.ascontiguousarray(scipy.fft.rfft2(d, axes=(1, 2), workers=workers))     # [i][ky][q], unnormalised, exp(-i ...)
    ref.solve_half(xc, Ly, Lz, nz, H)
    p = np.ascontiguousarray(scipy.fft.irfft2(H, s=(ny, nz), axes=(1, 2), workers=workers))
    ref.correct(xc, Ly, Lz, p, u, v, w, inplace=True)
    return p
