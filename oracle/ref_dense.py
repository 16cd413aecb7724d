"""Large-case CPU oracle of the projection step: the same definition as oracle/afid_ref.c, with every
DFT written as a product with the dense DFT matrix (a library matmul as the step, fp64).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/ref.py).  SURVEY.md 8(c) step 8 allows
fp64 sums with blocked partial sums for C3 and larger, where the long-double sums of afid_ref.c
would take hours; a BLAS dgemm is exactly that (blocked fp64 partial sums, error ~ eps sqrt(n)).
Still O(n^2) per line, no FFT.  Pinned to ref.project (long double) in tests/test_oracle_pins.py.

Steps (paper numbering), plane by plane in x:
  1   d = D(u, v, w)                                   (afid_ref_divergence, C)
  3   H(j, q) = sum_k d(j, k) exp(-2 pi i q k / nz),   q = 0..nz/2   (d real: the spectrum is Hermitian
      in kz, only the non-redundant half is kept)
  5   H(ky, q) = sum_j exp(-2 pi i ky j / ny) H(j, q)
  7   x-systems per (ky, q), long double Thomas        (afid_ref_solve_half, C)
  9   G(j, q) = sum_ky exp(+2 pi i ky j / ny) X(ky, q)
  11  phi(j, k) = 1/(ny nz) [ Re G(j,0) + (-1)^k Re G(j,nz/2) + 2 sum_{q=1}^{nz/2-1} Re(G(j,q) e^{+2 pi i q k/nz}) ]
      (the sum over all nz modes folded by the Hermitian symmetry)
  correction u -= G phi                                (afid_ref_correct, C)
Complex products are carried out as real matmuls on the real and imaginary parts.
"""
import numpy as np

from . import ref


def dft_matrix(n, rows=None):
    """(cos, sin) of 2 pi (q k mod n) / n for q < rows, k < n; index reduced in integers, long double angles."""
    rows = n if rows is None else rows
    m = (np.arange(rows, dtype=np.int64)[:, None] * np.arange(n, dtype=np.int64)[None, :]) % n
    tab = np.arange(n, dtype=np.longdouble) * (np.longdouble(2.0) * np.arccos(np.longdouble(-1.0)) / np.longdouble(n))
    c = np.cos(tab).astype(np.float64)
    s = np.sin(tab).astype(np.float64)
    return c[m], s[m]


def project_dense(xc, Ly, Lz, u, v, w):
    """u, v, w: C-contiguous float64 arrays, UPDATED IN PLACE.  Returns p."""
    xc = np.ascontiguousarray(xc, dtype=np.float64)
    nx, ny, nz = v.shape
    assert nz % 2 == 0 and u.shape == (nx + 1, ny, nz) and w.shape == v.shape
    for a in (u, v, w):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    nzh = nz // 2 + 1
    cz, sz = dft_matrix(nz, nzh)                      # [q][k]
    cy, sy = dft_matrix(ny)                           # [ky][j], symmetric
    czT, szT = np.ascontiguousarray(cz.T), np.ascontiguousarray(sz.T)
    H = np.empty((nx, ny, nzh), dtype=np.complex128)
    p = ref.divergence(xc, Ly, Lz, u, v, w)           # step 1; p serves as the real work array
    for i in range(nx):
        d = p[i]                                      # [ny][nz]
        hr, hi = d @ czT, -(d @ szT)                  # exp(-i t) = cos t - i sin t
        H[i].real = cy @ hr + sy @ hi                 # (cy - i sy)(hr + i hi)
        H[i].imag = cy @ hi - sy @ hr
    ref.solve_half(xc, Ly, Lz, nz, H)
    fold = np.full(nzh, 2.0)
    fold[0] = fold[-1] = 1.0
    scale = 1.0 / (float(ny) * float(nz))
    fc, fs = fold[:, None] * cz * scale, fold[:, None] * sz * scale     # [q][k]
    for i in range(nx):
        xr, xi = np.ascontiguousarray(H[i].real), np.ascontiguousarray(H[i].imag)
        gr = cy @ xr - sy @ xi                        # (cy + i sy)(xr + i xi)
        gi = cy @ xi + sy @ xr
        p[i] = gr @ fc - gi @ fs                      # Re(G e^{+i t}) = Gr cos t - Gi sin t
    del H
    ref.correct(xc, Ly, Lz, p, u, v, w, inplace=True)
    return p
