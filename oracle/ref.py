"""ctypes/numpy front end of the CPU oracle (oracle/afid_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from the CUDA
package and the CUDA package imports nothing from here.

Every function is a thin marshaller: numpy arrays in, the C routine does all arithmetic.
Citations ("P:L<n>" = /root/reference/PAPER.md line n) are in afid_ref.c.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.afid_ref_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _chk(rc, name):
    if rc != 0:
        raise RuntimeError(f"{name} failed with code {rc}")


def num_threads():
    return int(lib().afid_ref_num_threads())


def metrics(xc):
    """dx[i] (nx cell widths) and dc[i] (nx+1; centre-to-centre distances at faces 1..nx-1)."""
    xc = _f64(xc)
    nx = xc.size - 1
    dx = np.empty(nx)
    dc = np.empty(nx + 1)
    _chk(lib().afid_ref_metrics(C.c_int(nx), _p(xc), _p(dx), _p(dc)), "afid_ref_metrics")
    return dx, dc


def wavenumbers(n, L):
    lam = np.empty(n)
    _chk(lib().afid_ref_wavenumbers(C.c_int(n), C.c_double(L), _p(lam)), "afid_ref_wavenumbers")
    return lam


def divergence(xc, Ly, Lz, u, v, w):
    xc, u, v, w = _f64(xc), _f64(u), _f64(v), _f64(w)
    nx, ny, nz = v.shape
    assert u.shape == (nx + 1, ny, nz) and w.shape == v.shape and xc.size == nx + 1
    d = np.empty((nx, ny, nz))
    _chk(lib().afid_ref_divergence(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                                   C.c_double(Lz), _p(u), _p(v), _p(w), _p(d)), "afid_ref_divergence")
    return d


def correct(xc, Ly, Lz, phi, u, v, w, inplace=False):
    """Returns corrected copies (u - G phi); inplace=True updates the given contiguous fp64 arrays instead."""
    xc, phi = _f64(xc), _f64(phi)
    if inplace:
        assert all(isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous for a in (u, v, w))
    else:
        u, v, w = _f64(u).copy(), _f64(v).copy(), _f64(w).copy()
    nx, ny, nz = phi.shape
    _chk(lib().afid_ref_correct(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                                C.c_double(Lz), _p(phi), _p(u), _p(v), _p(w)), "afid_ref_correct")
    return u, v, w


def forward_spectrum(d):
    d = _f64(d)
    nx, ny, nz = d.shape
    out = np.empty((nx, ny, nz), dtype=np.complex128)
    _chk(lib().afid_ref_forward_spectrum(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(d), _p(out)),
         "afid_ref_forward_spectrum")
    return out


def inverse_spectrum(xhat):
    xhat = np.ascontiguousarray(xhat, dtype=np.complex128)
    nx, ny, nz = xhat.shape
    phi = np.empty((nx, ny, nz))
    mi = C.c_double(0.0)
    _chk(lib().afid_ref_inverse_spectrum(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xhat), _p(phi),
                                         C.byref(mi)), "afid_ref_inverse_spectrum")
    return phi, mi.value


def solve(xc, Ly, Lz, dhat):
    """Per-mode x-solves; returns a new complex array."""
    xc = _f64(xc)
    x = np.ascontiguousarray(dhat, dtype=np.complex128).copy()
    nx, ny, nz = x.shape
    _chk(lib().afid_ref_solve(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                              C.c_double(Lz), _p(x)), "afid_ref_solve")
    return x


def solve_one(xc, lam, rhs, singular=False):
    xc = _f64(xc)
    x = np.ascontiguousarray(rhs, dtype=np.complex128).copy()
    _chk(lib().afid_ref_solve_one(C.c_int(xc.size - 1), _p(xc), C.c_double(lam),
                                  C.c_int(1 if singular else 0), _p(x)), "afid_ref_solve_one")
    return x


def project(xc, Ly, Lz, u, v, w):
    """The whole step.  Returns (u, v, w, p, max_imag) as new arrays."""
    xc = _f64(xc)
    u, v, w = _f64(u).copy(), _f64(v).copy(), _f64(w).copy()
    nx, ny, nz = v.shape
    assert u.shape == (nx + 1, ny, nz) and w.shape == v.shape and xc.size == nx + 1
    p = np.empty((nx, ny, nz))
    mi = C.c_double(0.0)
    _chk(lib().afid_ref_project(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                                C.c_double(Lz), _p(u), _p(v), _p(w), _p(p), C.byref(mi)),
         "afid_ref_project")
    return u, v, w, p, mi.value


def solve_half(xc, Ly, Lz, nz, hhat):
    """Per-mode x-solves IN PLACE on a half spectrum [nx][ny][nz/2+1] (complex128, C-contiguous)."""
    xc = _f64(xc)
    assert isinstance(hhat, np.ndarray) and hhat.dtype == np.complex128 and hhat.flags.c_contiguous
    nx, ny, nzh = hhat.shape
    assert nzh == nz // 2 + 1 and xc.size == nx + 1
    _chk(lib().afid_ref_solve_half(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                                   C.c_double(Lz), _p(hhat)), "afid_ref_solve_half")
    return hhat


def max_cfl(xc, Ly, Lz, u, v, w):
    """Maximum CFL number of the paper's Listing 1, floor 1e-8."""
    xc, u, v, w = _f64(xc), _f64(u), _f64(v), _f64(w)
    nx, ny, nz = v.shape
    assert u.shape == (nx + 1, ny, nz) and w.shape == v.shape and xc.size == nx + 1
    out = C.c_double(0.0)
    _chk(lib().afid_ref_max_cfl(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(xc), C.c_double(Ly),
                                C.c_double(Lz), _p(u), _p(v), _p(w), C.byref(out)), "afid_ref_max_cfl")
    return out.value


def xsolve(a, c, lam, f):
    """Column-wise real tridiagonal solves in x of a field (nx, ny, nz); returns a new array."""
    a, c, lam = _f64(a), _f64(c), _f64(lam)
    x = _f64(f).copy()
    nx, ny, nz = x.shape
    assert a.size == nx and c.size == nx and lam.size == nx
    _chk(lib().afid_ref_xsolve(C.c_int(nx), C.c_int(ny), C.c_int(nz), _p(a), _p(c), _p(lam), _p(x)), "afid_ref_xsolve")
    return x
