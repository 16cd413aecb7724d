"""Pins of the oracle's batched real x-solve: library banded solver, dense solve, and the
closed-form eigenfunctions of the uniform Neumann and Dirichlet operators."""
import numpy as np
import scipy.linalg

from oracle import ref


def dense(a, c, lam):
    nx = a.size
    A = np.zeros((nx, nx))
    for i in range(nx):
        ai = 0.0 if i == 0 else a[i]
        ci = 0.0 if i == nx - 1 else c[i]
        A[i, i] = ai + ci + lam[i]
        if i > 0:
            A[i, i - 1] = -ai
        if i < nx - 1:
            A[i, i + 1] = -ci
    return A


def random_system(nx, rng):
    a = rng.uniform(0.1, 50.0, nx) * 10.0 ** rng.integers(-2, 3, nx)
    c = rng.uniform(0.1, 50.0, nx) * 10.0 ** rng.integers(-2, 3, nx)
    lam = rng.uniform(1e-3, 5.0, nx)
    return a, c, lam


def test_matches_dense_solve():
    rng = np.random.default_rng(11)
    for nx in (1, 2, 3, 17):
        a, c, lam = random_system(nx, rng)
        f = rng.standard_normal((nx, 3, 4))
        x = ref.xsolve(a, c, lam, f)
        want = np.linalg.solve(dense(a, c, lam), f.reshape(nx, -1)).reshape(f.shape)
        assert np.abs(x - want).max() <= 1e-12 * np.abs(want).max()


def test_matches_scipy_banded():
    rng = np.random.default_rng(12)
    nx = 200
    a, c, lam = random_system(nx, rng)
    f = rng.standard_normal((nx, 2, 5))
    ab = np.zeros((3, nx))
    ab[0, 1:] = -c[:-1]
    ab[1] = np.r_[0.0, a[1:]] + np.r_[c[:-1], 0.0] + lam
    ab[2, :-1] = -a[1:]
    want = scipy.linalg.solve_banded((1, 1), ab, f.reshape(nx, -1)).reshape(f.shape)
    x = ref.xsolve(a, c, lam, f)
    assert np.abs(x - want).max() <= 1e-11 * np.abs(want).max()


def test_neumann_eigenfunctions_closed_form():
    """a = c = kappa (a_0, c_last dropped): cos(pi m (i+1/2)/nx) is an eigenvector of the zero-flux operator
    with eigenvalue 2 kappa (1 - cos(pi m/nx)); so x = f / (lam + that)."""
    nx, kappa, lam0 = 48, 7.5, 0.3
    a = np.full(nx, kappa); c = np.full(nx, kappa); lam = np.full(nx, lam0)
    i = np.arange(nx)
    for m in (0, 1, 5, 47):
        e = np.cos(np.pi * m * (i + 0.5) / nx)
        f = np.broadcast_to(e[:, None, None], (nx, 2, 2)).copy()
        x = ref.xsolve(a, c, lam, f)
        want = f / (lam0 + 2 * kappa * (1 - np.cos(np.pi * m / nx)))
        assert np.abs(x - want).max() <= 1e-13 * np.abs(want).max()


def test_dirichlet_eigenfunctions_closed_form():
    """Cell-centred Dirichlet walls by ghost cells: the wall rows get 2 kappa more on the diagonal (folded into
    lam_0, lam_last); sin(pi m (i+1/2)/nx) is then an eigenvector with eigenvalue 2 kappa (1 - cos(pi m/nx))."""
    nx, kappa, lam0 = 40, 3.0, 1.7
    a = np.full(nx, kappa); c = np.full(nx, kappa); lam = np.full(nx, lam0)
    lam[0] += 2 * kappa; lam[-1] += 2 * kappa
    i = np.arange(nx)
    for m in (1, 2, 9, 40):
        e = np.sin(np.pi * m * (i + 0.5) / nx)
        f = np.broadcast_to(e[:, None, None], (nx, 1, 3)).copy()
        x = ref.xsolve(a, c, lam, f)
        want = f / (lam0 + 2 * kappa * (1 - np.cos(np.pi * m / nx)))
        assert np.abs(x - want).max() <= 1e-13 * np.abs(want).max()


def test_columns_are_independent_and_linear():
    rng = np.random.default_rng(13)
    nx = 33
    a, c, lam = random_system(nx, rng)
    f = rng.standard_normal((nx, 4, 6)); g = rng.standard_normal((nx, 4, 6))
    x, y = ref.xsolve(a, c, lam, f), ref.xsolve(a, c, lam, g)
    z = ref.xsolve(a, c, lam, 2 * f - 3 * g)
    assert np.abs(z - (2 * x - 3 * y)).max() <= 1e-12 * np.abs(z).max()
    f2 = f.copy(); f2[:, 1, 2] += 1.0                       # touching one column changes only that column
    x2 = ref.xsolve(a, c, lam, f2)
    d = np.abs(x2 - x); d[:, 1, 2] = 0.0
    assert d.max() == 0.0
