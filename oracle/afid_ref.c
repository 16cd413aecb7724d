/*
 * afid_ref.c -- CPU ORACLE for the AFiD pressure-correction (projection) step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_1705_01423_b200/csrc/ and includes nothing from include/.
 *
 * Plain, slow, obviously-correct implementation written from the paper
 * (/root/reference/PAPER.md, "P:L<n>" = line n) and the readings R0..R18 listed in
 * DESIGN.md.  Everything is the definition written out:
 *
 *   - staggered, conservative, 2nd-order central differences (Fig. 1);
 *   - fractional step: provisional velocity -> Poisson equation for the correction phi
 *     -> velocity and pressure updated, velocity divergence-free;
 *   - Poisson solve by Fourier expansion in the two periodic directions with modified
 *     wavenumbers and one tridiagonal (Thomas) solve in x per mode,
 *     following the paper's step list minus the pencil transposes
 *     (one address space here, so steps 2,4,6,8,10,12 are no-ops);
 *   - the Fourier transforms are NAIVE O(n^2) DFT sums (no FFT, no library), each sum
 *     accumulated in long double; the tridiagonal recurrences run in long double.
 *
 * Array layout (all host pointers, C order, z fastest, 64-bit indexing):
 *   u : (nx+1)*ny*nz  u_x on x-faces   xc[i]            (planes 0 and nx are the walls)
 *   v :  nx   *ny*nz  u_y on y-faces   (xm_i, j*dy, (k+1/2)dz)
 *   w :  nx   *ny*nz  u_z on z-faces   (xm_i, (j+1/2)dy, k*dz)
 *   p :  nx   *ny*nz  cell centres
 *   complex arrays: interleaved (re,im) doubles, FULL spectrum [nx][ny][nz].
 *
 * Parity pins: tests/test_oracle_*.py (closed-form eigenfunction, manufactured
 * Helmholtz split, dense brute force on 4^3 / 8^3, invariants, numpy.fft / scipy
 * special cases).  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

#define IDX(i, j, k) ((((size_t)(i)) * (size_t)ny + (size_t)(j)) * (size_t)nz + (size_t)(k))

int afid_ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * Step 1 (R1,R4): metrics of the wall-normal grid from the nx+1 face
 * coordinates xc.  dx[i] = xc[i+1]-xc[i]  (cell width, i=0..nx-1);
 * dc[i] = (xc[i+1]-xc[i-1])/2 (distance between the centres of cells i-1 and i,
 * i=1..nx-1; dc[0] and dc[nx] are wall faces, unused, set to 0).
 * Each is one fp64 subtraction of the inputs (never a difference of midpoints).
 * Paper: non-uniform x grid, uniform periodic y,z.
 * ---------------------------------------------------------------------------------- */
int afid_ref_metrics(int nx, const double *xc, double *dx, double *dc)
{
    if (nx < 2 || !xc || !dx || !dc) return -1;
    for (int i = 0; i < nx; ++i) {
        dx[i] = xc[i + 1] - xc[i];
        if (!(dx[i] > 0.0)) return -2;
    }
    dc[0] = 0.0;
    dc[nx] = 0.0;
    for (int i = 1; i < nx; ++i) dc[i] = (xc[i + 1] - xc[i - 1]) / 2.0;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Paper step 1 ("Calculate the local divergence"), stencil P:L87:
 *   d = (u[i+1]-u[i])/dx_i + (v[j+1]-v[j])/dy + (w[k+1]-w[k])/dz, periodic in j,k.
 * ---------------------------------------------------------------------------------- */
int afid_ref_divergence(int nx, int ny, int nz, const double *xc, double Ly, double Lz,
                        const double *u, const double *v, const double *w, double *d)
{
    double *dx = (double *)malloc(sizeof(double) * (size_t)nx);
    double *dc = (double *)malloc(sizeof(double) * (size_t)(nx + 1));
    if (!dx || !dc) { free(dx); free(dc); return -3; }
    int rc = afid_ref_metrics(nx, xc, dx, dc);
    if (rc) { free(dx); free(dc); return rc; }
    const double dy = Ly / ny, dz = Lz / nz;
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j) {
            const int jp = (j + 1) % ny;
            for (int k = 0; k < nz; ++k) {
                const int kp = (k + 1) % nz;
                d[IDX(i, j, k)] = (u[IDX(i + 1, j, k)] - u[IDX(i, j, k)]) / dx[i]
                                + (v[IDX(i, jp, k)] - v[IDX(i, j, k)]) / dy
                                + (w[IDX(i, j, kp)] - w[IDX(i, j, k)]) / dz;
            }
        }
    free(dx); free(dc);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Velocity / pressure correction ("the corrected velocities and pressures are
 * computed directly"): u -= G phi with G the staggered gradient, zero on the
 * wall faces (Neumann); wall planes of u are not touched.
 *   u[i] -= (phi[i]-phi[i-1])/dc_i   (i=1..nx-1)
 *   v[j] -= (phi[j]-phi[j-1])/dy     (periodic)
 *   w[k] -= (phi[k]-phi[k-1])/dz     (periodic)
 * ---------------------------------------------------------------------------------- */
int afid_ref_correct(int nx, int ny, int nz, const double *xc, double Ly, double Lz,
                     const double *phi, double *u, double *v, double *w)
{
    double *dx = (double *)malloc(sizeof(double) * (size_t)nx);
    double *dc = (double *)malloc(sizeof(double) * (size_t)(nx + 1));
    if (!dx || !dc) { free(dx); free(dc); return -3; }
    int rc = afid_ref_metrics(nx, xc, dx, dc);
    if (rc) { free(dx); free(dc); return rc; }
    const double dy = Ly / ny, dz = Lz / nz;
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < nx; ++i)
        for (int j = 0; j < ny; ++j) {
            const int jm = (j + ny - 1) % ny;
            for (int k = 0; k < nz; ++k) {
                const int km = (k + nz - 1) % nz;
                const double ph = phi[IDX(i, j, k)];
                if (i >= 1) u[IDX(i, j, k)] -= (ph - phi[IDX(i - 1, j, k)]) / dc[i];
                v[IDX(i, j, k)] -= (ph - phi[IDX(i, jm, k)]) / dy;
                w[IDX(i, j, k)] -= (ph - phi[IDX(i, j, km)]) / dz;
            }
        }
    free(dx); free(dc);
    return 0;
}

/* Twiddle table exp(-2 pi i m / n), m = 0..n-1, long double.  Indices are always
 * reduced mod n in integers before the lookup (never sin of a large argument). */
static int make_twiddles(int n, ld **cs, ld **sn)
{
    *cs = (ld *)malloc(sizeof(ld) * (size_t)n);
    *sn = (ld *)malloc(sizeof(ld) * (size_t)n);
    if (!*cs || !*sn) return -3;
    const ld twopi = 2.0L * acosl(-1.0L);
    for (int m = 0; m < n; ++m) {
        (*cs)[m] = cosl(twopi * (ld)m / (ld)n);
        (*sn)[m] = -sinl(twopi * (ld)m / (ld)n);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * One naive DFT line of length n with stride `stride` (in complex elements):
 *   out[q] = sum_m in[m] * exp(sign * 2 pi i q m / n)      sign = -1 forward, +1 inverse
 * Unnormalised.  Accumulated in long double.  (the transforms;
 * evaluated as their definition, O(n^2).)
 * ---------------------------------------------------------------------------------- */
static void dft_line(int n, const double *in, size_t stride, double *out, int sign,
                     const ld *cs, const ld *sn)
{
    for (int q = 0; q < n; ++q) {
        ld sr = 0.0L, si = 0.0L;
        for (int m = 0; m < n; ++m) {
            const int t = (int)(((long long)q * (long long)m) % n);
            const ld c = cs[t];
            const ld s = (sign < 0) ? sn[t] : -sn[t];
            const ld xr = in[2 * stride * (size_t)m], xi = in[2 * stride * (size_t)m + 1];
            sr += xr * c - xi * s;
            si += xr * s + xi * c;
        }
        out[2 * stride * (size_t)q] = (double)sr;
        out[2 * stride * (size_t)q + 1] = (double)si;
    }
}

/* 2-D DFT over (j,k) of every x-plane of a complex array [nx][ny][nz], in -> out
 * (out may not alias in; `tmp` same size).  sign=-1: z lines then y lines (paper steps
 * 3,5 in our axis naming, R11: the order of the two directions is
 * unobservable); sign=+1: y lines then z lines (steps 9,11).  No scaling. */
static int dft2_planes(int nx, int ny, int nz, const double *in, double *tmp, double *out, int sign)
{
    ld *cy, *sy, *cz, *sz;
    if (make_twiddles(ny, &cy, &sy) || make_twiddles(nz, &cz, &sz)) return -3;
    if (sign < 0) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nx; ++i)
            for (int j = 0; j < ny; ++j)
                dft_line(nz, in + 2 * IDX(i, j, 0), 1, tmp + 2 * IDX(i, j, 0), sign, cz, sz);
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nx; ++i)
            for (int k = 0; k < nz; ++k)
                dft_line(ny, tmp + 2 * IDX(i, 0, k), (size_t)nz, out + 2 * IDX(i, 0, k), sign, cy, sy);
    } else {
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nx; ++i)
            for (int k = 0; k < nz; ++k)
                dft_line(ny, in + 2 * IDX(i, 0, k), (size_t)nz, tmp + 2 * IDX(i, 0, k), sign, cy, sy);
#pragma omp parallel for collapse(2) schedule(static)
        for (int i = 0; i < nx; ++i)
            for (int j = 0; j < ny; ++j)
                dft_line(nz, tmp + 2 * IDX(i, j, 0), 1, out + 2 * IDX(i, j, 0), sign, cz, sz);
    }
    free(cy); free(sy); free(cz); free(sz);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Forward spectrum (paper steps 3 and 5):
 *   dhat(i,ky,kz) = sum_j sum_k d(i,j,k) exp(-2 pi i (ky j/ny + kz k/nz)), all ky,kz.
 * d real [nx][ny][nz] -> dhat complex [nx][ny][nz] (interleaved).
 * ---------------------------------------------------------------------------------- */
int afid_ref_forward_spectrum(int nx, int ny, int nz, const double *d, double *dhat)
{
    const size_t N = (size_t)nx * ny * nz;
    double *a = (double *)malloc(sizeof(double) * 2 * N);
    double *b = (double *)malloc(sizeof(double) * 2 * N);
    if (!a || !b) { free(a); free(b); return -3; }
    for (size_t t = 0; t < N; ++t) { a[2 * t] = d[t]; a[2 * t + 1] = 0.0; }
    int rc = dft2_planes(nx, ny, nz, a, b, dhat, -1);
    free(a); free(b);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Inverse spectrum (paper steps 9 and 11):
 *   phi(i,j,k) = 1/(ny nz) sum_ky sum_kz xhat exp(+2 pi i (ky j/ny + kz k/nz)).
 * Returns the real part in phi; *max_imag receives max |imag part| (round-off only for
 * Hermitian input; the tests assert it is negligible).
 * ---------------------------------------------------------------------------------- */
int afid_ref_inverse_spectrum(int nx, int ny, int nz, const double *xhat, double *phi, double *max_imag)
{
    const size_t N = (size_t)nx * ny * nz;
    double *a = (double *)malloc(sizeof(double) * 2 * N);
    double *b = (double *)malloc(sizeof(double) * 2 * N);
    if (!a || !b) { free(a); free(b); return -3; }
    int rc = dft2_planes(nx, ny, nz, xhat, a, b, +1);
    if (!rc) {
        const ld scale = 1.0L / ((ld)ny * (ld)nz);
        double mi = 0.0;
        for (size_t t = 0; t < N; ++t) {
            phi[t] = (double)((ld)b[2 * t] * scale);
            const double im = fabs((double)((ld)b[2 * t + 1] * scale));
            if (im > mi) mi = im;
        }
        if (max_imag) *max_imag = mi;
    }
    free(a); free(b);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Modified wavenumbers (formula from BASELINE.json north_star):
 *   lam(q) = 2 (1 - cos(2 pi q / n)) / Delta^2,  Delta = L/n, q = 0..n-1
 * evaluated as 4 sin^2(pi q / n) / Delta^2 (identical value, no cancellation at small q)
 * in long double, rounded to fp64.  -lam is the eigenvalue of the periodic second
 * difference for the mode exp(2 pi i q j / n).
 * ---------------------------------------------------------------------------------- */
int afid_ref_wavenumbers(int n, double L, double *lam)
{
    if (n < 1 || !(L > 0.0) || !lam) return -1;
    const ld pi = acosl(-1.0L);
    const ld delta = (ld)L / (ld)n;
    for (int q = 0; q < n; ++q) {
        const ld s = sinl(pi * (ld)q / (ld)n);
        lam[q] = (double)(4.0L * s * s / (delta * delta));
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * One x-system (paper step 7, "tridiagonal Thomas solver"):
 *   a_i x_{i-1} - (a_i + c_i + lam) x_i + c_i x_{i+1} = rhs_i ,  i = 0..nx-1
 *   a_i = 1/(dx_i dc_i) (a_0 = 0),  c_i = 1/(dx_i dc_{i+1}) (c_{nx-1} = 0)   [Neumann walls]
 * real matrix, complex rhs (stride in complex elements), solution overwrites rhs.
 * Thomas elimination written in the cancellation-free form of DESIGN.md R9:
 *   s_0 = lam; pi_i = c_i + s_i; y_i = (-rhs_i + a_i y_{i-1})/pi_i; g_i = c_i/pi_i;
 *   s_{i+1} = lam + a_{i+1} s_i/pi_i;   back: x_{n-1} = y_{n-1}, x_i = y_i + g_i x_{i+1}
 * (pi_i is the Thomas pivot -(b_i - a_i g_{i-1}) with b_i = -(a_i+c_i+lam); s_i is the
 * part of it that does not cancel).  All in long double.
 * singular != 0 (the lam = 0 mean mode, R7): the last pivot is exactly 0; pin
 * x_{n-1} := 0 (drop the last, redundant equation), back-substitute, then subtract the
 * dx-weighted mean so that sum_i x_i dx_i = 0.
 * ---------------------------------------------------------------------------------- */
static void solve_x_system(int nx, const ld *a, const ld *c, const double *dx, ld lam,
                           int singular, double *rhs, size_t stride, ld *yr, ld *yi, ld *g)
{
    ld s = lam;
    ld pr = 0.0L, pi_ = 0.0L; /* y_{i-1} */
    for (int i = 0; i < nx; ++i) {
        const ld piv = c[i] + s;
        const ld rr = -(ld)rhs[2 * stride * (size_t)i], ri = -(ld)rhs[2 * stride * (size_t)i + 1];
        if (singular && i == nx - 1) { /* piv == 0: pinned */
            yr[i] = 0.0L; yi[i] = 0.0L; g[i] = 0.0L;
            break;
        }
        yr[i] = (rr + a[i] * pr) / piv;
        yi[i] = (ri + a[i] * pi_) / piv;
        g[i] = c[i] / piv;
        if (i + 1 < nx) s = lam + a[i + 1] * (s / piv);
        pr = yr[i]; pi_ = yi[i];
    }
    ld xr = yr[nx - 1], xi = yi[nx - 1];
    for (int i = nx - 2; i >= 0; --i) {
        yr[i] = yr[i] + g[i] * xr;
        yi[i] = yi[i] + g[i] * xi;
        xr = yr[i]; xi = yi[i];
    }
    if (singular) {
        ld mr = 0.0L, mi = 0.0L, vol = 0.0L;
        for (int i = 0; i < nx; ++i) { mr += yr[i] * (ld)dx[i]; mi += yi[i] * (ld)dx[i]; vol += (ld)dx[i]; }
        mr /= vol; mi /= vol;
        for (int i = 0; i < nx; ++i) { yr[i] -= mr; yi[i] -= mi; }
    }
    for (int i = 0; i < nx; ++i) {
        rhs[2 * stride * (size_t)i] = (double)yr[i];
        rhs[2 * stride * (size_t)i + 1] = (double)yi[i];
    }
}

/* Exposed single-system solve for the tests (pin P5: scipy.linalg.solve_banded). */
int afid_ref_solve_one(int nx, const double *xc, double lam, int singular, double *rhs_complex)
{
    double *dx = (double *)malloc(sizeof(double) * (size_t)nx);
    double *dc = (double *)malloc(sizeof(double) * (size_t)(nx + 1));
    ld *a = (ld *)malloc(sizeof(ld) * (size_t)nx), *c = (ld *)malloc(sizeof(ld) * (size_t)nx);
    ld *yr = (ld *)malloc(sizeof(ld) * (size_t)nx), *yi = (ld *)malloc(sizeof(ld) * (size_t)nx);
    ld *g = (ld *)malloc(sizeof(ld) * (size_t)nx);
    int rc = (!dx || !dc || !a || !c || !yr || !yi || !g) ? -3 : afid_ref_metrics(nx, xc, dx, dc);
    if (!rc) {
        for (int i = 0; i < nx; ++i) {
            a[i] = (i >= 1) ? 1.0L / ((ld)dx[i] * (ld)dc[i]) : 0.0L;
            c[i] = (i <= nx - 2) ? 1.0L / ((ld)dx[i] * (ld)dc[i + 1]) : 0.0L;
        }
        solve_x_system(nx, a, c, dx, (ld)lam, singular, rhs_complex, 1, yr, yi, g);
    }
    free(dx); free(dc); free(a); free(c); free(yr); free(yi); free(g);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Paper step 7 for every mode: xhat(:,ky,kz) solves the x-system with
 * lam = lam_y(ky) + lam_z(kz) and rhs = dhat(:,ky,kz); in place on the complex array.
 * Mode (0,0) is the singular one (pinned, zero dx-weighted mean).
 * ---------------------------------------------------------------------------------- */
int afid_ref_solve(int nx, int ny, int nz, const double *xc, double Ly, double Lz, double *dhat)
{
    double *dx = (double *)malloc(sizeof(double) * (size_t)nx);
    double *dc = (double *)malloc(sizeof(double) * (size_t)(nx + 1));
    double *ly = (double *)malloc(sizeof(double) * (size_t)ny);
    double *lz = (double *)malloc(sizeof(double) * (size_t)nz);
    ld *a = (ld *)malloc(sizeof(ld) * (size_t)nx), *c = (ld *)malloc(sizeof(ld) * (size_t)nx);
    int rc = (!dx || !dc || !ly || !lz || !a || !c) ? -3 : afid_ref_metrics(nx, xc, dx, dc);
    if (!rc) rc = afid_ref_wavenumbers(ny, Ly, ly);
    if (!rc) rc = afid_ref_wavenumbers(nz, Lz, lz);
    if (!rc) {
        for (int i = 0; i < nx; ++i) {
            a[i] = (i >= 1) ? 1.0L / ((ld)dx[i] * (ld)dc[i]) : 0.0L;
            c[i] = (i <= nx - 2) ? 1.0L / ((ld)dx[i] * (ld)dc[i + 1]) : 0.0L;
        }
        const size_t stride = (size_t)ny * (size_t)nz;
#pragma omp parallel
        {
            ld *yr = (ld *)malloc(sizeof(ld) * (size_t)nx), *yi = (ld *)malloc(sizeof(ld) * (size_t)nx);
            ld *g = (ld *)malloc(sizeof(ld) * (size_t)nx);
#pragma omp for collapse(2) schedule(static)
            for (int j = 0; j < ny; ++j)
                for (int k = 0; k < nz; ++k) {
                    const ld lam = (ld)ly[j] + (ld)lz[k];
                    solve_x_system(nx, a, c, dx, lam, (j == 0 && k == 0), dhat + 2 * IDX(0, j, k),
                                   stride, yr, yi, g);
                }
            free(yr); free(yi); free(g);
        }
    }
    free(dx); free(dc); free(ly); free(lz); free(a); free(c);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * The whole step (R0): phi solves D G phi = D u* with zero
 * dx-weighted mean; u <- u* - G phi; p = phi (output only, R6).
 * u,v,w are updated in place; p is written.  max_imag (may be NULL) as above.
 * ---------------------------------------------------------------------------------- */
int afid_ref_project(int nx, int ny, int nz, const double *xc, double Ly, double Lz,
                     double *u, double *v, double *w, double *p, double *max_imag)
{
    if (nx < 2 || ny < 1 || nz < 1 || !xc || !(Ly > 0.0) || !(Lz > 0.0) || !u || !v || !w || !p) return -1;
    const size_t N = (size_t)nx * ny * nz;
    double *d = (double *)malloc(sizeof(double) * N);
    double *dhat = (double *)malloc(sizeof(double) * 2 * N);
    if (!d || !dhat) { free(d); free(dhat); return -3; }
    int rc = afid_ref_divergence(nx, ny, nz, xc, Ly, Lz, u, v, w, d);
    if (!rc) rc = afid_ref_forward_spectrum(nx, ny, nz, d, dhat);
    if (!rc) rc = afid_ref_solve(nx, ny, nz, xc, Ly, Lz, dhat);
    if (!rc) rc = afid_ref_inverse_spectrum(nx, ny, nz, dhat, p, max_imag);
    if (!rc) rc = afid_ref_correct(nx, ny, nz, xc, Ly, Lz, p, u, v, w);
    free(d); free(dhat);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Paper step 7 on a HALF spectrum [nx][ny][nz/2+1] (kz = 0..nz/2): the x-systems of the
 * large-case oracle oracle/ref_dense.py, which keeps only the
 * non-redundant half of the Hermitian spectrum of the real divergence.  Same long-double
 * Thomas recurrences, same singular-mode handling as afid_ref_solve.  nz must be even.
 * ---------------------------------------------------------------------------------- */
int afid_ref_solve_half(int nx, int ny, int nz, const double *xc, double Ly, double Lz, double *hhat)
{
    if (nx < 2 || ny < 1 || nz < 2 || (nz & 1) || !xc || !hhat) return -1;
    const int nzh = nz / 2 + 1;
    double *dx = (double *)malloc(sizeof(double) * (size_t)nx);
    double *dc = (double *)malloc(sizeof(double) * (size_t)(nx + 1));
    double *ly = (double *)malloc(sizeof(double) * (size_t)ny);
    double *lz = (double *)malloc(sizeof(double) * (size_t)nz);
    ld *a = (ld *)malloc(sizeof(ld) * (size_t)nx), *c = (ld *)malloc(sizeof(ld) * (size_t)nx);
    int rc = (!dx || !dc || !ly || !lz || !a || !c) ? -3 : afid_ref_metrics(nx, xc, dx, dc);
    if (!rc) rc = afid_ref_wavenumbers(ny, Ly, ly);
    if (!rc) rc = afid_ref_wavenumbers(nz, Lz, lz);
    if (!rc) {
        for (int i = 0; i < nx; ++i) {
            a[i] = (i >= 1) ? 1.0L / ((ld)dx[i] * (ld)dc[i]) : 0.0L;
            c[i] = (i <= nx - 2) ? 1.0L / ((ld)dx[i] * (ld)dc[i + 1]) : 0.0L;
        }
        const size_t stride = (size_t)ny * (size_t)nzh;
#pragma omp parallel
        {
            ld *yr = (ld *)malloc(sizeof(ld) * (size_t)nx), *yi = (ld *)malloc(sizeof(ld) * (size_t)nx);
            ld *g = (ld *)malloc(sizeof(ld) * (size_t)nx);
#pragma omp for collapse(2) schedule(static)
            for (int j = 0; j < ny; ++j)
                for (int q = 0; q < nzh; ++q) {
                    const ld lam = (ld)ly[j] + (ld)lz[q];
                    solve_x_system(nx, a, c, dx, lam, (j == 0 && q == 0),
                                   hhat + 2 * ((size_t)j * (size_t)nzh + (size_t)q), stride, yr, yi, g);
                }
            free(yr); free(yi); free(g);
        }
    }
    free(dx); free(dc); free(ly); free(lz); free(a); free(c);
    return rc;
}

/* ------------------------------------------------------------------------------------
 * the maximum CFL number, the one routine the paper prints in full
 * (Listing 1 "CalcMaxCFL"):
 *     cflm = max( 1e-8, max over cells of
 *                 0.5 * ( |vz(i) + vz(i+1)| * dz + |vy(j) + vy(j+1)| * dy + |vx(k) + vx(k+1)| * udx3m(k) ) )
 * In AFiD dz, dy and udx3m are INVERSE spacings (R20); in this file's notation
 * (u wall-normal on x-faces, v, w periodic):
 *     q(i,j,k) = |w(i,j,k) + w(i,j,k+1)| / dz + |v(i,j,k) + v(i,j+1,k)| / dy + |u(i,j,k) + u(i+1,j,k)| / dx_i
 * with periodic wrap in j and k.  Plain loops, fp64, the paper's order of operations.
 * ------------------------------------------------------------------------------------ */
int afid_ref_max_cfl(int nx, int ny, int nz, const double *xc, double Ly, double Lz,
                     const double *u, const double *v, const double *w, double *cflm)
{
    if (nx < 1 || ny < 1 || nz < 1 || !xc || !u || !v || !w || !cflm) return -1;
    const double rdy = (double)ny / Ly, rdz = (double)nz / Lz;
    double best = 0.00000001;
    for (int i = 0; i < nx; ++i) {
        const double udx = 1.0 / (xc[i + 1] - xc[i]);
        for (int j = 0; j < ny; ++j) {
            const int jp = (j + 1) % ny;
            for (int k = 0; k < nz; ++k) {
                const int kp = (k + 1) % nz;
                const double qcf = fabs((w[IDX(i, j, k)] + w[IDX(i, j, kp)]) * rdz)
                                 + fabs((v[IDX(i, j, k)] + v[IDX(i, jp, k)]) * rdy)
                                 + fabs((u[IDX(i, j, k)] + u[IDX(i + 1, j, k)]) * udx);
                if (qcf * 0.5 > best) best = qcf * 0.5;
            }
        }
    }
    *cflm = best;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * batched real tridiagonal solves in x on a field f[i][j][k], in place -- the
 * implicit wall-normal step of the time integrator ("batched tridiagonal solvers ...
 * each thread in a block solves a system").  For every column (j,k):
 *     -a_i x_{i-1} + (a_i + c_i + lam_i) x_i - c_i x_{i+1} = f_i ,  i = 0..nx-1,  a_0 := 0, c_{nx-1} := 0.
 * Textbook Thomas algorithm (forward elimination, back substitution) in long double, one column at a time.
 * ------------------------------------------------------------------------------------ */
int afid_ref_xsolve(int nx, int ny, int nz, const double *a, const double *c, const double *lam, double *f)
{
    if (nx < 1 || ny < 1 || nz < 1 || !a || !c || !lam || !f) return -1;
    int rc = 0;
#pragma omp parallel
    {
        ld *cp = (ld *)malloc(sizeof(ld) * (size_t)nx);
        ld *dp = (ld *)malloc(sizeof(ld) * (size_t)nx);
        if (!cp || !dp) {
#pragma omp critical
            rc = -3;
        } else {
#pragma omp for collapse(2) schedule(static)
            for (int j = 0; j < ny; ++j)
                for (int k = 0; k < nz; ++k) {
                    for (int i = 0; i < nx; ++i) {
                        const ld sub = (i == 0) ? 0.0L : -(ld)a[i];
                        const ld sup = (i == nx - 1) ? 0.0L : -(ld)c[i];
                        const ld diag = ((i == 0) ? 0.0L : (ld)a[i]) + ((i == nx - 1) ? 0.0L : (ld)c[i]) + (ld)lam[i];
                        const ld den = (i == 0) ? diag : diag - sub * cp[i - 1];
                        cp[i] = sup / den;
                        dp[i] = ((ld)f[IDX(i, j, k)] - ((i == 0) ? 0.0L : sub * dp[i - 1])) / den;
                    }
                    ld x = dp[nx - 1];
                    f[IDX(nx - 1, j, k)] = (double)x;
                    for (int i = nx - 2; i >= 0; --i) {
                        x = dp[i] - cp[i] * x;
                        f[IDX(i, j, k)] = (double)x;
                    }
                }
        }
        free(cp); free(dp);
    }
    return rc;
}
