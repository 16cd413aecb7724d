"""Manufactured discrete Helmholtz split (pin P2 of the oracle, reused as a full-size GPU check).

Test helper, torch ops only; it shares nothing with the CUDA path or with oracle/.

For ARBITRARY arrays psi[nx][ny][nz], chi[nx+1][ny][nz] (chi = 0 on the two wall planes) and
phi[nx][ny][nz] the staggered operators of P:L87 satisfy identically (exact arithmetic):

    u_sol =  d_y chi / dy                       (x-faces; 0 on the walls)
    v_sol = -d_x chi / dx_i + d_z psi / dz
    w_sol = -d_y psi / dy
    D(u_sol, v_sol, w_sol) = 0

so the projection of  u* = u_sol + G phi  must return exactly (u_sol, phi) when phi has zero
dx-weighted mean: the expected output is known by construction at any grid size.
"""
import numpy as np
import torch

from paper_1705_01423_b200 import synth


def _field(cfg, xc, comp, seed, device):
    """An arbitrary seeded smooth-plus-noise array shaped like velocity component `comp`."""
    c = dict(cfg)
    c.update(seed=seed, sigma=max(cfg.get("sigma", 0.0), 1e-2), shear=0.0, A=1.0)
    nx, ny, nz = c["nx"], c["ny"], c["nz"]
    shape = (nx + 1, ny, nz) if comp == 0 else (nx, ny, nz)
    f = torch.empty(shape, dtype=torch.float64, device=device)
    xc_t = torch.as_tensor(np.asarray(xc, dtype=np.float64)).to(device)
    chunk = max(1, (1 << 24) // (ny * nz))
    for i0, i1, blk in synth._component(c, xc_t, comp, torch.device(device), chunk):
        f[i0:i1] = blk
    if comp == 0:
        f[0].zero_()
        f[nx].zero_()
    return f


def _metrics(xc, device):
    xc_t = torch.as_tensor(np.asarray(xc, dtype=np.float64)).to(device)
    dx = xc_t[1:] - xc_t[:-1]
    dc = (xc_t[2:] - xc_t[:-2]) / 2.0  # faces 1..nx-1
    return dx, dc


def potentials(cfg, xc, device, seed=1000):
    """(phi, psi, chi): phi has zero dx-weighted mean."""
    dx, _ = _metrics(xc, device)
    phi = _field(cfg, xc, 2, seed + 3, device)
    wsum = torch.zeros((), dtype=torch.float64, device=device)
    for i in range(phi.shape[0]):  # plane by plane: no full-size temporaries
        wsum += phi[i].sum() * dx[i]
    phi -= wsum / (dx.sum() * phi.shape[1] * phi.shape[2])
    psi = _field(cfg, xc, 1, seed + 1, device)
    chi = _field(cfg, xc, 0, seed + 2, device)
    return phi, psi, chi


def solenoidal_into(cfg, xc, psi, chi, u, v, w):
    """Write (u_sol, v_sol, w_sol) into preallocated u (nx+1 planes), v, w; plane by plane."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dy, dz = cfg["Ly"] / ny, cfg["Lz"] / nz
    dx, _ = _metrics(xc, u.device)
    for i in range(nx + 1):
        u[i] = (torch.roll(chi[i], -1, 0) - chi[i]) / dy
    for i in range(nx):
        v[i] = -(chi[i + 1] - chi[i]) / dx[i] + (torch.roll(psi[i], -1, 1) - psi[i]) / dz
        w[i] = -(torch.roll(psi[i], -1, 0) - psi[i]) / dy


def add_gradient(cfg, xc, phi, u, v, w):
    """u += G phi (interior faces only), v += d_y phi / dy, w += d_z phi / dz; plane by plane."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dy, dz = cfg["Ly"] / ny, cfg["Lz"] / nz
    _, dc = _metrics(xc, u.device)
    for i in range(nx):
        if i >= 1:
            u[i] += (phi[i] - phi[i - 1]) / dc[i - 1]
        v[i] += (phi[i] - torch.roll(phi[i], 1, 0)) / dy
        w[i] += (phi[i] - torch.roll(phi[i], 1, 1)) / dz


def max_abs_divergence(cfg, xc, u, v, w):
    """max |D(u,v,w)| with torch ops (P:L87 stencil), plane by plane."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    dy, dz = cfg["Ly"] / ny, cfg["Lz"] / nz
    dx, _ = _metrics(xc, u.device)
    m = torch.zeros((), dtype=torch.float64, device=u.device)
    for i in range(nx):
        d = (u[i + 1] - u[i]) / dx[i] + (torch.roll(v[i], -1, 0) - v[i]) / dy + (torch.roll(w[i], -1, 1) - w[i]) / dz
        m = torch.maximum(m, d.abs().max())
    return float(m)


def rel_l2(a, b):
    """||a-b||_2 / ||b||_2 accumulated plane by plane (a, b same-shape 3-D tensors)."""
    num = torch.zeros((), dtype=torch.float64, device=a.device)
    den = torch.zeros((), dtype=torch.float64, device=a.device)
    for i in range(a.shape[0]):
        num += ((a[i] - b[i]) ** 2).sum()
        den += (b[i] ** 2).sum()
    return float(torch.sqrt(num / den))
