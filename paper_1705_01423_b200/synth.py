"""Seeded synthetic inputs for the projection step.

This module holds NONE of the method's arithmetic (no divergence, transform, solve or
correction): it only builds wall-normal grids and velocity fields.  It is the one module
that serves both the CUDA path and the CPU oracle: callers generate an array ONCE and hand
the same bytes to both sides.  It stands in for the paper's Rayleigh-Benard and plane
Couette DNS fields (Tables 3-4), which are not available.

Everything is written with torch ops so the same recipe runs on the CPU (small configs)
and on the GPU (C3-C5, where a field is 4-19 GB).  Random numbers come from a stateless
counter-based generator (splitmix64 of (seed, stream, counter)), so any plane can be
regenerated independently.
"""
import math

import numpy as np
import torch

# The five BASELINE.json configs.
CONFIGS = {
    "C1": dict(nx=32, ny=32, nz=32, grid="uniform", s=0.0, x_lo=0.0, x_hi=1.0, Ly=1.0, Lz=1.0,
               M=8, expo=0.0, A=1.0, sigma=1e-2, shear=0.0, seed=0),
    "C2": dict(nx=256, ny=256, nz=256, grid="tanh", s=3.0, x_lo=0.0, x_hi=1.0, Ly=1.0, Lz=1.0,
               M=8, expo=0.0, A=1.0, sigma=1e-2, shear=0.0, seed=0),
    "C3": dict(nx=512, ny=1024, nz=1024, grid="tanh", s=3.0, x_lo=0.0, x_hi=1.0, Ly=2.0, Lz=2.0,
               M=32, expo=-5.0 / 6.0, A=1.0, sigma=0.0, shear=0.0, seed=0),
    "C4": dict(nx=1024, ny=1536, nz=1536, grid="tanh", s=3.0, x_lo=0.0, x_hi=1.0, Ly=1.5, Lz=1.5,
               M=32, expo=-5.0 / 6.0, A=1.0, sigma=1e-3, shear=0.0, seed=0),
    "C5": dict(nx=384, ny=4096, nz=1024, grid="erf", s=1.5, x_lo=-1.0, x_hi=1.0,
               Ly=8.0 * math.pi, Lz=2.0 * math.pi,
               M=32, expo=-5.0 / 6.0, A=0.1, sigma=0.0, shear=1.0, seed=0),
}


def config(name, **overrides):
    cfg = dict(CONFIGS[name])
    cfg.update(overrides)
    cfg["name"] = name
    return cfg


def grid_faces(cfg):
    """nx+1 face coordinates xc (numpy fp64), strictly increasing, walls exact.

    uniform: x = lo + (hi-lo) xi;  tanh(s): x = lo + (hi-lo)/2 [1 + tanh(s(xi-1/2))/tanh(s/2)];
    erf(s):  x = mid + (hi-lo)/2 erf(s(2xi-1))/erf(s);   xi = i/nx.
    """
    nx, lo, hi, s = cfg["nx"], cfg["x_lo"], cfg["x_hi"], cfg["s"]
    xi = np.arange(nx + 1, dtype=np.longdouble) / np.longdouble(nx)
    kind = cfg["grid"]
    if kind == "uniform":
        x01 = xi
    elif kind == "tanh":
        x01 = 0.5 * (1.0 + np.tanh(np.longdouble(s) * (xi - 0.5)) / np.tanh(np.longdouble(s) / 2))
    elif kind == "erf":
        e = np.array([math.erf(float(s) * (2.0 * float(t) - 1.0)) for t in xi]) / math.erf(float(s))
        x01 = 0.5 * (1.0 + e.astype(np.longdouble))
    else:
        raise ValueError(kind)
    xc = (np.longdouble(lo) + np.longdouble(hi - lo) * x01).astype(np.float64)
    xc[0], xc[-1] = lo, hi
    assert np.all(np.diff(xc) > 0)
    return xc


# ---- counter-based RNG: splitmix64 on int64 tensors (wrap-around arithmetic) -----------------
def _i64(c):
    c &= (1 << 64) - 1
    return c - (1 << 64) if c >= (1 << 63) else c


_GOLD = _i64(0x9E3779B97F4A7C15)
_M1 = _i64(0xBF58476D1CE4E5B9)
_M2 = _i64(0x94D049BB133111EB)


def _lsr(z, s):
    return (z >> s) & ((1 << (64 - s)) - 1)


def _splitmix64(x):
    z = x + _GOLD
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    return z ^ _lsr(z, 31)


def _key(seed, stream):
    k = torch.tensor([_i64(seed * 0x632BE59BD9B4E019 + stream * 0xD1342543DE82EF95 + 0x1234567)],
                     dtype=torch.int64)
    return int(_splitmix64(k)[0])


def uniform01(seed, stream, counter):
    """U(0,1) doubles, strictly inside (0,1), from int64 counter tensor."""
    z = _splitmix64(counter * _GOLD + _key(seed, stream))
    return (_lsr(z, 11).to(torch.float64) + 0.5) * (2.0 ** -53)


def normal(seed, stream, counter):
    """N(0,1) by Box-Muller from counters 2c and 2c+1."""
    u1 = uniform01(seed, stream, 2 * counter)
    u2 = uniform01(seed, stream, 2 * counter + 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def mode_table(cfg, comp):
    """Per-component random Fourier modes: integer (q,r,p), amplitude g*kappa^expo, phase."""
    M, ny, nz, seed = cfg["M"], cfg["ny"], cfg["nz"], cfg["seed"]
    K = max(1, min(ny, nz) // 8)
    c = torch.arange(M, dtype=torch.int64)
    st = 100 + 10 * comp
    q = torch.floor(uniform01(seed, st + 0, c) * (2 * K + 1)).to(torch.int64) - K
    r = torch.floor(uniform01(seed, st + 1, c) * (2 * K + 1)).to(torch.int64) - K
    p = torch.floor(uniform01(seed, st + 2, c) * 9).to(torch.int64)
    g = normal(seed, st + 3, c)
    th = 2.0 * math.pi * uniform01(seed, st + 4, c)
    kappa = torch.clamp(torch.sqrt((q * q + r * r + p * p).to(torch.float64)), min=1.0)
    amp = g * kappa ** cfg["expo"]
    return q, r, p, amp, th


def _component(cfg, xc_t, comp, device, chunk):
    """Generator of (i0, i1, block) x-chunks of one velocity component (0:u, 1:v, 2:w)."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    Ly, Lz, lo, hi = cfg["Ly"], cfg["Lz"], cfg["x_lo"], cfg["x_hi"]
    Lx = hi - lo
    f64 = torch.float64
    q, r, p, amp, th = [t.to(device) for t in mode_table(cfg, comp)]
    jj = torch.arange(ny, dtype=f64, device=device)
    kk = torch.arange(nz, dtype=f64, device=device)
    # staggered locations (Fig. 1): u,w at y-centres; u,v at z-centres
    Y = (jj + (0.0 if comp == 1 else 0.5)) * (Ly / ny)
    Z = (kk + (0.0 if comp == 2 else 0.5)) * (Lz / nz)
    if comp == 0:
        X = xc_t
    else:
        X = 0.5 * (xc_t[:-1] + xc_t[1:])
    nplanes = X.numel()
    ay = 2.0 * math.pi * q.to(f64)[:, None] * (Y / Ly)[None, :] + th[:, None]   # [M, ny]
    az = 2.0 * math.pi * r.to(f64)[:, None] * (Z / Lz)[None, :]                 # [M, nz]
    # cos(ay+az+ax) = cos(ay+az) cos(ax) - sin(ay+az) sin(ax)
    cyz = (torch.cos(ay)[:, :, None] * torch.cos(az)[:, None, :]
           - torch.sin(ay)[:, :, None] * torch.sin(az)[:, None, :]).reshape(cfg["M"], ny * nz)
    syz = (torch.sin(ay)[:, :, None] * torch.cos(az)[:, None, :]
           + torch.cos(ay)[:, :, None] * torch.sin(az)[:, None, :]).reshape(cfg["M"], ny * nz)
    B = torch.cat([cyz, syz], dim=0)                                             # [2M, ny*nz]
    for i0 in range(0, nplanes, chunk):
        i1 = min(nplanes, i0 + chunk)
        Xc = X[i0:i1]
        ax = math.pi * p.to(f64)[None, :] * ((Xc - lo) / Lx)[:, None]            # [c, M]
        damp = torch.sin(math.pi * (Xc - lo) / Lx)[:, None]
        Acoef = torch.cat([torch.cos(ax) * amp[None, :], -torch.sin(ax) * amp[None, :]], dim=1)
        blk = (cfg["A"] * damp * Acoef) @ B                                       # [c, ny*nz]
        if cfg["sigma"] != 0.0:
            idx = torch.arange(i0 * ny * nz, i1 * ny * nz, dtype=torch.int64, device=device)
            blk += cfg["sigma"] * normal(cfg["seed"], 200 + comp, idx).reshape(i1 - i0, ny * nz)
        if comp == 1 and cfg["shear"] != 0.0:
            blk += cfg["shear"] * Xc[:, None]
        yield i0, i1, blk.reshape(i1 - i0, ny, nz)


def velocity(cfg, xc, device="cpu", chunk=None, out=None):
    """Provisional velocity (u, v, w) as torch fp64 tensors on `device`.

    u: (nx+1, ny, nz) with both wall planes exactly 0;  v, w: (nx, ny, nz).
    `out` may hold three preallocated tensors to fill in place.
    """
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    device = torch.device(device)
    xc_t = torch.as_tensor(np.asarray(xc, dtype=np.float64)).to(device)
    if chunk is None:
        chunk = max(1, min(nx + 1, (1 << 25) // (ny * nz) or 1))
    shapes = [(nx + 1, ny, nz), (nx, ny, nz), (nx, ny, nz)]
    res = []
    for comp in range(3):
        f = out[comp] if out is not None else torch.empty(shapes[comp], dtype=torch.float64, device=device)
        assert tuple(f.shape) == shapes[comp]
        for i0, i1, blk in _component(cfg, xc_t, comp, device, chunk):
            f[i0:i1] = blk
        if comp == 0:
            f[0].zero_()
            f[nx].zero_()
        res.append(f)
    return tuple(res)
