"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by
element on the same seeded inputs, plus the full-size checks of the bench configurations.

Tolerances (BASELINE.json north_star): relative L2 <= 1e-11 in p and in the corrected u, v, w;
post-projection max|div| <= 1e-10 * max|div_in|.
"""
import math

import numpy as np
import pytest
import torch

import paper_1705_01423_b200 as afid
from paper_1705_01423_b200 import synth
from oracle import ref

import manufactured as mf

pytestmark = pytest.mark.gpu

TOL = 1e-11
DIV_TOL = 1e-10


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def gpu_project(cfg, xc, u, v, w, calls=1):
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
    p = torch.full((nx, ny, nz), float("nan"), dtype=torch.float64, device="cuda")
    outs = []
    for _ in range(calls):
        plan.project(ud, vd, wd, p)
        torch.cuda.synchronize()
        outs.append((ud.cpu().numpy().copy(), vd.cpu().numpy().copy(), wd.cpu().numpy().copy(), p.cpu().numpy().copy()))
    plan.destroy()
    return outs


def check_against_oracle(cfg, xc, u, v, w):
    un, vn, wn = u.numpy(), v.numpy(), w.numpy()
    uo, vo, wo, po, max_imag = ref.project(xc, cfg["Ly"], cfg["Lz"], un, vn, wn)
    ug, vg, wg, pg = gpu_project(cfg, xc, u, v, w)[0]
    errs = dict(p=rel(pg, po), u=rel(ug, uo), v=rel(vg, vo), w=rel(wg, wo))
    assert all(e <= TOL for e in errs.values()), errs
    # invariants on the GPU output, evaluated with the oracle's operators
    din = np.abs(ref.divergence(xc, cfg["Ly"], cfg["Lz"], un, vn, wn)).max()
    dout = np.abs(ref.divergence(xc, cfg["Ly"], cfg["Lz"], ug, vg, wg)).max()
    assert dout <= DIV_TOL * din, (dout, din)
    dx = np.diff(xc)
    mean = (pg * dx[:, None, None]).sum() / (dx.sum() * cfg["ny"] * cfg["nz"])
    assert abs(mean) <= 1e-13 * np.abs(pg).max()
    nx = cfg["nx"]
    assert np.array_equal(ug[0], un[0]) and np.array_equal(ug[nx], un[nx])  # wall planes bit-unchanged
    return errs


def test_c1_parity():
    cfg = synth.config("C1")
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    check_against_oracle(cfg, xc, u, v, w)


# odd shapes: radix-3 lengths, ny != nz, ragged last x-chunk (nx % 16 != 0, nx % 4 != 0),
# the three K3 instantiations (nx < 64, <= 1024, > 1024), minimum sizes
SHAPES = [
    dict(nx=2, ny=8, nz=16, grid="uniform"),
    dict(nx=5, ny=24, nz=48, grid="tanh", s=3.0, Ly=1.3, Lz=0.7),
    dict(nx=63, ny=32, nz=64, grid="tanh", s=3.0),
    dict(nx=65, ny=96, nz=64, grid="tanh", s=3.0, Ly=2.0, Lz=0.5),
    dict(nx=33, ny=192, nz=384, grid="erf", s=1.5, x_lo=-1.0, x_hi=1.0, Ly=8 * math.pi, Lz=2 * math.pi, shear=1.0),
    dict(nx=100, ny=48, nz=96, grid="tanh", s=3.0),
    dict(nx=1030, ny=8, nz=32, grid="tanh", s=3.0),
    dict(nx=40, ny=64, nz=128, grid="tanh", s=3.0, M=32, expo=-5.0 / 6.0),
    dict(nx=17, ny=128, nz=256, grid="uniform"),
    dict(nx=16, ny=384, nz=192, grid="tanh", s=3.0),
    # lengths 5 * 2^a (radix-5 passes), every such plan at least once in y and in z
    dict(nx=6, ny=40, nz=80, grid="tanh", s=3.0, Ly=1.3),
    dict(nx=9, ny=160, nz=320, grid="tanh", s=3.0),
    dict(nx=4, ny=80, nz=1280, grid="uniform", Lz=2.5),
    dict(nx=3, ny=640, nz=160, grid="tanh", s=3.0),
    dict(nx=2, ny=1280, nz=640, grid="uniform"),
    dict(nx=2, ny=2560, nz=80, grid="tanh", s=3.0),
    dict(nx=5, ny=320, nz=80, grid="tanh", s=3.0),
    # the largest instantiations: nz/2 = 1024, ny = 3072, nx = afid_max_nx()
    dict(nx=3, ny=8, nz=2048, grid="uniform"),
    dict(nx=2, ny=3072, nz=16, grid="uniform"),
    dict(nx=1536, ny=8, nz=16, grid="tanh", s=3.0),
    # every length 2^a 3^b with b >= 2 (repeated radix-3/6/12 passes), each plan at least
    # once in y (complex length ny) and once in z (complex length nz/2)
    dict(nx=4, ny=8, nz=24, grid="uniform"),
    dict(nx=5, ny=16, nz=36, grid="tanh", s=3.0, Ly=0.8),
    dict(nx=6, ny=24, nz=72, grid="tanh", s=3.0),
    dict(nx=3, ny=48, nz=108, grid="uniform", Lz=1.7),
    dict(nx=7, ny=72, nz=144, grid="tanh", s=3.0),
    dict(nx=3, ny=96, nz=216, grid="tanh", s=3.0),
    dict(nx=4, ny=144, nz=288, grid="tanh", s=3.0),
    dict(nx=2, ny=128, nz=324, grid="uniform"),
    dict(nx=3, ny=216, nz=432, grid="tanh", s=3.0),
    dict(nx=2, ny=288, nz=576, grid="tanh", s=3.0),
    dict(nx=2, ny=256, nz=648, grid="uniform"),
    dict(nx=2, ny=432, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=576, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=648, nz=16, grid="uniform"),
    dict(nx=2, ny=864, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=1152, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=1296, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=1728, nz=16, grid="uniform"),
    dict(nx=2, ny=2304, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=2592, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=3456, nz=16, grid="uniform"),
    dict(nx=2, ny=8, nz=864, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=1152, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=1296, grid="uniform"),
    dict(nx=2, ny=8, nz=1728, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=2304, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=2560, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=2592, grid="uniform"),
    # the paper's grid families as slabs (Table 3: 768 x 768 x 1296, wall-normal 1296;
    # P:L319-L329 Table 2: 2048 x 3072 x 3072): nx = 1296 and 2048 = afid_max_nx(), ny = 3072, nz = 3072
    dict(nx=1296, ny=24, nz=16, grid="tanh", s=3.0),
    dict(nx=2048, ny=8, nz=16, grid="tanh", s=3.0),
    dict(nx=2040, ny=8, nz=16, grid="tanh", s=3.0),
    dict(nx=2, ny=8, nz=3072, grid="tanh", s=3.0),
    dict(nx=3, ny=768, nz=48, grid="tanh", s=3.0),
]


@pytest.mark.parametrize("ov", SHAPES, ids=lambda o: f"{o['nx']}x{o['ny']}x{o['nz']}")
def test_shapes_parity(ov):
    cfg = synth.config("C1", **ov)
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    check_against_oracle(cfg, xc, u, v, w)


@pytest.mark.parametrize("ov", [SHAPES[1], SHAPES[4], SHAPES[7], dict(nx=256, ny=256, nz=256, grid="tanh", s=3.0)],
                         ids=lambda o: f"{o['nx']}x{o['ny']}x{o['nz']}")
def test_max_cfl_parity(ov):
    """afid_max_cfl (paper's Listing 1) against the oracle, on the provisional and on the projected field, and
    the 1e-8 floor.  Both sides form each cell's value by the same three products and two additions in fp64;
    the reciprocal spacings are rounded differently (the oracle divides ny/Ly and 1/dx in fp64, the plan
    rounds 1/(Ly/ny) and 1/dx once from long double), each within one ulp, so the maxima agree to a few ulp:
    tolerance 2e-15 relative."""
    cfg = synth.config("C1", **ov)
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    u, v, w = synth.velocity(cfg, xc)
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
    got = float(plan.max_cfl(ud, vd, wd).cpu())
    want = ref.max_cfl(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
    assert abs(got - want) <= 2e-15 * want, (got, want)
    p = torch.empty_like(vd)
    plan.project(ud, vd, wd, p)
    got2 = float(plan.max_cfl(ud, vd, wd).cpu())
    want2 = ref.max_cfl(xc, cfg["Ly"], cfg["Lz"], ud.cpu().numpy(), vd.cpu().numpy(), wd.cpu().numpy())
    assert abs(got2 - want2) <= 2e-15 * want2, (got2, want2)
    z = torch.zeros_like(vd)
    assert float(plan.max_cfl(torch.zeros_like(ud), z, z).cpu()) == 1e-8
    plan.destroy()


@pytest.mark.parametrize("ov", [SHAPES[1], SHAPES[4], SHAPES[7], dict(nx=256, ny=256, nz=256, grid="tanh", s=3.0),
                                dict(nx=40, ny=8, nz=16), dict(nx=3, ny=40, nz=1280), dict(nx=130, ny=768, nz=64, grid="tanh", s=3.0)],
                         ids=lambda o: f"{o['nx']}x{o['ny']}x{o['nz']}")
def test_project_cfl_fused(ov):
    """afid_project_cfl (fused form): u, v, w, p bit-identical to afid_project's; the CFL number
    bit-identical to afid_max_cfl on the projected field (a maximum over the same per-cell values) and within
    2e-15 of the oracle's Listing 1 on the oracle's projected field (the oracle's field differs from the GPU's
    by the parity tolerance, so that comparison carries 1e-11); repeated calls (flags re-zeroed) agree; the
    accumulate mode goes through the same kernel."""
    cfg = synth.config("C1", **ov)
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    u, v, w = synth.velocity(cfg, xc)
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    a = [t.cuda() for t in (u, v, w)]
    b = [t.cuda() for t in (u, v, w)]
    pa, pb = torch.empty_like(a[1]), torch.empty_like(a[1])
    plan.project(*a, pa)
    sep = float(plan.max_cfl(*a).cpu())
    for rep in range(2):
        for t, src in zip(b, (u, v, w)):
            t.copy_(src)
        pb.fill_(float("nan"))
        fused = float(plan.project_cfl(*b, pb).cpu())
        for x, y in zip(a + [pa], b + [pb]):
            assert torch.equal(x, y)
        assert fused == sep, (fused, sep)
    if nx * ny * nz <= 2_000_000:   # (the naive-DFT oracle projection of 256^3 is covered by test_c2)
        uo, vo, wo, po, _ = ref.project(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
        want = ref.max_cfl(xc, cfg["Ly"], cfg["Lz"], uo, vo, wo)
        assert abs(fused - want) <= 1e-11 * want, (fused, want)
    want_gpu_field = ref.max_cfl(xc, cfg["Ly"], cfg["Lz"], a[0].cpu().numpy(), a[1].cpu().numpy(), a[2].cpu().numpy())
    assert abs(fused - want_gpu_field) <= 2e-15 * want_gpu_field, (fused, want_gpu_field)
    # accumulate mode: p += phi through the fused kernel
    plan.set_accumulate(True)
    for t, src in zip(b, (u, v, w)):
        t.copy_(src)
    pc = torch.ones_like(pb)
    fused2 = float(plan.project_cfl(*b, pc).cpu())
    assert fused2 == sep
    assert torch.equal(b[0], a[0]) and torch.equal(b[1], a[1]) and torch.equal(b[2], a[2])
    assert rel(pc.cpu().numpy(), 1.0 + pa.cpu().numpy()) <= 1e-15
    plan.set_accumulate(False)
    plan.destroy()


@pytest.mark.parametrize("shape", [(5, 8, 16), (33, 24, 48), (64, 32, 64), (100, 16, 32), (256, 64, 64), (1030, 8, 32), (1024, 16, 64), (2048, 8, 32), (1700, 8, 16)],
                         ids=lambda t: "x".join(map(str, t)))
def test_xsolve_parity(shape):
    """afid_xsolve_apply against the oracle's long-double Thomas: every K3 instantiation
    (nx < 64, <= 1024 with 8- and 4-wide tiles, > 1024; full and ragged chunks), coefficients of an implicit
    diffusion step on the stretched grid with Dirichlet walls, plus a rough random M-matrix."""
    nx, ny, nz = shape
    cfg = synth.config("C1", nx=nx, ny=ny, nz=nz, grid="tanh", s=3.0)
    xc = synth.grid_faces(cfg)
    dx, dc = ref.metrics(xc)
    a = np.zeros(nx); c = np.zeros(nx)
    a[1:] = 1.0 / (dx[1:] * dc[1:nx]); c[:-1] = 1.0 / (dx[:-1] * dc[1:nx])
    theta = 1e-3                                           # (I - theta L_x) x = r  <=>  lam = 1/theta
    lam = np.full(nx, 1.0 / theta)
    lam[0] += 2.0 / dx[0] ** 2; lam[-1] += 2.0 / dx[-1] ** 2  # Dirichlet walls by ghost cells
    rng = np.random.default_rng(7)
    plan = afid.Plan(nx, ny, nz, xc, 1.0, 1.0)
    for (aa, cc, ll) in ((a, c, lam), (rng.uniform(0.1, 1e4, nx), rng.uniform(0.1, 1e4, nx), rng.uniform(1e-2, 10.0, nx))):
        f = torch.from_numpy(rng.standard_normal((nx, ny, nz)))
        want = ref.xsolve(aa, cc, ll, f.numpy())
        xs = plan.xsolve(aa, cc, ll)
        fd = f.cuda()
        xs.apply(fd)
        torch.cuda.synchronize()
        assert rel(fd.cpu().numpy(), want) <= 1e-13, rel(fd.cpu().numpy(), want)
        xs.destroy()
    with pytest.raises(afid.AfidError) as e:               # not an M-matrix
        plan.xsolve(a, c, np.zeros(nx))
    assert e.value.code == -4
    plan.destroy()


def test_cuda_graph_capture_replays_bit_identically():
    """afid_project only enqueues kernels on the given stream, so it can be captured in a CUDA graph
    (C1 is launch-latency bound: six launches; a replay takes about half the eager time)."""
    cfg = synth.config("C1")
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    u, v, w = synth.velocity(cfg, xc)
    u0, v0, w0 = u.cuda(), v.cuda(), w.cuda()
    ud, vd, wd = u0.clone(), v0.clone(), w0.clone()
    p = torch.empty_like(vd)
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    plan.project(ud, vd, wd, p)
    torch.cuda.synchronize()
    eager = (ud.clone(), vd.clone(), wd.clone(), p.clone())
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    ud.copy_(u0); vd.copy_(v0); wd.copy_(w0)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            plan.project(ud, vd, wd, p, stream=torch.cuda.current_stream())
    for _ in range(2):
        ud.copy_(u0); vd.copy_(v0); wd.copy_(w0); p.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert all(torch.equal(a, b) for a, b in zip(eager, (ud, vd, wd, p)))
    plan.destroy()


def test_bitwise_deterministic():
    """No atomics and no data-dependent scheduling on the default path: the same input gives the same bits."""
    cfg = synth.config("C2", nx=128, ny=96, nz=192)
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    plan = afid.Plan(cfg["nx"], cfg["ny"], cfg["nz"], xc, cfg["Ly"], cfg["Lz"])
    outs = []
    for _ in range(3):
        ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
        p = torch.empty_like(vd)
        plan.project(ud, vd, wd, p)
        torch.cuda.synchronize()
        outs.append((ud, vd, wd, p))
    for o in outs[1:]:
        assert all(torch.equal(a, b) for a, b in zip(outs[0], o))
    plan.destroy()


def test_accumulate_mode_parity():
    """afid_plan_set_accumulate(1): p_out = p_in + phi (P:L91, P:L116 delta form); the velocities as before."""
    cfg = synth.config("C1", nx=40, ny=64, nz=128, grid="tanh", s=3.0)
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    u, v, w = synth.velocity(cfg, xc)
    uo, vo, wo, po, _ = ref.project(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
    p_in = torch.from_numpy(np.random.default_rng(3).standard_normal((nx, ny, nz)))
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    plan.set_accumulate(True)
    ud, vd, wd, pd = u.cuda(), v.cuda(), w.cuda(), p_in.cuda()
    plan.project(ud, vd, wd, pd)
    torch.cuda.synchronize()
    assert rel(pd.cpu().numpy() - p_in.numpy(), po) <= 1e-11
    assert rel(ud.cpu().numpy(), uo) <= TOL and rel(vd.cpu().numpy(), vo) <= TOL and rel(wd.cpu().numpy(), wo) <= TOL
    plan.set_accumulate(False)
    ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
    plan.project(ud, vd, wd, pd)
    torch.cuda.synchronize()
    assert rel(pd.cpu().numpy(), po) <= TOL
    plan.destroy()


def test_stage_taps_parity():
    """Forward spectrum and x-solve separately (stage boundaries of the paper's step list)."""
    cfg = synth.config("C1", nx=37, ny=48, nz=96, grid="tanh", s=3.0, Ly=1.5, Lz=0.75)
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    nzh = nz // 2 + 1
    u, v, w = synth.velocity(cfg, xc)
    d = ref.divergence(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
    dh = ref.forward_spectrum(d)                       # [nx][ny][nz], unnormalised
    want_fwd = -dh[:, :, :nzh].transpose(0, 2, 1) / (ny * nz)
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    spec = torch.zeros(2 * nx * nzh * ny, dtype=torch.float64, device="cuda")
    plan.stage_forward(u.cuda(), v.cuda(), w.cuda(), spec)
    torch.cuda.synchronize()
    got = spec.cpu().numpy().view(np.complex128).reshape(nx, nzh, ny)
    assert rel(got, want_fwd) <= 1e-13
    xs = ref.solve(xc, cfg["Ly"], cfg["Lz"], dh)       # oracle solves a x - (a+c+lam) x + c x = dhat
    want_sol = xs[:, :, :nzh].transpose(0, 2, 1) / (ny * nz)
    spec2 = torch.from_numpy(np.ascontiguousarray(want_fwd).view(np.float64).ravel().copy()).cuda()
    plan.stage_solve(spec2)
    torch.cuda.synchronize()
    got2 = spec2.cpu().numpy().view(np.complex128).reshape(nx, nzh, ny)
    assert rel(got2, want_sol) <= 1e-13
    assert np.abs(got2[:, 0, 0] - want_sol[:, 0, 0]).max() <= 1e-13 * np.abs(want_sol[:, 0, 0]).max()
    plan.destroy()


def test_idempotent_and_back_to_back():
    """C2-shaped (reduced in y,z so the oracle takes seconds): parity on call 1, a second
    projection of the projected field changes nothing beyond round-off (invariant P4 iii)."""
    cfg = synth.config("C2", ny=64, nz=64)
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    check_against_oracle(cfg, xc, u, v, w)
    (u1, v1, w1, p1), (u2, v2, w2, p2) = gpu_project(cfg, xc, u, v, w, calls=2)
    assert np.linalg.norm(p2) <= 1e-10 * np.linalg.norm(p1)
    assert rel(u2, u1) <= 1e-12 and rel(v2, v1) <= 1e-12 and rel(w2, w1) <= 1e-12


def test_c2_full_parity():
    """BASELINE config 2 at full size (256^3, tanh grid) against the full oracle."""
    cfg = synth.config("C2")
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    check_against_oracle(cfg, xc, u, v, w)


def test_two_live_plans_of_different_nx_and_an_xsolve_handle():
    """One kernel instantiation serves many nx and several live plans: the dynamic shared-memory limit of a function
    is raised once and never lowered by a later, smaller plan.  Plan nx = 512 first, then nx = 384
    (same k_solve_x instantiation, smaller tile) and an xsolve handle; the OLDER plan must still project."""
    cfgs = [synth.config("C1", nx=512, ny=8, nz=16, grid="tanh", s=3.0), synth.config("C1", nx=384, ny=8, nz=16, grid="tanh", s=3.0)]
    xcs = [synth.grid_faces(c) for c in cfgs]
    plans = [afid.Plan(c["nx"], c["ny"], c["nz"], xc, c["Ly"], c["Lz"]) for c, xc in zip(cfgs, xcs)]
    xs = plans[1].xsolve(np.full(384, 2.0), np.full(384, 3.0), np.full(384, 10.0))
    for k in (0, 1, 0):                                    # the older plan first, and again after the newer one ran
        cfg, xc, plan = cfgs[k], xcs[k], plans[k]
        u, v, w = synth.velocity(cfg, xc)
        uo, vo, wo, po, _ = ref.project(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
        ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
        p = torch.empty_like(vd)
        plan.project(ud, vd, wd, p)
        torch.cuda.synchronize()
        assert rel(p.cpu().numpy(), po) <= TOL and rel(ud.cpu().numpy(), uo) <= TOL
        assert rel(vd.cpu().numpy(), vo) <= TOL and rel(wd.cpu().numpy(), wo) <= TOL
    f = torch.ones((384, 8, 16), dtype=torch.float64, device="cuda")
    xs.apply(f)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(f).all())
    xs.destroy()
    for pl in plans:
        pl.destroy()


def test_error_codes():
    xc = np.linspace(0.0, 1.0, 33)
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 56, 32, xc, 1.0, 1.0)           # 56 = 7 * 8 is not a supported FFT length
    assert e.value.code == -3
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 32, 30, xc, 1.0, 1.0)           # nz/2 = 15
    assert e.value.code == -3
    bad = xc.copy()
    bad[5] = bad[4]
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 32, 32, bad, 1.0, 1.0)
    assert e.value.code == -4
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 32, 32, xc, -1.0, 1.0)
    assert e.value.code == -4
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(afid.max_nx() + 1, 32, 32, np.linspace(0, 1, afid.max_nx() + 2), 1.0, 1.0)
    assert e.value.code == -3
    plan = afid.Plan(32, 32, 32, xc, 1.0, 1.0)
    n = 32 ** 3
    big = torch.zeros(n + 32 * 32 + 1, dtype=torch.float64, device="cuda")
    v = torch.zeros(n, dtype=torch.float64, device="cuda")
    with pytest.raises(afid.AfidError) as e:            # u shifted by 8 bytes: misaligned
        plan.project(big[1:], v, v.clone(), v.clone())
    assert e.value.code == -2
    plan.destroy()


# ---------------------------------------------------------------------------------------
# Full-size configurations (C3, C4 = the bench workload, C5): the oracle's O(N (ny+nz)) DFT
# cannot run there, so (a) a manufactured Helmholtz split whose exact answer is known by
# construction, (b) the invariants, (c) oracle-computed samples of the forward spectrum.
# ---------------------------------------------------------------------------------------
def _full_size_checks(name, sample_planes):
    cfg = synth.config(name)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    nzh = nz // 2 + 1
    need = (4 * nx * ny * nz * 8 + 2 * nx * nzh * ny * 16) * 1.35
    import gc
    gc.collect()
    torch.cuda.empty_cache()          # give back what earlier tests' caches still hold
    free, _ = torch.cuda.mem_get_info()
    if free < need:
        pytest.skip(f"{name} needs {need / 2**30:.0f} GiB of device memory")
    xc = synth.grid_faces(cfg)
    dev = "cuda"
    u = torch.empty((nx + 1, ny, nz), dtype=torch.float64, device=dev)
    v = torch.empty((nx, ny, nz), dtype=torch.float64, device=dev)
    w = torch.empty_like(v)
    phi, psi, chi = mf.potentials(cfg, xc, dev)
    mf.solenoidal_into(cfg, xc, psi, chi, u, v, w)
    mf.add_gradient(cfg, xc, phi, u, v, w)
    del phi, psi, chi
    torch.cuda.empty_cache()
    div_in = mf.max_abs_divergence(cfg, xc, u, v, w)
    wall0, wall1 = u[0].clone(), u[nx].clone()

    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    # (c) sampled forward spectrum against the oracle's naive DFT of the oracle's divergence
    if sample_planes:
        spec = torch.empty(2 * nx * nzh * ny, dtype=torch.float64, device=dev)
        plan.stage_forward(u, v, w, spec)
        torch.cuda.synchronize()
        sg = spec.view(nx, nzh, ny, 2)
        for i in sample_planes:
            i = min(i, nx - 2)
            d2 = ref.divergence(xc[i:i + 3], cfg["Ly"], cfg["Lz"], u[i:i + 3].cpu().numpy(),
                                v[i:i + 2].cpu().numpy(), w[i:i + 2].cpu().numpy())
            dh = ref.forward_spectrum(d2[:1])[0]        # [ny][nz]
            want = -dh[:, :nzh].T / (ny * nz)           # [kz][ky]
            got = sg[i].cpu().numpy().view(np.complex128).reshape(nzh, ny)
            assert rel(got, want) <= 1e-12, (name, i, rel(got, want))
        del spec, sg
        torch.cuda.empty_cache()
    p = torch.full((nx, ny, nz), float("nan"), dtype=torch.float64, device=dev)
    plan.project(u, v, w, p)
    torch.cuda.synchronize()
    plan.destroy()
    torch.cuda.empty_cache()

    # (b) invariants
    div_out = mf.max_abs_divergence(cfg, xc, u, v, w)
    assert div_out <= DIV_TOL * div_in, (div_out, div_in)
    assert torch.equal(u[0], wall0) and torch.equal(u[nx], wall1)
    dx = torch.as_tensor(np.diff(xc)).to(dev)
    wsum = sum(float(p[i].sum()) * float(dx[i]) for i in range(nx))
    assert abs(wsum / (float(dx.sum()) * ny * nz)) <= 1e-13 * float(p.abs().max())
    # (a) exact answer by construction
    phi, psi, chi = mf.potentials(cfg, xc, dev)
    e_p = mf.rel_l2(p, phi)
    del p
    torch.cuda.empty_cache()
    us = torch.empty_like(u)
    mf.solenoidal_into(cfg, xc, psi, chi, us, phi, psi)   # v_sol -> phi's storage, w_sol -> psi's storage
    e_u, e_v, e_w = mf.rel_l2(u, us), mf.rel_l2(v, phi), mf.rel_l2(w, psi)
    print(f"{name}: rel L2 vs the manufactured answer p {e_p:.2e} u {e_u:.2e} v {e_v:.2e} w {e_w:.2e}; "
          f"max|div_out|/max|div_in| = {div_out / div_in:.2e}")
    assert max(e_p, e_u, e_v, e_w) <= TOL, dict(p=e_p, u=e_u, v=e_v, w=e_w)


def test_manufactured_small():
    """The same construction on a size the oracle handles: both must agree with the known answer."""
    cfg = synth.config("C2", nx=48, ny=32, nz=64)
    xc = synth.grid_faces(cfg)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    u = torch.empty((nx + 1, ny, nz), dtype=torch.float64)
    v = torch.empty((nx, ny, nz), dtype=torch.float64)
    w = torch.empty_like(v)
    phi, psi, chi = mf.potentials(cfg, xc, "cpu")
    mf.solenoidal_into(cfg, xc, psi, chi, u, v, w)
    us, vs, ws = u.clone(), v.clone(), w.clone()
    mf.add_gradient(cfg, xc, phi, u, v, w)
    uo, vo, wo, po, _ = ref.project(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
    assert rel(po, phi.numpy()) <= 1e-12 and rel(uo, us.numpy()) <= 1e-12
    ug, vg, wg, pg = gpu_project(cfg, xc, u, v, w)[0]
    assert rel(pg, phi.numpy()) <= TOL and rel(ug, us.numpy()) <= TOL
    assert rel(vg, vs.numpy()) <= TOL and rel(wg, ws.numpy()) <= TOL


def test_c3_full_size():
    _full_size_checks("C3", sample_planes=[0, 300])


def test_c4_full_size_bench_workload():
    _full_size_checks("C4", sample_planes=[511])


def test_c5_full_size():
    _full_size_checks("C5", sample_planes=[383])
