"""the sharded projection (afid_shard_*), R logical ranks on ONE device.

Every rank's plan runs the real kernels on its x-slab / kz range; the two all-to-alls and the phi halo are done here
with device copies that follow afid_shard_layout (what torch.distributed does between GPUs).  The result must equal
the unsharded afid_project bit for bit: the same kernels run on the same lines and systems.  (One builder GPU: no
multi-GPU hardware number is produced; the exchange schedule itself is covered on CPU over gloo.)
"""
import numpy as np
import pytest
import torch

import paper_1705_01423_b200 as afid
from paper_1705_01423_b200 import synth
from oracle import ref

pytestmark = pytest.mark.gpu


def local_all_to_all(plans, phase):
    bufs = [pl.buffers(phase) for pl in plans]
    for d, pd in enumerate(plans):
        _, _, rc, ro = pd.layout[phase]
        for s, ps in enumerate(plans):
            sc, so, _, _ = ps.layout[phase]
            assert sc[d] == rc[s]
            bufs[d][1][ro[s]:ro[s] + rc[s]].copy_(bufs[s][0][so[d]:so[d] + sc[d]])


def sharded_project(cfg, xc, u, v, w, R):
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    plans = [afid.ShardPlan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"], r, R) for r in range(R)]
    us = [u[pl.xs:pl.xe + 1].contiguous().cuda() for pl in plans]     # slab + upper halo plane
    vs = [v[pl.xs:pl.xe].contiguous().cuda() for pl in plans]
    ws = [w[pl.xs:pl.xe].contiguous().cuda() for pl in plans]
    ps = [torch.full_like(x, float("nan")) for x in vs]
    for pl, a, b, c in zip(plans, us, vs, ws):
        pl.forward(a, b, c)
    local_all_to_all(plans, 1)
    for pl in plans:
        pl.solve()
    local_all_to_all(plans, 2)
    for pl, p in zip(plans, ps):
        pl.inverse(p)
    for r, pl in enumerate(plans):
        halo = ps[r - 1][-1].contiguous() if r > 0 else None
        pl.correct(us[r], vs[r], ws[r], ps[r], halo)
    torch.cuda.synchronize()
    uo = torch.cat([x[:-1] for x in us] + [us[-1][-1:]]).cpu().numpy()
    out = uo, torch.cat(vs).cpu().numpy(), torch.cat(ws).cpu().numpy(), torch.cat(ps).cpu().numpy()
    for pl in plans:
        pl.destroy()
    return out


CASES = [
    (dict(nx=20, ny=24, nz=48, grid="tanh", s=3.0, Ly=1.3), 2),
    (dict(nx=20, ny=24, nz=48, grid="tanh", s=3.0, Ly=1.3), 3),
    (dict(nx=65, ny=32, nz=64, grid="tanh", s=3.0), 4),
    (dict(nx=130, ny=64, nz=32, grid="erf", s=1.5, x_lo=-1.0, x_hi=1.0, shear=1.0), 8),
    (dict(nx=33, ny=40, nz=80, grid="uniform"), 5),
    (dict(nx=16, ny=8, nz=16, grid="uniform"), 1),
]


@pytest.mark.parametrize("ov,R", CASES, ids=lambda o: str(o) if isinstance(o, int) else f"{o['nx']}x{o['ny']}x{o['nz']}")
def test_sharded_equals_unsharded_bitwise(ov, R):
    cfg = synth.config("C1", **ov)
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    ud, vd, wd = u.cuda(), v.cuda(), w.cuda()
    p = torch.empty_like(vd)
    plan.project(ud, vd, wd, p)
    torch.cuda.synchronize()
    want = ud.cpu().numpy(), vd.cpu().numpy(), wd.cpu().numpy(), p.cpu().numpy()
    plan.destroy()
    got = sharded_project(cfg, xc, u, v, w, R)
    for name, a, b in zip("uvwp", got, want):
        assert np.array_equal(a, b), (name, float(np.abs(a - b).max()))


def test_sharded_against_oracle():
    """and, independently of the unsharded CUDA path, against the CPU oracle."""
    cfg = synth.config("C1", nx=24, ny=32, nz=48, grid="tanh", s=3.0, Lz=0.7)
    xc = synth.grid_faces(cfg)
    u, v, w = synth.velocity(cfg, xc)
    uo, vo, wo, po, _ = ref.project(xc, cfg["Ly"], cfg["Lz"], u.numpy(), v.numpy(), w.numpy())
    got = sharded_project(cfg, xc, u, v, w, 3)
    for name, a, b in zip("uvwp", got, (uo, vo, wo, po)):
        err = float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
        assert err <= 1e-11, (name, err)


def test_sharded_plan_rejects_unsharded_calls_and_bad_ranks():
    cfg = synth.config("C1")
    xc = synth.grid_faces(cfg)
    pl = afid.ShardPlan(32, 32, 32, xc, 1.0, 1.0, 1, 2)
    z = torch.zeros(16 * 32 * 32, dtype=torch.float64, device="cuda")
    zu = torch.zeros(17 * 32 * 32, dtype=torch.float64, device="cuda")
    rc = afid.lib().afid_project(pl._h, zu.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), None)
    assert rc == -3
    with pytest.raises(afid.AfidError):        # rank 1 needs the phi halo
        pl.correct(zu, z, z, z, None)
    pl.destroy()
    for rank, nranks in ((2, 2), (0, 65), (0, 33)):   # rank out of range, too many ranks, more ranks than kz modes (17) / planes
        with pytest.raises(afid.AfidError):
            afid.ShardPlan(32, 32, 32, xc, 1.0, 1.0, rank, nranks)
