"""Worker of test_shard_exchange_schedule_gloo (run under torchrun on CPU ranks, gloo): the two all-to-alls of the
sharded projection (include/afid.h, afid_shard_*) with the counts and offsets of afid_shard_layout, on index-tagged
payloads.  Every (i, ky, kz) must leave its slab exactly once and land where the x-solve kernel expects it
(C[kz_local][i][ky] over ALL planes), and come back to T_loc[kz][ky/8][i_local][ky%8] of its slab.  The strided
re-layouts the library does on the device (afid_shard_solve) are restated here from the header's description."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_1705_01423_b200 as afid  # noqa: E402  (host arithmetic only: no device is touched)

nx, ny, nz = (int(x) for x in sys.argv[1:4])
dist.init_process_group("gloo")
r, R = dist.get_rank(), dist.get_world_size()
nzh = nz // 2 + 1
xs, xe = afid.shard_bounds(nx, R, r)
ks, ke = afid.shard_bounds(nzh, R, r)
nxl, nkz, nkt = xe - xs, ke - ks, ny // 8
bx = [afid.shard_bounds(nx, R, q) for q in range(R)]
bk = [afid.shard_bounds(nzh, R, q) for q in range(R)]


def tag(i, ky, kz):      # a unique complex tag per mode and plane
    return (i * ny + ky) + 1j * kz


def exchange(phase, send):
    sc, so, rc, ro = afid.shard_layout(nx, ny, nz, R, r, phase)
    assert so == list(np.cumsum([0] + sc[:-1])) and ro == list(np.cumsum([0] + rc[:-1]))   # blocks back to back, in rank order
    assert sum(sc) == send.size
    recv = torch.empty(sum(rc), dtype=torch.complex128)
    dist.all_to_all_single(recv, torch.from_numpy(send.ravel()), output_split_sizes=rc, input_split_sizes=sc)
    return recv.numpy(), rc, ro


# ---- exchange 1: C_loc[kz][i_local][ky] (all kz, my planes) -> C[kz_local][i][ky] (my kz, all planes)
KZ, I, KY = np.meshgrid(np.arange(nzh), np.arange(xs, xe), np.arange(ny), indexing="ij")
recv, rc, ro = exchange(1, tag(I, KY, KZ))
C = np.full((nkz, nx, ny), np.nan + 0j)
for s in range(R):       # block of peer s = [my kz][planes of s][ky] -> rows bx[s] of every kz
    x0, x1 = bx[s]
    assert rc[s] == nkz * (x1 - x0) * ny
    C[:, x0:x1, :] = recv[ro[s]:ro[s] + rc[s]].reshape(nkz, x1 - x0, ny)
KZ, I, KY = np.meshgrid(np.arange(ks, ke), np.arange(nx), np.arange(ny), indexing="ij")
assert np.array_equal(C, tag(I, KY, KZ)), "exchange 1: a mode did not arrive where the x-solve reads it"

# ---- exchange 2: T[kz_local][kyt][i][8] (my kz, all planes) -> T_loc[kz][kyt][i_local][8] (all kz, my planes)
KZ, KT, I, K8 = np.meshgrid(np.arange(ks, ke), np.arange(nkt), np.arange(nx), np.arange(8), indexing="ij")
T = tag(I, KT * 8 + K8, KZ)
send = np.concatenate([T[:, :, bx[d][0]:bx[d][1], :].ravel() for d in range(R)])   # block of peer d = [my kz][kyt][planes of d][8]
recv, rc, ro = exchange(2, send)
KZ, KT, I, K8 = np.meshgrid(np.arange(nzh), np.arange(nkt), np.arange(xs, xe), np.arange(8), indexing="ij")
assert np.array_equal(recv.reshape(nzh, nkt, nxl, 8), tag(I, KT * 8 + K8, KZ)), "exchange 2: the slab did not get its modes back"
for s in range(R):
    assert ro[s] == bk[s][0] * nkt * nxl * 8 and rc[s] == (bk[s][1] - bk[s][0]) * nkt * nxl * 8

# every element was sent exactly once per exchange: the counts add up to the whole half spectrum
tot = torch.tensor([nxl * nzh * ny, nx * nkz * ny], dtype=torch.int64)
dist.all_reduce(tot)
assert int(tot[0]) == nx * nzh * ny and int(tot[1]) == nx * nzh * ny
dist.barrier()
dist.destroy_process_group()
print(f"gloo_shard_worker ok rank {r}/{R}", flush=True)
