"""Host-side checks that need no GPU: the C-ABI library builds and loads, exports every symbol
include/afid.h declares, fails loudly without a device, and the product never touches oracle/."""
import ctypes
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "afid.h")


@pytest.fixture(scope="module")
def built_lib():
    from paper_1705_01423_b200 import build
    return build.build()


def declared_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(afid_[a-z0-9_]+)\s*\(", txt)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for name in ("afid_plan_create", "afid_project", "afid_plan_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol(built_lib):
    lib = ctypes.CDLL(built_lib)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    import paper_1705_01423_b200 as afid
    assert sorted(afid.SYMBOLS) == declared_symbols()
    assert b"sm_100a" in ctypes.cast(afid.lib().afid_version, ctypes.CFUNCTYPE(ctypes.c_char_p))()


def test_library_is_sm100a_only(built_lib):
    out = subprocess.run(["cuobjdump", "-lelf", built_lib], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_supported_sizes_host_queries(built_lib):
    import paper_1705_01423_b200 as afid
    for n in (16, 32, 128, 256, 512, 768, 1024, 1536, 4096, 40, 320, 1280, 2560):
        assert afid.fft_length_supported(n), n
    # include/afid.h: every multiple of 8 of the form 2^a 3^b in [8, 4096] with b <= 4 is a supported y length
    for a in range(3, 13):
        for b in range(0, 5):
            n = 2 ** a * 3 ** b
            if 8 <= n <= 4096:
                assert afid.fft_length_supported(n), n
    for n in (0, 7, 15, 20, 100, 1000, 5000, 3200, 36, 324, 1944):
        assert not afid.fft_length_supported(n), n
    for n in (8, 768, 1024, 40, 640, 1280, 1536, 648, 1296, 36):
        assert afid.fft_half_length_supported(n), n
    for n in (2048, 50, 1728):
        assert not afid.fft_half_length_supported(n), n
    assert afid.max_nx() >= 2048


def test_no_cpu_fallback_without_device(built_lib):
    """On a box without a GPU plan creation must fail with an error, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import paper_1705_01423_b200 as afid
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 32, 32, np.linspace(0.0, 1.0, 33), 1.0, 1.0)
    assert e.value.code == -6
    # argument validation happens before the device is touched
    with pytest.raises(afid.AfidError) as e:
        afid.Plan(32, 56, 32, np.linspace(0.0, 1.0, 33), 1.0, 1.0)
    assert e.value.code == -3


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1705_01423_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|libafid_ref|afid_ref\.c|#include\s+\".*oracle", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), (dirpath, f)
    for f in ("afid_ref.c", "ref.py", "build.py"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_1705_01423_b200" not in src and "libafid_b200" not in src and "#include \"afid" not in src


def test_bench_rank_aggregation_gloo_world2():
    """N>1 path of bench.py = independent replicas; its only cross-rank step is the max-over-
    ranks of the device time and the sum of points.  Run it on 2 CPU ranks over gloo."""
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29631",
                          os.path.join(ROOT, "tests", "gloo_worker.py")],
                         capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    assert "gloo_worker ok rank 0" in res.stdout and "gloo_worker ok rank 1" in res.stdout


def test_bench_gpus_flag_spawns_the_ranks_itself():
    """`python bench.py --gpus 2` without a launcher starts its own two ranks (torch.distributed.run on 127.0.0.1).
    CPU dry run through the reference arm: rank 0 alone times the oracle and prints ONE line with n_gpus = 2,
    the other rank exits 0 without work."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--workload", "C1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["impl"] == "reference" and line["steps"] == 1


def test_bench_gpus_flag_fails_loudly_without_enough_devices():
    """The CUDA arm with more ranks than visible devices exits non-zero with a clear message (no CPU fallback);
    a launcher whose WORLD_SIZE disagrees with --gpus is an error too."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", str(have + 1 if have else 2)],
                         capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode != 0
    assert "CUDA device(s) are visible" in res.stderr, res.stderr[-500:]
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--impl", "reference"],
                         capture_output=True, text=True, env=dict(env, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0"), timeout=600)
    assert res.returncode != 0 and "WORLD_SIZE=2" in res.stderr


@pytest.mark.parametrize("world,shape", [(2, (20, 24, 48)), (3, (13, 8, 16)), (4, (65, 32, 64))])
def test_shard_exchange_schedule_gloo(world, shape):
    """the two all-to-alls of the sharded projection, world_size > 1 on CPU over gloo, with the
    counts / offsets of afid_shard_layout (host arithmetic of the library, no device)."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
                          "--master-addr", "127.0.0.1", "--master-port", str(port),
                          os.path.join(ROOT, "tests", "gloo_shard_worker.py")] + [str(x) for x in shape],
                         capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, res.stdout[-1500:] + res.stderr[-3000:]
    assert res.stdout.count("gloo_shard_worker ok") == world


def test_shard_bounds_partition():
    import paper_1705_01423_b200 as afid
    for n, R in ((1024, 8), (769, 8), (13, 3), (5, 5)):
        b = [afid.shard_bounds(n, R, r) for r in range(R)]
        assert b[0][0] == 0 and b[-1][1] == n
        assert all(b[r][1] == b[r + 1][0] for r in range(R - 1)) and all(hi > lo for lo, hi in b)
        assert max(hi - lo for lo, hi in b) - min(hi - lo for lo, hi in b) <= 1
    with pytest.raises(afid.AfidError):
        afid.shard_bounds(3, 4, 0)


def test_bench_traffic_comes_only_from_a_matching_capture(built_lib):
    """bench.py's roofline.traffic is the committed ncu capture's DRAM bytes per point scaled to the workload; it is
    withheld when the capture has another cross-section or when the captured kernel (by mangled name) is no longer the
    one in the built library."""
    import shutil
    sys.path.insert(0, ROOT)
    import bench
    n = 1024 * 1536 * 1536
    t, src = bench.ncu_traffic("k_correct", 1536, 1536, 1024, n)
    if shutil.which("cuobjdump") is None:
        assert t is None
    else:
        assert t is not None and 55.0 <= t / n <= 57.0 and "r2_dram_traffic.csv" in src   # algorithmic 56 B/pt
    assert bench.ncu_traffic("k_correct", 1024, 1024, 512, 1)[0] is None                  # another cross-section
    assert bench.ncu_traffic("k_c2r_z", 1536, 1536, 1024, n)[0] is None                   # kernel changed since the capture
    assert bench.ncu_traffic("no_such_kernel", 1536, 1536, 1024, n) == (None, None)


@pytest.mark.parametrize("nx,ny", [(1, 8), (3, 8), (5, 40), (7, 36), (64, 128), (9, 1536)])
def test_fused_cfl_schedule_is_deadlock_free_and_covers_every_cell(built_lib, nx, ny):
    """afid_project_cfl (fused form): ticket t corrects item t and then reduces item t - lag.  From the
    library's own schedule arithmetic (afid_cfl_schedule, host only): the items are a bijection onto (plane, line
    group); every dependency of a reduce step is an item at most 8 tickets after it (so with lag > 8 every wait is
    for an EARLIER ticket: no deadlock for any CTA order); each dependency is exactly an item that owns a line the
    step reads (lines lo..hi+1 of planes i and i+1, line 0 for the wrap); and the reduce steps of a plane cover
    every line exactly once."""
    import paper_1705_01423_b200 as afid
    ngrp = ny // 4
    seen, cover = set(), {}
    for s in range(nx * ngrp):
        i, jg, lo, hi, extra, deps = afid.cfl_schedule(nx, ny, s)
        assert 0 <= i < nx and 0 <= jg < ngrp and (i, jg) not in seen
        seen.add((i, jg))
        lines = list(range(lo, hi + 1)) + ([extra] if extra >= 0 else [])
        for j in lines:
            assert (i, j) not in cover
            cover[(i, j)] = s
        need = set()                                   # owners of everything the cells (i, lines, :) read
        for j in lines:
            for (pi, pj) in ((i, j), (i + 1, j), (i, (j + 1) % ny)):
                if pi < nx:                            # plane nx is the wall plane: never written
                    need.add((pi, pj // 4))
        got = set()
        for d in deps:
            if d >= 0:
                assert d <= s + 8, (s, d)              # lag = resident CTAs + 16 > 8
                di, dg = afid.cfl_schedule(nx, ny, d)[:2]
                got.add((di, dg))
        assert got == need, (s, got, need)
    assert len(seen) == nx * ngrp and len(cover) == nx * ny
    with pytest.raises(afid.AfidError):
        afid.cfl_schedule(nx, ny, nx * ngrp)
