"""paper_1705_01423_b200 -- B200-native (sm_100a, fp64) projection step of AFiD (arXiv 1705.01423).

Thin Python binding of the C ABI in include/afid.h (same names: afid_plan_create,
afid_project, afid_plan_destroy, stage taps).  It only marshals arguments: every step of
the path runs in the hand-written CUDA kernels of csrc/.  PyTorch is used by callers for
device memory and streams; this module takes raw pointers from tensors.

There is no CPU fallback: if the shared library is missing or cannot be loaded, importing
`lib()` raises.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafid_b200.so")

AFID_OK = 0
ERRORS = {-1: "AFID_ERR_NULL", -2: "AFID_ERR_ALIGN", -3: "AFID_ERR_UNSUPPORTED_SIZE", -4: "AFID_ERR_GRID",
          -5: "AFID_ERR_NOMEM", -6: "AFID_ERR_CUDA"}

# every symbol include/afid.h declares
SYMBOLS = ["afid_plan_create", "afid_project", "afid_plan_destroy", "afid_plan_workspace_bytes",
           "afid_plan_num_launches", "afid_stage_forward", "afid_stage_solve", "afid_fft_length_supported",
           "afid_max_nx", "afid_last_error", "afid_last_error_code", "afid_version",
           "afid_plan_enable_timing", "afid_plan_kernel_times", "afid_plan_kernel_name",
           "afid_fft_half_length_supported", "afid_max_cfl", "afid_project_cfl", "afid_cfl_schedule", "afid_plan_set_accumulate", "afid_xsolve_create", "afid_xsolve_apply",
           "afid_xsolve_destroy", "afid_plan_set_pipeline", "afid_plan_set_l2_hints", "afid_plan_num_timed",
           "afid_shard_plan_create", "afid_shard_bounds", "afid_shard_layout", "afid_shard_buffers", "afid_shard_info",
           "afid_shard_forward", "afid_shard_solve", "afid_shard_inverse", "afid_shard_correct"]

_lib = None


class AfidError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


def lib():
    """Load libafid_b200.so (built by `python -m paper_1705_01423_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1705_01423_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        L.afid_plan_create.restype = vp
        L.afid_plan_create.argtypes = [i, i, i, vp, d, d]
        L.afid_project.restype = i
        L.afid_project.argtypes = [vp, vp, vp, vp, vp, vp]
        L.afid_plan_destroy.restype = i
        L.afid_plan_destroy.argtypes = [vp]
        L.afid_plan_workspace_bytes.restype = C.c_size_t
        L.afid_plan_workspace_bytes.argtypes = [vp]
        L.afid_plan_num_launches.restype = i
        L.afid_plan_num_launches.argtypes = [vp]
        L.afid_stage_forward.restype = i
        L.afid_stage_forward.argtypes = [vp, vp, vp, vp, vp, vp]
        L.afid_stage_solve.restype = i
        L.afid_stage_solve.argtypes = [vp, vp, vp]
        L.afid_xsolve_create.restype = vp
        L.afid_xsolve_create.argtypes = [vp, vp, vp, vp]
        L.afid_xsolve_apply.restype = i
        L.afid_xsolve_apply.argtypes = [vp, vp, vp]
        L.afid_xsolve_destroy.restype = i
        L.afid_xsolve_destroy.argtypes = [vp]
        L.afid_plan_set_accumulate.restype = i
        L.afid_plan_set_accumulate.argtypes = [vp, i]
        L.afid_cfl_schedule.restype = i
        L.afid_cfl_schedule.argtypes = [i, i, i, vp, vp, vp, vp, vp, vp]
        L.afid_project_cfl.restype = i
        L.afid_project_cfl.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.afid_max_cfl.restype = i
        L.afid_max_cfl.argtypes = [vp, vp, vp, vp, vp, vp]
        L.afid_fft_length_supported.restype = i
        L.afid_fft_length_supported.argtypes = [i]
        L.afid_fft_half_length_supported.restype = i
        L.afid_fft_half_length_supported.argtypes = [i]
        L.afid_max_nx.restype = i
        L.afid_last_error.restype = C.c_char_p
        L.afid_last_error_code.restype = i
        L.afid_version.restype = C.c_char_p
        L.afid_plan_enable_timing.restype = i
        L.afid_plan_enable_timing.argtypes = [vp, i]
        L.afid_plan_kernel_times.restype = i
        L.afid_plan_kernel_times.argtypes = [vp, vp, i]
        L.afid_plan_set_pipeline.restype = i
        L.afid_plan_set_pipeline.argtypes = [vp, i, i]
        L.afid_plan_set_l2_hints.restype = i
        L.afid_plan_set_l2_hints.argtypes = [vp, i]
        L.afid_plan_num_timed.restype = i
        L.afid_plan_num_timed.argtypes = [vp]
        L.afid_plan_kernel_name.restype = C.c_char_p
        L.afid_plan_kernel_name.argtypes = [vp, i]
        L.afid_shard_plan_create.restype = vp
        L.afid_shard_plan_create.argtypes = [i, i, i, vp, d, d, i, i]
        L.afid_shard_bounds.restype = i
        L.afid_shard_bounds.argtypes = [i, i, i, vp, vp]
        L.afid_shard_layout.restype = i
        L.afid_shard_layout.argtypes = [i, i, i, i, i, i, vp, vp, vp, vp]
        L.afid_shard_buffers.restype = i
        L.afid_shard_buffers.argtypes = [vp, i, vp, vp]
        L.afid_shard_info.restype = i
        L.afid_shard_info.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.afid_shard_forward.restype = i
        L.afid_shard_forward.argtypes = [vp, vp, vp, vp, vp]
        L.afid_shard_solve.restype = i
        L.afid_shard_solve.argtypes = [vp, vp]
        L.afid_shard_inverse.restype = i
        L.afid_shard_inverse.argtypes = [vp, vp, vp]
        L.afid_shard_correct.restype = i
        L.afid_shard_correct.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        _lib = L
    return _lib


def _last_error():
    L = lib()
    return L.afid_last_error_code(), L.afid_last_error().decode()


def _check(rc):
    if rc != AFID_OK:
        raise AfidError(rc, lib().afid_last_error().decode())


def _dev_ptr(t, n, name):
    """Raw device pointer of a contiguous fp64 CUDA tensor with n elements."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float64 CUDA tensor")
    if t.numel() != n:
        raise ValueError(f"{name} has {t.numel()} elements, expected {n}")
    return C.c_void_p(t.data_ptr())


def fft_length_supported(n):
    return bool(lib().afid_fft_length_supported(int(n)))


def fft_half_length_supported(n):
    return bool(lib().afid_fft_half_length_supported(int(n)))


def max_nx():
    return int(lib().afid_max_nx())


def version():
    return lib().afid_version().decode()


class Plan:
    """afid_plan_create / afid_project / afid_plan_destroy for one grid on the current device."""

    def __init__(self, nx, ny, nz, xc, Ly, Lz):
        import numpy as np
        xc = np.ascontiguousarray(xc, dtype=np.float64)
        if xc.size != nx + 1:
            raise ValueError("xc must hold nx+1 face coordinates")
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.nzh = self.nz // 2 + 1
        self._h = lib().afid_plan_create(self.nx, self.ny, self.nz, xc.ctypes.data_as(C.c_void_p),
                                         float(Ly), float(Lz))
        if not self._h:
            raise AfidError(*_last_error())

    @property
    def workspace_bytes(self):
        return int(lib().afid_plan_workspace_bytes(self._h))

    @property
    def num_launches(self):
        return int(lib().afid_plan_num_launches(self._h))

    def _stream(self, stream):
        import torch
        if stream is None:
            stream = torch.cuda.current_stream()
        return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))

    def project(self, u, v, w, p, stream=None):
        """afid_project: u, v, w updated in place, p overwritten with phi (enqueued, no sync)."""
        n = self.nx * self.ny * self.nz
        _check(lib().afid_project(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"),
                                  _dev_ptr(w, n, "w"), _dev_ptr(p, n, "p"), self._stream(stream)))

    def project_cfl(self, u, v, w, p, out=None, stream=None):
        """afid_project_cfl: afid_project plus the maximum CFL number of the corrected field, reduced inside the
        correction launch, into a 1-element fp64 CUDA tensor (enqueued, no sync)."""
        import torch
        n = self.nx * self.ny * self.nz
        if out is None:
            out = torch.empty(1, dtype=torch.float64, device=u.device)
        _check(lib().afid_project_cfl(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"),
                                      _dev_ptr(w, n, "w"), _dev_ptr(p, n, "p"), _dev_ptr(out, 1, "cfl"), self._stream(stream)))
        return out

    def stage_forward(self, u, v, w, spec, stream=None):
        """afid_stage_forward: spec (fp64 tensor of 2*nx*nzh*ny, complex [i][kz][ky]) <- -(D u)^/(ny nz)."""
        n = self.nx * self.ny * self.nz
        m = 2 * self.nx * self.nzh * self.ny
        _check(lib().afid_stage_forward(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"),
                                        _dev_ptr(w, n, "w"), _dev_ptr(spec, m, "spec"), self._stream(stream)))

    def stage_solve(self, spec, stream=None):
        """afid_stage_solve: in-place x-solves on a [i][kz][ky] spectrum."""
        m = 2 * self.nx * self.nzh * self.ny
        _check(lib().afid_stage_solve(self._h, _dev_ptr(spec, m, "spec"), self._stream(stream)))

    def xsolve(self, a, c, lam):
        """afid_xsolve_create: handle for in-place real tridiagonal solves in x on fields of this plan's shape."""
        return XSolve(self, a, c, lam)

    def set_accumulate(self, on=True):
        """afid_plan_set_accumulate: p += phi instead of p = phi."""
        _check(lib().afid_plan_set_accumulate(self._h, 1 if on else 0))

    def max_cfl(self, u, v, w, out=None, stream=None):
        """afid_max_cfl: maximum CFL number (paper's Listing 1) into a 1-element fp64 CUDA tensor (enqueued)."""
        import torch
        n = self.nx * self.ny * self.nz
        if out is None:
            out = torch.empty(1, dtype=torch.float64, device=u.device)
        _check(lib().afid_max_cfl(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"),
                                  _dev_ptr(w, n, "w"), _dev_ptr(out, 1, "cfl"), self._stream(stream)))
        return out

    def set_pipeline(self, planes_per_batch, rotation=2):
        """afid_plan_set_pipeline: plane-pipelined sweeps with L2-resident intermediates (0 = off)."""
        _check(lib().afid_plan_set_pipeline(self._h, int(planes_per_batch), int(rotation)))

    def set_l2_hints(self, mask):
        """afid_plan_set_l2_hints: bit mask of L2 eviction-priority hints (timing only)."""
        _check(lib().afid_plan_set_l2_hints(self._h, int(mask)))

    def enable_timing(self, on=True):
        """afid_plan_enable_timing: record CUDA events around each kernel of project()."""
        _check(lib().afid_plan_enable_timing(self._h, 1 if on else 0))

    def kernel_times(self):
        """afid_plan_kernel_times: {kernel name: ms} of the most recent project() (synchronises)."""
        n = int(lib().afid_plan_num_timed(self._h))
        ms = (C.c_float * n)()
        _check(lib().afid_plan_kernel_times(self._h, C.cast(ms, C.c_void_p), n))
        return {lib().afid_plan_kernel_name(self._h, k).decode(): float(ms[k]) for k in range(n)}

    def destroy(self):
        if getattr(self, "_h", None):
            lib().afid_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class XSolve:
    """afid_xsolve_create / afid_xsolve_apply / afid_xsolve_destroy."""

    def __init__(self, plan, a, c, lam):
        import numpy as np
        self.plan = plan
        arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (a, c, lam)]
        if any(x.size != plan.nx for x in arrs):
            raise ValueError("a, c, lam must hold nx values each")
        self._h = lib().afid_xsolve_create(plan._h, *[x.ctypes.data_as(C.c_void_p) for x in arrs])
        if not self._h:
            raise AfidError(*_last_error())

    def apply(self, f, stream=None):
        """afid_xsolve_apply: f (nx, ny, nz) fp64 CUDA tensor, solved in place column by column (enqueued)."""
        n = self.plan.nx * self.plan.ny * self.plan.nz
        _check(lib().afid_xsolve_apply(self._h, _dev_ptr(f, n, "f"), self.plan._stream(stream)))

    def destroy(self):
        if getattr(self, "_h", None):
            lib().afid_xsolve_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------
# the projection sharded over ranks (include/afid.h, afid_shard_*)
# ------------------------------------------------------------------------------------------
def cfl_schedule(nx, ny, item):
    """afid_cfl_schedule (host arithmetic): (i, jg, line_lo, line_hi, extra_line, deps[5]) of item `item`."""
    out = [C.c_int() for _ in range(5)]
    deps = (C.c_int * 5)()
    _check(lib().afid_cfl_schedule(int(nx), int(ny), int(item), *[C.byref(o) for o in out], deps))
    return tuple(o.value for o in out) + (list(deps),)


def shard_bounds(n, nranks, rank):
    """afid_shard_bounds: part `rank` of n items, [lo, hi) (host arithmetic, no device)."""
    lo, hi = C.c_int(0), C.c_int(0)
    _check(lib().afid_shard_bounds(int(n), int(nranks), int(rank), C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def shard_layout(nx, ny, nz, nranks, rank, phase):
    """afid_shard_layout: (send_count, send_off, recv_count, recv_off), lists of nranks ints in complex elements
    (host arithmetic, no device)."""
    arr = [(C.c_longlong * nranks)() for _ in range(4)]
    _check(lib().afid_shard_layout(int(nx), int(ny), int(nz), int(nranks), int(rank), int(phase),
                                   *[C.cast(a, C.c_void_p) for a in arr]))
    return tuple([int(x) for x in a] for a in arr)


class _DevView:
    """A raw device allocation as a __cuda_array_interface__ object (so torch can wrap it without a copy)."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (nbytes // 8,), "typestr": "<f8", "data": (int(ptr), False), "version": 3}


class ShardPlan:
    """afid_shard_plan_create and the four stages of a sharded projection for rank `rank` of `nranks`.
    nx is the GLOBAL number of planes, xc the global nx+1 faces; u holds this rank's planes xs..xe (the slab plus
    its upper halo plane), v, w, p the planes xs..xe-1."""

    def __init__(self, nx, ny, nz, xc, Ly, Lz, rank, nranks):
        import numpy as np
        xc = np.ascontiguousarray(xc, dtype=np.float64)
        if xc.size != nx + 1:
            raise ValueError("xc must hold nx+1 face coordinates")
        self.gnx, self.ny, self.nz, self.rank, self.nranks = int(nx), int(ny), int(nz), int(rank), int(nranks)
        self.nzh = self.nz // 2 + 1
        self._h = lib().afid_shard_plan_create(self.gnx, self.ny, self.nz, xc.ctypes.data_as(C.c_void_p), float(Ly), float(Lz),
                                               self.rank, self.nranks)
        if not self._h:
            raise AfidError(*_last_error())
        v = [C.c_int(0) for _ in range(6)]
        _check(lib().afid_shard_info(self._h, *[C.byref(x) for x in v]))
        _, _, self.xs, self.xe, self.ks, self.ke = [x.value for x in v]
        self.nxl, self.nkz = self.xe - self.xs, self.ke - self.ks
        self.layout = {ph: shard_layout(self.gnx, self.ny, self.nz, self.nranks, self.rank, ph) for ph in (1, 2)}

    _stream = Plan._stream

    def buffers(self, phase):
        """afid_shard_buffers: (send, recv) as flat complex128 CUDA tensors over the plan's work arrays."""
        import torch
        s, r = C.c_void_p(0), C.c_void_p(0)
        _check(lib().afid_shard_buffers(self._h, int(phase), C.byref(s), C.byref(r)))
        n = max(self.nxl * self.nzh, self.gnx * self.nkz) * self.ny * 16
        dev = torch.device("cuda", torch.cuda.current_device())
        return tuple(torch.view_as_complex(torch.as_tensor(_DevView(x.value, n), device=dev).view(-1, 2)) for x in (s, r))

    def forward(self, u, v, w, stream=None):
        n = self.nxl * self.ny * self.nz
        _check(lib().afid_shard_forward(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"), _dev_ptr(w, n, "w"),
                                        self._stream(stream)))

    def solve(self, stream=None):
        _check(lib().afid_shard_solve(self._h, self._stream(stream)))

    def inverse(self, p, stream=None):
        _check(lib().afid_shard_inverse(self._h, _dev_ptr(p, self.nxl * self.ny * self.nz, "p"), self._stream(stream)))

    def correct(self, u, v, w, p, p_halo, stream=None):
        n = self.nxl * self.ny * self.nz
        ph = C.c_void_p(0) if p_halo is None else _dev_ptr(p_halo, self.ny * self.nz, "p_halo")
        _check(lib().afid_shard_correct(self._h, _dev_ptr(u, n + self.ny * self.nz, "u"), _dev_ptr(v, n, "v"), _dev_ptr(w, n, "w"),
                                        _dev_ptr(p, n, "p"), ph, self._stream(stream)))

    def exchange(self, phase, group=None):
        """The all-to-all of `phase` over torch.distributed (NCCL): plumbing only, the blocks are already laid out."""
        import torch.distributed as dist
        sc, so, rc, ro = self.layout[phase]
        send, recv = self.buffers(phase)
        # the per-peer blocks are back to back in rank order, so the split sizes describe them completely
        dist.all_to_all_single(recv[:sum(rc)], send[:sum(sc)], output_split_sizes=rc, input_split_sizes=sc, group=group)

    def project(self, u, v, w, p, group=None):
        """One sharded projection on this rank (all ranks of `group` call it): stages, two exchanges, phi halo."""
        import torch
        import torch.distributed as dist
        self.forward(u, v, w)
        self.exchange(1, group)
        self.solve()
        self.exchange(2, group)
        self.inverse(p)
        halo = None
        ops = []
        if self.rank + 1 < self.nranks:
            ops.append(dist.P2POp(dist.isend, p[self.nxl - 1].contiguous(), self.rank + 1, group))
        if self.rank > 0:
            halo = torch.empty((self.ny, self.nz), dtype=torch.float64, device=p.device)
            ops.append(dist.P2POp(dist.irecv, halo, self.rank - 1, group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        self.correct(u, v, w, p, halo)

    def destroy(self):
        if getattr(self, "_h", None):
            lib().afid_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
