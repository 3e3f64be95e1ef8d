"""Thin Python binding of libdr (include/dr.h): argument marshalling only.

PyTorch supplies device memory (workspace, K/G, exported fields) and the CUDA stream; every step of the
path runs in the library's kernels.  There is no fallback: if libdr.so cannot be loaded or no CUDA device
is present, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DR_LIB") or os.path.join(_HERE, "libdr.so")     # DR_LIB: an alternative build (A/B timing)

OK, ERR_ARG, ERR_WORKSPACE, ERR_CUDA, ERR_DIVERGED, ERR_STATE, MAXITER = range(7)
CFL, ST_FACTOR, NCHECK, GAVG, VOID_REL, BC_MODE, KERNEL, ZCHUNK, FORM, PALETTE, STAG_TOL = range(11)
STOP_NONE, STOP_RESIDUAL, STOP_STAGNATION, STOP_MAXITER = range(4)
PARAM_IDS = dict(cfl=CFL, st_factor=ST_FACTOR, ncheck=NCHECK, gavg=GAVG, void_rel=VOID_REL, bc_mode=BC_MODE, kernel=KERNEL, zchunk=ZCHUNK, form=FORM, palette=PALETTE, stag_tol=STAG_TOL)
FIELDS = ("vx", "vy", "vz", "sxx", "syy", "szz", "tyz", "txz", "txy")
EXPORTS = ("dr_workspace_bytes", "dr_workspace_bytes_six", "dr_solve_all", "dr_info_lc", "dr_create", "dr_create_segmented", "dr_solve_image_host_segmented", "dr_set_param", "dr_solve", "dr_solve_six", "dr_effective_C_six", "dr_step", "dr_iterate",
           "dr_effective_C", "dr_avg_stress", "dr_offdiag_direct", "dr_info", "dr_get_field", "dr_solve_image_host", "dr_contribution_tensor",
           "dr_uses_palette", "dr_active_kernel", "dr_stop_reason", "dr_launch_count", "dr_last_error", "dr_destroy", "dr_avg_stress_static")
STATIC_MAX_ROWS = 1048576          # DR_STATIC_MAX_ROWS of include/dr.h

_lib = None


def lib():
    """Load libdr.so (built in-tree by paper_2410_20441_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libdr.so is not built: run `python -m paper_2410_20441_b200.build` "
                               "(needs nvcc; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        dp, vp = C.POINTER(C.c_double), C.c_void_p
        L.dr_workspace_bytes.argtypes = [C.c_int] * 3
        L.dr_workspace_bytes.restype = C.c_size_t
        if hasattr(L, "dr_workspace_bytes_six"):
            L.dr_workspace_bytes_six.argtypes = [C.c_int] * 3
            L.dr_workspace_bytes_six.restype = C.c_size_t
            L.dr_solve_all.argtypes = [vp, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_int)]
            L.dr_info_lc.argtypes = [vp, C.c_int, C.POINTER(C.c_int), dp, C.POINTER(C.c_int)]
        L.dr_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, vp, vp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.dr_set_param.argtypes = [vp, C.c_int, C.c_double]
        L.dr_solve.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_int]
        L.dr_step.argtypes = [vp, C.c_int, C.c_double, C.c_int]
        if hasattr(L, "dr_solve_six"):          # absent only in older builds loaded through DR_LIB for A/B timing
            L.dr_solve_six.argtypes = [C.POINTER(vp), C.c_double, C.c_double, C.c_int, C.POINTER(C.c_int)]
            L.dr_effective_C_six.argtypes = [C.POINTER(vp), dp]
        L.dr_iterate.argtypes = [vp, C.c_int, C.c_double, C.c_int]
        L.dr_effective_C.argtypes = [vp, dp]
        L.dr_avg_stress.argtypes = [vp, dp]
        if hasattr(L, "dr_offdiag_direct"):
            L.dr_offdiag_direct.argtypes = [vp, dp]
        L.dr_info.argtypes = [vp, C.POINTER(C.c_int), dp, dp]
        L.dr_get_field.argtypes = [vp, C.c_int, vp, C.c_size_t]
        if hasattr(L, "dr_create_segmented"):
            L.dr_create_segmented.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, vp, C.c_int, dp, dp, vp, C.c_size_t, vp, C.POINTER(vp)]
            L.dr_solve_image_host_segmented.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, vp, C.c_int, dp, dp, vp, vp, C.c_size_t, vp,
                                                        C.c_double, C.c_double, C.c_int, C.c_int, dp, C.POINTER(C.c_int)]
        L.dr_solve_image_host.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, vp, vp, vp, vp, C.c_size_t, vp,
                                          C.c_double, C.c_double, C.c_int, C.c_int, dp, C.POINTER(C.c_int)]
        if hasattr(L, "dr_contribution_tensor"):
            L.dr_contribution_tensor.argtypes = [dp, dp, C.c_double, dp]
        if hasattr(L, "dr_uses_palette"):
            L.dr_uses_palette.argtypes = [vp]
        if hasattr(L, "dr_active_kernel"):
            L.dr_active_kernel.argtypes = [vp]
        if hasattr(L, "dr_stop_reason"):
            L.dr_stop_reason.argtypes = [vp]
        if hasattr(L, "dr_avg_stress_static"):
            L.dr_avg_stress_static.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(vp), vp, vp, C.c_char_p, C.c_size_t]
        L.dr_launch_count.argtypes = [vp]
        L.dr_launch_count.restype = C.c_longlong
        L.dr_last_error.argtypes = [vp]
        L.dr_last_error.restype = C.c_char_p
        L.dr_destroy.argtypes = [vp]
        L.dr_destroy.restype = None
        _lib = L
    return _lib


class DrError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("libdr status %d: %s" % (status, msg))
        self.status = status


def workspace_bytes(nx, ny, nz, six=False):
    return lib().dr_workspace_bytes_six(nx, ny, nz) if six else lib().dr_workspace_bytes(nx, ny, nz)


def field_shape(nx, ny, nz, f):
    return {0: (nz, ny, nx + 1), 1: (nz, ny + 1, nx), 2: (nz + 1, ny, nx),
            3: (nz, ny, nx), 4: (nz, ny, nx), 5: (nz, ny, nx),
            6: (nz + 1, ny + 1, nx), 7: (nz + 1, ny, nx + 1), 8: (nz, ny + 1, nx + 1)}[f]


class Solver:
    """dr_create .. dr_destroy.  K, G: torch.float64 CUDA tensors of shape (nz, ny, nx), x fastest."""

    def __init__(self, K, G, h=1.0, stream=None, workspace=None, six=False, phase=None, **params):
        """K, G: the modulus fields -- or, with phase= (torch.uint8 CUDA tensor (nz, ny, nx) of phase ids), the per-phase
        tables (sequences of nphase floats): dr_create_segmented."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libdr needs a CUDA device (there is no CPU fallback)")
        if phase is not None:
            if not (phase.is_cuda and phase.dtype == torch.uint8 and phase.dim() == 3):
                raise TypeError("phase must be a uint8 CUDA tensor of shape (nz, ny, nx)")
            import numpy as np
            Kt = np.ascontiguousarray(K, dtype=np.float64).ravel()
            Gt = np.ascontiguousarray(G, dtype=np.float64).ravel()
            assert Kt.size == Gt.size
            K = phase
        elif not (K.is_cuda and G.is_cuda and K.dtype == torch.float64 and G.dtype == torch.float64):
            raise TypeError("K and G must be float64 CUDA tensors")
        else:
            assert K.shape == G.shape
        assert K.dim() == 3
        self.nz, self.ny, self.nx = (int(s) for s in K.shape)
        self.device = K.device
        self._torch = torch
        need = workspace_bytes(self.nx, self.ny, self.nz, six)
        if need == 0:
            raise DrError(ERR_ARG, "invalid grid size")
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=K.device)
        self.workspace = workspace
        self.stream = stream if stream is not None else torch.cuda.current_stream(K.device)
        self._h = C.c_void_p()
        # dr_create reads K, G on self.stream: order it behind whatever produced them on the caller's current stream,
        # and make any contiguous() copy on self.stream too
        self.stream.wait_stream(torch.cuda.current_stream(K.device))
        with torch.cuda.device(K.device), torch.cuda.stream(self.stream):
            K = K.contiguous()
            if phase is not None:
                dp = C.POINTER(C.c_double)
                st = lib().dr_create_segmented(self.nx, self.ny, self.nz, float(h), K.data_ptr(), int(Kt.size),
                                               Kt.ctypes.data_as(dp), Gt.ctypes.data_as(dp),
                                               workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                               self.stream.cuda_stream, C.byref(self._h))
            else:
                G = G.contiguous()
                st = lib().dr_create(self.nx, self.ny, self.nz, float(h), K.data_ptr(), G.data_ptr(),
                                     workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                     self.stream.cuda_stream, C.byref(self._h))
        if st != OK:
            raise DrError(st, "dr_create failed (status %d)" % st)
        for k, v in params.items():
            self.set_param(k, v)

    def _check(self, st, soft=(OK,)):
        if st not in soft:
            raise DrError(st, lib().dr_last_error(self._h).decode())
        return st

    def set_param(self, name, value):
        self._check(lib().dr_set_param(self._h, PARAM_IDS[name], float(value)))

    def solve(self, lc, eps0=1e-4, tol=1e-8, maxiter=100000):
        return self._check(lib().dr_solve(self._h, lc, eps0, tol, maxiter), soft=(OK, MAXITER))

    def step(self, lc, eps0, niter):
        return self._check(lib().dr_step(self._h, lc, eps0, niter))

    def iterate(self, lc, eps0, niter):
        return self._check(lib().dr_iterate(self._h, lc, eps0, niter))

    def effective_C(self):
        import numpy as np
        out = np.zeros(36)
        self._check(lib().dr_effective_C(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out.reshape(6, 6)

    def avg_stress(self):
        import numpy as np
        out = np.zeros(6)
        self._check(lib().dr_avg_stress(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def offdiag_direct(self):
        """dr_offdiag_direct: (C12, C13, C23) by Eq. 27-29 from the triaxial test (load case 6) and load cases 0-2"""
        import numpy as np
        out = np.zeros(3)
        self._check(lib().dr_offdiag_direct(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def info(self):
        it, r, ms = C.c_int(), C.c_double(), C.c_double()
        lib().dr_info(self._h, C.byref(it), C.byref(r), C.byref(ms))
        return it.value, r.value, ms.value

    def get_field(self, f):
        if isinstance(f, str):
            f = FIELDS.index(f)
        out = self._torch.empty(field_shape(self.nx, self.ny, self.nz, f), dtype=self._torch.float64, device=self.device)
        self._check(lib().dr_get_field(self._h, f, out.data_ptr(), out.numel()))
        return out

    def stop_reason(self):
        return lib().dr_stop_reason(self._h)

    def active_kernel(self):
        return lib().dr_active_kernel(self._h)

    def uses_palette(self):
        return bool(lib().dr_uses_palette(self._h))

    def launch_count(self):
        return lib().dr_launch_count(self._h)

    def solve_all_batched(self, eps0=1e-4, tol=1e-8, maxiter=100000):
        """dr_solve_all: six load cases per launch (Solver(..., six=True)).  Returns (C[6,6], [(status, iters, residual, stop)]*6)."""
        stat = (C.c_int * 6)()
        self._check(lib().dr_solve_all(self._h, eps0, tol, maxiter, stat), soft=(OK, MAXITER))
        log = []
        for lc in range(6):
            it, r, sp = C.c_int(), C.c_double(), C.c_int()
            lib().dr_info_lc(self._h, lc, C.byref(it), C.byref(r), C.byref(sp))
            log.append((stat[lc], it.value, r.value, sp.value))
        return self.effective_C(), log

    def solve_all(self, eps0=1e-4, tol=1e-8, maxiter=100000):
        log = []
        for lc in range(6):
            st = self.solve(lc, eps0, tol, maxiter)
            it, r, ms = self.info()
            log.append((st, it, r, ms, self.stop_reason()))
        return self.effective_C(), log

    def close(self):
        if getattr(self, "_h", None) and self._h:
            lib().dr_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def avg_stress_static(fields, out=None, stream=None):
    """dr_avg_stress_static: <sigma> (Eq. 7) of six dense stress fields with no handle, no workspace and no allocation inside the
    library -- for callers that cannot allocate device memory (a hook beside a running solve, where cudaMalloc would stall the
    device; a plug-in whose host owns the free memory).  The scratch is a 6 MiB array inside libdr.so, shared by all calls:
    keep them on one stream.  Limit (ny+1)*(nz+1) <= STATIC_MAX_ROWS, else DrError(ERR_ARG) naming the limit.

    fields: the six float64 CUDA tensors Solver.get_field(3..8) returns (sxx, syy, szz, tyz, txz, txy).  out: float64 CUDA
    tensor of 6 elements; a caller that must not allocate passes its own (None: torch allocates one here, outside the library).
    Enqueues on `stream` (default: torch's current stream) and does not synchronise; returns out."""
    import torch
    assert len(fields) == 6
    nz, ny, nx = (int(s) for s in fields[0].shape)
    for f, t in zip(range(3, 9), fields):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == field_shape(nx, ny, nz, f)):
            raise TypeError("field %s must be a contiguous float64 CUDA tensor of shape %s" % (FIELDS[f], (field_shape(nx, ny, nz, f),)))
    dev = fields[0].device
    if out is None:
        out = torch.empty(6, dtype=torch.float64, device=dev)
    elif not (out.is_cuda and out.device == dev and out.dtype == torch.float64 and out.numel() == 6 and out.is_contiguous()):
        raise TypeError("out must be a contiguous float64 tensor of 6 elements on the device of the fields")
    ptrs = (C.c_void_p * 6)(*[t.data_ptr() for t in fields])
    err = C.create_string_buffer(512)
    with torch.cuda.device(dev):
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib().dr_avg_stress_static(nx, ny, nz, ptrs, out.data_ptr(), st.cuda_stream, err, len(err))
    if rc != OK:
        raise DrError(rc, err.value.decode())
    return out


def contribution_tensor(C_eff, C_matrix, phi):
    """dr_contribution_tensor: H = (inv(C_eff) - inv(C_matrix)) / phi (Eq. 23 of the paper), 6x6 numpy arrays."""
    import numpy as np
    a = np.ascontiguousarray(C_eff, dtype=np.float64).reshape(36)
    b = np.ascontiguousarray(C_matrix, dtype=np.float64).reshape(36)
    out = np.zeros(36)
    dp = C.POINTER(C.c_double)
    st = lib().dr_contribution_tensor(a.ctypes.data_as(dp), b.ctypes.data_as(dp), float(phi), out.ctypes.data_as(dp))
    if st != OK:
        raise DrError(st, "dr_contribution_tensor: bad argument or singular matrix")
    return out.reshape(6, 6)


def solve_six(K, G, h=1.0, eps0=1e-4, tol=1e-8, maxiter=100000, **params):
    """dr_solve_six: six Solver handles (own workspace, own torch stream each), load case lc on handle lc.
    Returns (C[6,6], [(status, iters, residual)]*6, solvers)."""
    import numpy as np
    import torch
    cur = torch.cuda.current_stream(K.device)
    solvers = []
    for lc in range(6):
        st = torch.cuda.Stream(device=K.device)
        st.wait_stream(cur)
        solvers.append(Solver(K, G, h=h, stream=st, **params))
    arr = (C.c_void_p * 6)(*[s._h for s in solvers])
    stat = (C.c_int * 6)()
    with torch.cuda.device(K.device):
        rc = lib().dr_solve_six(arr, eps0, tol, maxiter, stat)
    if rc not in (OK, MAXITER):
        raise DrError(rc, "dr_solve_six failed: " + "; ".join(lib().dr_last_error(s._h).decode() for s in solvers))
    out = np.zeros(36)
    rc2 = lib().dr_effective_C_six(arr, out.ctypes.data_as(C.POINTER(C.c_double)))
    if rc2 != OK:
        raise DrError(rc2, "dr_effective_C_six failed")
    log = [(stat[lc],) + solvers[lc].info()[:2] for lc in range(6)]
    return out.reshape(6, 6), log, solvers


def solve_image_host(K_host, G_host, h=1.0, eps0=1e-4, tol=1e-8, maxiter=100000, ncheck=0,
                     stage=None, workspace=None, device="cuda:0", six=False):
    """End-to-end call with HOST arrays (numpy or CPU torch tensors, (nz,ny,nx) float64): host->device copies,
    six solves and the 6x6 result read back, all inside dr_solve_image_host.  Returns (C, iters, status)."""
    import numpy as np
    import torch
    Kt = torch.as_tensor(K_host)
    Gt = torch.as_tensor(G_host)
    assert Kt.dtype == torch.float64 and Kt.is_contiguous() and Gt.is_contiguous() and not Kt.is_cuda
    nz, ny, nx = (int(s) for s in Kt.shape)
    N = nx * ny * nz
    if stage is None:
        stage = torch.empty(2 * N, dtype=torch.float64, device=device)
    if workspace is None:
        workspace = torch.empty(workspace_bytes(nx, ny, nz, six), dtype=torch.uint8, device=device)
    Cout = np.zeros(36)
    iters = (C.c_int * 6)()
    with torch.cuda.device(stage.device):
        st = lib().dr_solve_image_host(nx, ny, nz, float(h), Kt.data_ptr(), Gt.data_ptr(), stage.data_ptr(),
                                       workspace.data_ptr(), workspace.numel(), torch.cuda.current_stream().cuda_stream,
                                       eps0, tol, maxiter, ncheck, Cout.ctypes.data_as(C.POINTER(C.c_double)), iters)
    if st not in (OK, MAXITER):
        raise DrError(st, "dr_solve_image_host failed")
    return Cout.reshape(6, 6), list(iters), st


def solve_image_host_segmented(phase_host, K_table, G_table, h=1.0, eps0=1e-4, tol=1e-8, maxiter=100000, ncheck=0,
                               stage=None, workspace=None, device="cuda:0", six=False):
    """dr_solve_image_host_segmented: HOST uint8 phase ids (numpy or CPU torch tensor, (nz,ny,nx)) + per-phase tables.
    Returns (C, iters, status)."""
    import numpy as np
    import torch
    Pt = torch.as_tensor(phase_host)
    assert Pt.dtype == torch.uint8 and Pt.is_contiguous() and not Pt.is_cuda and Pt.dim() == 3
    nz, ny, nx = (int(s) for s in Pt.shape)
    N = nx * ny * nz
    Kt = np.ascontiguousarray(K_table, dtype=np.float64).ravel()
    Gt = np.ascontiguousarray(G_table, dtype=np.float64).ravel()
    assert Kt.size == Gt.size
    if stage is None:
        stage = torch.empty(N, dtype=torch.uint8, device=device)
    if workspace is None:
        workspace = torch.empty(workspace_bytes(nx, ny, nz, six), dtype=torch.uint8, device=device)
    Cout = np.zeros(36)
    iters = (C.c_int * 6)()
    dp = C.POINTER(C.c_double)
    with torch.cuda.device(stage.device):
        st = lib().dr_solve_image_host_segmented(nx, ny, nz, float(h), Pt.data_ptr(), int(Kt.size), Kt.ctypes.data_as(dp), Gt.ctypes.data_as(dp),
                                                 stage.data_ptr(), workspace.data_ptr(), workspace.numel(), torch.cuda.current_stream().cuda_stream,
                                                 eps0, tol, maxiter, ncheck, Cout.ctypes.data_as(dp), iters)
    if st not in (OK, MAXITER):
        raise DrError(st, "dr_solve_image_host_segmented failed (status %d)" % st)
    return Cout.reshape(6, 6), list(iters), st

