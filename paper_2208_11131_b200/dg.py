"""Thin ctypes binding of the C-ABI in include/dg.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libdg_b200.so; this module never computes.  PyTorch
is used for device memory (the solver workspace is one torch tensor) and for the stream the work runs on.
If the library is missing it is built with nvcc (paper_2208_11131_b200.build); if that is impossible the
import of the library fails loudly -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

DG_OK, DG_EINVAL, DG_ENOMEM, DG_EUNPHYSICAL, DG_ECUDA = 0, -1, -2, -3, -4

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdg_b200.so")
_lib = None


class DGError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("dg error %d: %s" % (code, text))
        self.code = code


class dg_mesh(C.Structure):
    _fields_ = [("dim", C.c_int), ("ncell", C.c_int * 3), ("origin", C.c_double * 3), ("h", C.c_double),
                ("periodic", C.c_int * 3)]


class dg_options(C.Structure):
    _fields_ = [("f_cfl", C.c_double), ("rk_stages", C.c_int), ("av_enable", C.c_int), ("f_v", C.c_double),
                ("f_tau", C.c_double), ("f_w", C.c_double), ("s_onset0", C.c_double), ("alpha_max", C.c_double),
                ("fixed_dt", C.c_double), ("use_graph", C.c_int), ("limiter_enable", C.c_int), ("basis", C.c_int),
                ("tracer_enable", C.c_int), ("eta", C.c_double)]


class dg_diagnostics(C.Structure):
    _fields_ = [("t", C.c_double), ("last_dt", C.c_double), ("c_max", C.c_double), ("v_max", C.c_double),
                ("alpha_max_seen", C.c_double), ("steps", C.c_longlong), ("unphysical", C.c_int)]


# every symbol include/dg.h declares: name -> (restype, argtypes)
_P = C.c_void_p
SYMBOLS = {
    "dg_default_options": (C.c_int, [C.POINTER(dg_options)]),
    "dg_init": (C.c_int, [C.POINTER(_P), C.POINTER(dg_mesh), C.c_int, C.c_double, C.c_double, C.c_double,
                          C.POINTER(dg_options)]),
    "dg_workspace_bytes": (C.c_int, [C.POINTER(dg_mesh), C.c_int, C.POINTER(dg_options), C.POINTER(C.c_size_t)]),
    "dg_init_workspace": (C.c_int, [C.POINTER(_P), C.POINTER(dg_mesh), C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.POINTER(dg_options), _P, C.c_size_t]),
    "dg_set_stream": (C.c_int, [_P, _P]),
    "dg_set_state": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_set_alpha": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_step": (C.c_int, [_P, C.c_int]),
    "dg_step_async": (C.c_int, [_P, C.c_int]),
    "dg_sync": (C.c_int, [_P]),
    "dg_get_state": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_get_alpha": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_conserved_totals": (C.c_int, [_P, C.POINTER(C.c_double * 5)]),
    "dg_tracer_total": (C.c_int, [_P, C.POINTER(C.c_double)]),
    "dg_eval_rhs": (C.c_int, [_P, _P, C.c_size_t, _P, C.c_size_t]),
    "dg_get_time": (C.c_int, [_P, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "dg_set_options": (C.c_int, [_P, C.POINTER(dg_options)]),
    "dg_get_diagnostics": (C.c_int, [_P, C.POINTER(dg_diagnostics)]),
    "dg_get_sensor": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_set_sensor": (C.c_int, [_P, _P, C.c_size_t]),
    "dg_set_time": (C.c_int, [_P, C.c_double]),
    "dg_kernel_info": (C.c_int, [_P, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "dg_profile_stage": (C.c_int, [_P, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "dg_apply_limiter": (C.c_int, [_P]),
    "dg_launch_count": (C.c_int, [_P, C.POINTER(C.c_longlong)]),
    "dg_measure_fp64_peak": (C.c_int, [C.c_int, C.POINTER(C.c_double), _P]),
    "dg_totals_noalloc": (C.c_int, [_P, C.c_int, C.c_longlong, C.c_double, _P, _P]),
    "dg_free": (C.c_int, [_P]),
    "dg_last_error": (C.c_char_p, []),
}


def load_library(build_if_missing: bool = True):
    """dlopen libdg_b200.so (building it first if needed) and set the ctypes prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        if not build_if_missing:
            raise OSError("libdg_b200.so is not built (run `python -m paper_2208_11131_b200.build`)")
        from . import build as _build
        _build.build()
    lib = C.CDLL(_LIB_PATH)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)   # AttributeError if the library does not export a declared symbol
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _check(rc):
    if rc != DG_OK:
        raise DGError(rc, load_library().dg_last_error().decode())


def default_options(**kw) -> dg_options:
    o = dg_options()
    _check(load_library().dg_default_options(C.byref(o)))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError("unknown option " + k)
        setattr(o, k, v)
    return o


def _buf(x):
    """(pointer, element count, keep-alive) of a float64 numpy array (host) or torch tensor (host or cuda)."""
    if isinstance(x, np.ndarray):
        if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"]:
            raise TypeError("numpy buffers must be C-contiguous float64")
        return x.ctypes.data, x.size, x
    import torch
    if isinstance(x, torch.Tensor):
        if x.dtype != torch.float64 or not x.is_contiguous():
            raise TypeError("torch buffers must be contiguous float64")
        return x.data_ptr(), x.numel(), x
    raise TypeError("expected a numpy array or a torch tensor")


class Solver:
    """One dg_solver handle.  Method names mirror the C-ABI (dg_set_state -> set_state, ...)."""

    def __init__(self, dim, ncell, h, order, gamma, nu=0.0, chi=0.0, options: dg_options | None = None,
                 origin=(0.0, 0.0, 0.0), device="cuda:0", torch_workspace=True):
        lib = load_library()
        self._lib = lib
        self._h = _P()
        self.dim, self.order, self.h = int(dim), int(order), float(h)
        self.ncell = tuple(int(c) for c in ncell[:dim])
        self.ncells = int(np.prod(self.ncell))
        self.M = order ** dim
        self.opt = options if options is not None else default_options()
        self.Vc = dim + 2 + (1 if self.opt.tracer_enable else 0)
        mesh = dg_mesh()
        mesh.dim = dim
        for a in range(3):
            mesh.ncell[a] = self.ncell[a] if a < dim else 1
            mesh.origin[a] = origin[a] if a < len(origin) else 0.0
            mesh.periodic[a] = 1
        mesh.h = h
        self._ws = None
        if torch_workspace:
            import torch
            if not torch.cuda.is_available():
                raise DGError(DG_ECUDA, "no CUDA device: the DG hot path has no CPU fallback")
            need = C.c_size_t()
            _check(lib.dg_workspace_bytes(C.byref(mesh), order, C.byref(self.opt), C.byref(need)))
            self._ws = torch.empty(need.value + 256, dtype=torch.uint8, device=device)
            ptr = (self._ws.data_ptr() + 255) // 256 * 256
            _check(lib.dg_init_workspace(C.byref(self._h), C.byref(mesh), order, gamma, nu, chi, C.byref(self.opt),
                                         ptr, need.value))
            self.set_stream(torch.cuda.current_stream(self._ws.device).cuda_stream)
        else:
            _check(lib.dg_init(C.byref(self._h), C.byref(mesh), order, gamma, nu, chi, C.byref(self.opt)))

    # ---- C-ABI calls ----
    def set_stream(self, cuda_stream: int):
        _check(self._lib.dg_set_stream(self._h, cuda_stream))

    def set_state(self, w):
        p, n, _keep = _buf(w)
        _check(self._lib.dg_set_state(self._h, p, n))

    def set_alpha(self, alpha):
        p, n, _keep = _buf(alpha)
        _check(self._lib.dg_set_alpha(self._h, p, n))

    def step(self, nsteps=1):
        _check(self._lib.dg_step(self._h, nsteps))

    def step_async(self, nsteps=1):
        _check(self._lib.dg_step_async(self._h, nsteps))

    def sync(self):
        _check(self._lib.dg_sync(self._h))

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.Vc * self.M * self.ncells)
        p, n, _keep = _buf(out)
        _check(self._lib.dg_get_state(self._h, p, n))
        return out

    def get_alpha(self, out=None):
        if out is None:
            out = np.empty(self.M * self.ncells)
        p, n, _keep = _buf(out)
        _check(self._lib.dg_get_alpha(self._h, p, n))
        return out

    def conserved_totals(self):
        t = (C.c_double * 5)()
        _check(self._lib.dg_conserved_totals(self._h, C.byref(t)))
        return np.array(t[:self.dim + 2])

    def tracer_total(self):
        t = C.c_double()
        _check(self._lib.dg_tracer_total(self._h, C.byref(t)))
        return t.value

    def eval_rhs(self, with_alpha=False, out=None, alpha_out=None):
        """dw/dt of the current state.  `out` / `alpha_out` may be numpy arrays or torch tensors (host or cuda)."""
        if out is None:
            out = np.empty(self.Vc * self.M * self.ncells)
        if alpha_out is None and with_alpha:
            alpha_out = np.empty(self.M * self.ncells)
        po, no, _ = _buf(out)
        pa, na = None, 0
        if alpha_out is not None:
            pa, na, _ = _buf(alpha_out)
        _check(self._lib.dg_eval_rhs(self._h, po, no, pa, na))
        return (out, alpha_out) if alpha_out is not None else out

    def get_time(self):
        t, dt = C.c_double(), C.c_double()
        _check(self._lib.dg_get_time(self._h, C.byref(t), C.byref(dt)))
        return t.value, dt.value

    def set_options(self, **kw):
        """dg_set_options with the keyword arguments applied to a copy of the current options; `self.opt` changes only
        when the library has accepted them (a rejected call leaves the binding and the solver in agreement)."""
        new = dg_options()
        C.memmove(C.byref(new), C.byref(self.opt), C.sizeof(dg_options))
        for k, v in kw.items():
            if not hasattr(new, k):
                raise TypeError("unknown option " + k)
            setattr(new, k, v)
        _check(self._lib.dg_set_options(self._h, C.byref(new)))
        self.opt = new

    def diagnostics(self):
        d = dg_diagnostics()
        _check(self._lib.dg_get_diagnostics(self._h, C.byref(d)))
        return {k: getattr(d, k) for k, _ in dg_diagnostics._fields_}

    def get_sensor(self, out=None):
        if out is None:
            out = np.empty(2 * self.ncells)
        p, n, _keep = _buf(out)
        _check(self._lib.dg_get_sensor(self._h, p, n))
        return out

    def set_sensor(self, sg):
        p, n, _keep = _buf(sg)
        _check(self._lib.dg_set_sensor(self._h, p, n))

    def set_time(self, t):
        _check(self._lib.dg_set_time(self._h, float(t)))

    def kernel_info(self):
        c, nt, sm, nb = C.c_int(), C.c_int(), C.c_int(), C.c_int()
        _check(self._lib.dg_kernel_info(self._h, C.byref(c), C.byref(nt), C.byref(sm), C.byref(nb)))
        return dict(cells_per_block=c.value, threads=nt.value, smem_bytes=sm.value, blocks=nb.value)

    def profile_stage(self, reps=3):
        """(face_ms, stage_ms): device time of the two kernels of one RK stage (CUDA events on the solver stream)."""
        f, g = C.c_double(), C.c_double()
        _check(self._lib.dg_profile_stage(self._h, reps, C.byref(f), C.byref(g)))
        return f.value, g.value

    def apply_limiter(self):
        _check(self._lib.dg_apply_limiter(self._h))

    def launch_count(self):
        n = C.c_longlong()
        _check(self._lib.dg_launch_count(self._h, C.byref(n)))
        return n.value

    def free(self):
        if self._h:
            self._lib.dg_free(self._h)
            self._h = _P()
        self._ws = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def measure_fp64_peak(iters=4096, cuda_stream=0):
    v = C.c_double()
    _check(load_library().dg_measure_fp64_peak(iters, C.byref(v), cuda_stream))
    return v.value


NOALLOC_MAX_CELLS, NOALLOC_MAX_VARS = 4194304, 8     # DG_NOALLOC_MAX_CELLS / DG_NOALLOC_MAX_VARS of include/dg.h


def totals_noalloc(w, nvars, ncells, cell_volume, out=None, cuda_stream=None):
    """dg_totals_noalloc: cell_volume * sum over cells of the cell means of the first `nvars` variables of the modal
    state `w`, for callers that may not allocate device memory (a hook on a GPU somebody else has filled, code inside
    a pool that owns the card, a process under a memory cap): the library's built-in scratch array is used, no
    solver handle and no workspace are needed, and meshes beyond NOALLOC_MAX_CELLS are refused.

    `w` is a cuda float64 tensor in the C-ABI state layout (at least nvars*ncells elements; only mode 0 is read);
    `out` (nvars float64 values) may be a numpy array, a host tensor or a cuda tensor -- with a cuda tensor nothing
    is waited for, and with out=None a new numpy array is returned.  The first call on a device should happen
    outside stream capture; calls that overlap on the GPU share the scratch array and race (see include/dg.h)."""
    pw, nw, _keep = _buf(w)
    if nw < int(nvars) * int(ncells):
        raise ValueError("w holds fewer than nvars*ncells values")
    if out is None:
        out = np.empty(int(nvars))
    po, no, _keep2 = _buf(out)
    if no < int(nvars):
        raise ValueError("out holds fewer than nvars values")
    if cuda_stream is None:
        import torch
        cuda_stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    _check(load_library().dg_totals_noalloc(pw, int(nvars), int(ncells), float(cell_volume), po, cuda_stream))
    return out


def from_workload(wl, **opt_kw) -> Solver:
    """Solver for a workloads.Workload (mesh, physics switches, Courant factor)."""
    opt = default_options(f_cfl=wl.f_cfl, av_enable=1 if wl.av else 0, **opt_kw)
    return Solver(wl.dim, wl.ncell, wl.h, wl.order, wl.gamma, wl.nu, wl.chi, opt, origin=wl.origin)
