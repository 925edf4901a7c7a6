"""paper_2503_07953_b200 — thin Python binding of the C-ABI library include/mfc_b200.h.

Argument marshalling only: every step of the hot path (cons->prim, WENO5-JS, HLLC, flux divergence,
alpha div(u) source, SSP-RK3 stage + clamp, CFL reduction) runs in the CUDA kernels of
csrc/mfc_b200.cu.  PyTorch supplies device memory and streams.  There is no CPU path: without the
compiled library or without a CUDA device every call raises.
"""
import ctypes as C
import os

from . import build as _build

BC_PERIODIC, BC_EXTRAP, BC_HALO = 0, 1, 2
WENO_JS, WENO_M, WENO_Z = 0, 1, 2
WENO_BY_NAME = {"js": WENO_JS, "m": WENO_M, "z": WENO_Z}
MODEL_ALLAIRE, MODEL_KAPILA = 0, 1
MODEL_BY_NAME = {"allaire": MODEL_ALLAIRE, "kapila": MODEL_KAPILA}
MFC_OK, MFC_ERR_ARG, MFC_ERR_ALLOC, MFC_ERR_CUDA, MFC_ERR_NONPHYSICAL = 0, 1, 2, 3, 4
EXPORTS = ("mfc_init_grid", "mfc_free_grid", "mfc_num_eqns", "mfc_num_cells", "mfc_prim_from_cons", "mfc_rhs",
           "mfc_rhs_dirs", "mfc_rk3_step", "mfc_rk3_steps", "mfc_cfl_dt", "mfc_check", "mfc_rhs_host",
           "mfc_rk3_steps_host", "mfc_advance", "mfc_advance_host", "mfc_set_profiling", "mfc_get_profile",
           "mfc_weno5_values", "mfc_hllc_faces", "mfc_launch_count", "mfc_set_segments", "mfc_last_error", "mfc_set_halo", "mfc_rk3_stage",
           "mfc_stage_input", "mfc_pack_halo", "mfc_measure_fp64", "mfc_rk3_stage_parts", "mfc_cfl_dt_static",
           "mfc_sqrt_ratio_values", "mfc_set_step_graph")
STATIC_MAX_CELLS = 2048 * 16384  # MFC_STATIC_MAX_CELLS of include/mfc_b200.h


KERNEL_CLASSES = ("prim", "sweep_x", "sweep_y", "sweep_z", "rk", "cfl")


class MfcParams(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("dx", C.c_double * 3), ("nfluids", C.c_int),
                ("gamma", C.POINTER(C.c_double)), ("pi_inf", C.POINTER(C.c_double)),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("weno_eps", C.c_double), ("alpha_floor", C.c_double), ("clamp", C.c_int), ("weno", C.c_int), ("model", C.c_int), ("eta", C.c_double),
                ("device", C.c_int), ("stream", C.c_void_p)]


class MfcError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"mfc status {status}: {text}")
        self.status = status


_lib = None


def lib_path():
    return _build.LIB


def lib():
    """Loads (building it first if the sources are newer) libmfc_b200.so.  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build() if os.path.exists(_build.NVCC) else _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing and nvcc is not available: the CUDA library is required (no fallback)")
        L = C.CDLL(path)
        vp, dp = C.c_void_p, C.c_void_p
        L.mfc_init_grid.argtypes = [C.POINTER(MfcParams), C.POINTER(vp)]
        L.mfc_free_grid.argtypes = [vp]
        L.mfc_num_eqns.argtypes = [vp]
        L.mfc_num_cells.argtypes = [vp]; L.mfc_num_cells.restype = C.c_longlong
        L.mfc_prim_from_cons.argtypes = [vp, dp, dp]
        L.mfc_rhs.argtypes = [vp, dp, dp]
        L.mfc_rhs_dirs.argtypes = [vp, dp, dp, C.c_int]
        L.mfc_rk3_step.argtypes = [vp, dp, C.c_double]
        L.mfc_rk3_steps.argtypes = [vp, dp, C.c_double, C.c_int]
        L.mfc_cfl_dt.argtypes = [vp, dp, C.c_double, C.POINTER(C.c_double)]
        L.mfc_check.argtypes = [vp]
        L.mfc_rhs_host.argtypes = [vp, dp, dp]
        L.mfc_rk3_steps_host.argtypes = [vp, dp, C.c_double, C.c_int]
        L.mfc_advance.argtypes = [vp, dp, C.c_double, C.c_int, C.POINTER(C.c_double)]
        L.mfc_advance_host.argtypes = [vp, dp, C.c_double, C.c_int, C.POINTER(C.c_double)]
        L.mfc_set_profiling.argtypes = [vp, C.c_int]
        L.mfc_get_profile.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.mfc_weno5_values.argtypes = [vp, dp, C.c_longlong, dp, dp]
        L.mfc_hllc_faces.argtypes = [vp, C.c_int, dp, dp, C.c_longlong, dp, dp]
        L.mfc_launch_count.argtypes = [vp]; L.mfc_launch_count.restype = C.c_longlong
        L.mfc_set_segments.argtypes = [vp, C.c_int, C.c_int, C.c_int]
        L.mfc_set_step_graph.argtypes = [vp, C.c_int]
        L.mfc_last_error.restype = C.c_char_p
        L.mfc_set_halo.argtypes = [vp, dp, dp]
        L.mfc_rk3_stage.argtypes = [vp, dp, C.c_double, C.c_int]
        L.mfc_rk3_stage_parts.argtypes = [vp, dp, C.c_double, C.c_int, C.c_int]
        L.mfc_stage_input.argtypes = [vp, dp, C.c_int, C.POINTER(C.c_void_p)]
        L.mfc_pack_halo.argtypes = [vp, dp, C.c_int, dp, dp]
        L.mfc_measure_fp64.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mfc_sqrt_ratio_values.argtypes = [vp, dp, dp, C.c_longlong, dp, dp]
        L.mfc_cfl_dt_static.argtypes = [C.POINTER(MfcParams), dp, C.c_double, dp, dp]
        _lib = L
    return _lib


def measure_fp64(device=0):
    """(TFLOP/s of DFMA chains with two loop-invariant operands, with three distinct register operands) on `device`"""
    a, b = C.c_double(), C.c_double()
    _ck(lib().mfc_measure_fp64(int(device), None, C.byref(a), C.byref(b)))
    return a.value, b.value


def cfl_dt_static(ndim, n, dx, gamma, pi_inf, q, cfl, dt_out, nonphysical_out=None, device=0, stream=None):
    """mfc_cfl_dt_static: the CFL time step of state q without a Grid and without any allocation by the library.

    For callers that cannot let the library allocate — a solver embedded in an application whose memory pool already
    holds all of the GPU's memory, or a step loop in which an allocation would stall the device.  The reduction's
    scratch is an array built into the library (129 KiB per GPU), which is why grids above STATIC_MAX_CELLS (2^25)
    cells are refused, and why two calls that overlap on one GPU must be serialised by the caller (same stream).
    q: CUDA float64 tensor, neq*cells elements; dt_out: CUDA float64 tensor of one element that receives dt;
    nonphysical_out: CUDA int32 tensor of one element (or None) that receives 1 if a cell was non-physical, else 0.
    Asynchronous on `stream` (default: torch's current stream); nothing is read back to the host here.  The first
    call on a device looks up the array's device address: make it outside of stream capture."""
    import torch
    nf = len(gamma)
    p = MfcParams()
    p.ndim, p.nfluids, p.device = int(ndim), nf, int(device)
    g_arr, pi_arr = (C.c_double * nf)(*gamma), (C.c_double * nf)(*pi_inf)
    for d in range(3):
        p.n[d] = n[d]
        p.dx[d] = dx[d]
    p.gamma = C.cast(g_arr, C.POINTER(C.c_double))
    p.pi_inf = C.cast(pi_arr, C.POINTER(C.c_double))
    p.stream = torch.cuda.current_stream(device).cuda_stream if stream is None else stream
    count = (2 * nf + int(ndim) + 1) * int(n[0]) * int(n[1]) * int(n[2])
    flag_ptr = None
    if nonphysical_out is not None:
        if not (nonphysical_out.is_cuda and nonphysical_out.dtype == torch.int32 and nonphysical_out.numel() == 1):
            raise TypeError("nonphysical_out: expected a CUDA int32 tensor of one element")
        flag_ptr = nonphysical_out.data_ptr()
    _ck(lib().mfc_cfl_dt_static(C.byref(p), _dev_ptr(q, count), float(cfl), _dev_ptr(dt_out, 1), flag_ptr))


def _ck(status):
    if status != MFC_OK:
        raise MfcError(status, lib().mfc_last_error().decode())


def _dev_ptr(t, count):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    if t.numel() != count:
        raise ValueError(f"expected {count} elements, got {t.numel()}")
    return t.data_ptr()


def _host_ptr(t, count):
    import numpy as np
    import torch
    if isinstance(t, torch.Tensor):
        if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
            raise TypeError("expected a contiguous float64 CPU tensor")
        if t.numel() != count:
            raise ValueError(f"expected {count} elements, got {t.numel()}")
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        if t.dtype != np.float64 or not t.flags["C_CONTIGUOUS"]:
            raise TypeError("expected a C-contiguous float64 array")
        if t.size != count:
            raise ValueError(f"expected {count} elements, got {t.size}")
        return t.ctypes.data
    raise TypeError("expected a numpy array or CPU tensor")


class Grid:
    """Handle of one grid (mfc_init_grid ... mfc_free_grid); methods carry the C names without the prefix."""

    def __init__(self, ndim, n, dx, gamma, pi_inf, bc_lo, bc_hi, weno_eps=1e-16, alpha_floor=1e-6, clamp=True,
                 device=0, stream=None, weno="js", model="allaire", eta=0.0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_07953_b200 needs a CUDA device (there is no CPU fallback)")
        self._h = C.c_void_p()
        p = MfcParams()
        p.ndim = ndim
        nf = len(gamma)
        self._gamma = (C.c_double * nf)(*gamma)
        self._pi = (C.c_double * nf)(*pi_inf)
        for d in range(3):
            p.n[d] = n[d]
            p.dx[d] = dx[d]
            p.bc_lo[d] = bc_lo[d]
            p.bc_hi[d] = bc_hi[d]
        p.nfluids = nf
        p.gamma = C.cast(self._gamma, C.POINTER(C.c_double))
        p.pi_inf = C.cast(self._pi, C.POINTER(C.c_double))
        p.weno_eps, p.alpha_floor, p.clamp = weno_eps, alpha_floor, int(bool(clamp))
        p.weno = WENO_BY_NAME[weno] if isinstance(weno, str) else int(weno)
        p.model = MODEL_BY_NAME[model] if isinstance(model, str) else int(model)
        p.eta = float(eta)
        p.device = device
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        p.stream = stream
        _ck(lib().mfc_init_grid(C.byref(p), C.byref(self._h)))
        self.neq = lib().mfc_num_eqns(self._h)
        self.cells = lib().mfc_num_cells(self._h)
        self.count = self.neq * self.cells
        self.shape = (self.neq, n[2], n[1], n[0])
        self.device = device

    @classmethod
    def from_case(cls, case, device=0, stream=None):
        """case: an mfc_workloads.Case-like object (ndim, n, dx, gamma, pi_inf, bc_lo, bc_hi, weno_eps, alpha_floor, clamp)."""
        return cls(case.ndim, case.n, case.dx, case.gamma, case.pi_inf, case.bc_lo, case.bc_hi, case.weno_eps,
                   case.alpha_floor, case.clamp, device, stream, getattr(case, "weno", "js"), getattr(case, "model", "allaire"), getattr(case, "eta", 0.0))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().mfc_free_grid(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:  # interpreter shutdown: module globals may already be gone
            pass

    def prim_from_cons(self, q, w):
        _ck(lib().mfc_prim_from_cons(self._h, _dev_ptr(q, self.count), _dev_ptr(w, self.count)))

    def rhs(self, q, rhs):
        _ck(lib().mfc_rhs(self._h, _dev_ptr(q, self.count), _dev_ptr(rhs, self.count)))

    def rhs_dirs(self, q, rhs, dir_mask):
        _ck(lib().mfc_rhs_dirs(self._h, _dev_ptr(q, self.count), _dev_ptr(rhs, self.count), dir_mask))

    def rk3_step(self, q, dt):
        _ck(lib().mfc_rk3_step(self._h, _dev_ptr(q, self.count), float(dt)))

    def rk3_steps(self, q, dt, nsteps):
        _ck(lib().mfc_rk3_steps(self._h, _dev_ptr(q, self.count), float(dt), int(nsteps)))

    def cfl_dt(self, q, cfl):
        dt = C.c_double()
        _ck(lib().mfc_cfl_dt(self._h, _dev_ptr(q, self.count), float(cfl), C.byref(dt)))
        return dt.value

    def check(self):
        _ck(lib().mfc_check(self._h))

    def rhs_host(self, q_host, rhs_host):
        _ck(lib().mfc_rhs_host(self._h, _host_ptr(q_host, self.count), _host_ptr(rhs_host, self.count)))

    def rk3_steps_host(self, q_host, dt, nsteps):
        _ck(lib().mfc_rk3_steps_host(self._h, _host_ptr(q_host, self.count), float(dt), int(nsteps)))

    def advance(self, q, cfl, nsteps):
        t = C.c_double()
        _ck(lib().mfc_advance(self._h, _dev_ptr(q, self.count), float(cfl), int(nsteps), C.byref(t)))
        return t.value

    def advance_host(self, q_host, cfl, nsteps):
        t = C.c_double()
        _ck(lib().mfc_advance_host(self._h, _host_ptr(q_host, self.count), float(cfl), int(nsteps), C.byref(t)))
        return t.value

    def set_profiling(self, on):
        _ck(lib().mfc_set_profiling(self._h, int(bool(on))))

    def get_profile(self):
        """{kernel class name: (total device ms, launches)} since set_profiling(True)"""
        out = {}
        for i, name in enumerate(KERNEL_CLASSES):
            ms, n = C.c_double(), C.c_longlong()
            _ck(lib().mfc_get_profile(self._h, i, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out

    def weno5_values(self, stencils, left, right):
        n = left.numel()
        _ck(lib().mfc_weno5_values(self._h, _dev_ptr(stencils, 5 * n), n, _dev_ptr(left, n), _dev_ptr(right, n)))

    def hllc_faces(self, direction, wL, wR, F, uf):
        n = uf.numel()
        _ck(lib().mfc_hllc_faces(self._h, int(direction), _dev_ptr(wL, n * self.neq), _dev_ptr(wR, n * self.neq), n,
                                 _dev_ptr(F, n * self.neq), _dev_ptr(uf, n)))

    def sqrt_ratio_values(self, a, b, out, seed_out=None):
        n = out.numel()
        _ck(lib().mfc_sqrt_ratio_values(self._h, _dev_ptr(a, n), _dev_ptr(b, n), n, _dev_ptr(out, n),
                                        _dev_ptr(seed_out, n) if seed_out is not None else None))

    def set_halo(self, halo_lo, halo_hi):
        """halo_lo / halo_hi: CUDA float64 tensors of neq*3*plane elements ([v][layer][plane]) or None; kept alive here"""
        self._halo = (halo_lo, halo_hi)
        lo = _dev_ptr(halo_lo, halo_lo.numel()) if halo_lo is not None else None
        hi = _dev_ptr(halo_hi, halo_hi.numel()) if halo_hi is not None else None
        _ck(lib().mfc_set_halo(self._h, lo, hi))

    def pack_halo(self, q, stage, send_lo, send_hi):
        lo = _dev_ptr(send_lo, send_lo.numel()) if send_lo is not None else None
        hi = _dev_ptr(send_hi, send_hi.numel()) if send_hi is not None else None
        _ck(lib().mfc_pack_halo(self._h, _dev_ptr(q, self.count), int(stage), lo, hi))

    def rk3_stage(self, q, dt, stage, parts=3):
        """parts: 1 = the sweeps before the last direction, 2 = the last sweep with the RK stage, 3 = both"""
        _ck(lib().mfc_rk3_stage_parts(self._h, _dev_ptr(q, self.count), float(dt), int(stage), int(parts)))

    def stage_input_ptr(self, q, stage):
        """device address of the array stage `stage` sweeps (stage 1: q itself)"""
        out = C.c_void_p()
        _ck(lib().mfc_stage_input(self._h, _dev_ptr(q, self.count), int(stage), C.byref(out)))
        return out.value

    def launch_count(self):
        return lib().mfc_launch_count(self._h)

    def set_step_graph(self, on):
        """False: advance() launches every kernel of every step itself also on small grids (default: a CUDA graph of two steps)"""
        _ck(lib().mfc_set_step_graph(self._h, int(bool(on))))

    def set_segments(self, seg_x=0, seg_y=0, seg_z=0):
        _ck(lib().mfc_set_segments(self._h, seg_x, seg_y, seg_z))
