"""ctypes binding of libsfft.so (include/sfft.h) -- argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device
memory and streams, nothing else.  There is no CPU fallback: a missing library or a
missing CUDA device raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import torch

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libsfft.so"

OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_CUDA, ERR_STATE, ERR_NOT_SPD = 0, -1, -2, -3, -4, -5
STAGES = ("a1_template", "a1_science", "a2_omega", "a2_theta", "a3_gather", "a4_factor",
          "a4_solve", "a5_subtract")
_STATUS = {0: "OK", -1: "INVALID_ARG", -2: "ALLOC", -3: "CUDA", -4: "STATE", -5: "NOT_SPD"}

# every symbol include/sfft.h declares (tests check the library exports all of them)
SYMBOLS = (
    "sfft_plan_create", "sfft_plan_create_ex", "sfft_plan_set_stream", "sfft_plan_destroy", "sfft_num_unknowns",
    "sfft_workspace_bytes", "sfft_build_system", "sfft_solve", "sfft_solve_constant_ratio", "sfft_set_constant_ratio", "sfft_subtract", "sfft_subtract_with",
    "sfft_set_template", "sfft_subtract_batch", "sfft_convolve_stamp", "sfft_resample_affine", "sfft_resample_affine_mask", "sfft_local_kernel",
    "sfft_decorrelation_stamp", "sfft_difference_host", "sfft_difference_host_batch", "sfft_sync_status",
    "sfft_get_system", "sfft_enable_timings", "sfft_get_timings", "sfft_kernel_timing_count",
    "sfft_kernel_timing_get", "sfft_launch_count",
    "sfft_last_error", "sfft_version", "sfft_debug_read", "sfft_probe_fp64",
    "sfft_solve_static", "sfft_solve_static_last_error",
)
SOLVE_STATIC_MAX_N = 1024  # include/sfft.h: SFFT_SOLVE_STATIC_MAX_N


class SfftError(RuntimeError):
    def __init__(self, code, where, detail=""):
        super().__init__(f"{where}: SFFT_ERR_{_STATUS.get(code, code)} {detail}".strip())
        self.code = code


_lib = None


def load_library():
    """dlopen libsfft.so (built by paper_2509_18544_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise FileNotFoundError(
            f"{LIB_PATH} not found: run `python -m paper_2509_18544_b200.build` (no CPU fallback exists)")
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, ci, dp = ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p
    lib.sfft_plan_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci]
    lib.sfft_plan_create_ex.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, ci, ctypes.c_uint]
    lib.sfft_plan_set_stream.argtypes = [vp, vp]
    lib.sfft_plan_destroy.argtypes = [vp]
    lib.sfft_num_unknowns.argtypes = [vp]
    lib.sfft_workspace_bytes.argtypes = [vp]
    lib.sfft_workspace_bytes.restype = ctypes.c_size_t
    lib.sfft_build_system.argtypes = [vp, dp, dp, dp]
    lib.sfft_solve.argtypes = [vp]
    lib.sfft_solve_constant_ratio.argtypes = [vp]
    lib.sfft_set_constant_ratio.argtypes = [vp, ci]
    lib.sfft_subtract.argtypes = [vp, dp, dp]
    lib.sfft_subtract_with.argtypes = [vp, dp, dp, dp]
    lib.sfft_convolve_stamp.argtypes = [vp, dp, dp, dp]
    cd = ctypes.c_double
    lib.sfft_resample_affine.argtypes = [vp, dp, ctypes.POINTER(cd), ci, cd, dp]
    lib.sfft_resample_affine_mask.argtypes = [vp, dp, ctypes.POINTER(cd), ci, dp]
    lib.sfft_local_kernel.argtypes = [vp, dp, cd, cd, dp]
    lib.sfft_decorrelation_stamp.argtypes = [vp, dp, ci, dp, dp, ci, cd, cd, ci, dp]
    lib.sfft_set_template.argtypes = [vp, dp, dp]
    lib.sfft_subtract_batch.argtypes = [vp, ctypes.POINTER(vp), ci, ctypes.POINTER(vp), dp]
    lib.sfft_difference_host.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.sfft_difference_host_batch.argtypes = [vp, dp, dp, ctypes.POINTER(vp), ci, ctypes.POINTER(vp), dp]
    lib.sfft_sync_status.argtypes = [vp]
    lib.sfft_get_system.argtypes = [vp, dp, dp]
    lib.sfft_enable_timings.argtypes = [vp, ci]
    lib.sfft_get_timings.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ci]
    lib.sfft_kernel_timing_count.argtypes = [vp]
    lib.sfft_kernel_timing_get.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_char_p), ctypes.POINTER(ctypes.c_float)]
    lib.sfft_launch_count.argtypes = [vp]
    lib.sfft_launch_count.restype = ctypes.c_longlong
    lib.sfft_last_error.argtypes = [vp]
    lib.sfft_last_error.restype = ctypes.c_char_p
    lib.sfft_version.restype = ctypes.c_char_p
    lib.sfft_debug_read.argtypes = [vp, ci, ci, vp, ctypes.c_size_t]
    lib.sfft_probe_fp64.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_double)]
    lib.sfft_solve_static.argtypes = [dp, dp, dp, ci, vp]
    lib.sfft_solve_static_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def version() -> str:
    return load_library().sfft_version().decode()


def probe_fp64(kind: int, iters: int = 4096) -> float:
    """Measured FP64 rate in TFLOP/s: kind 0 = DFMA, 1 = DMMA m8n8k4."""
    out = ctypes.c_double()
    rc = load_library().sfft_probe_fp64(kind, iters, ctypes.byref(out))
    if rc:
        raise SfftError(rc, "sfft_probe_fp64")
    return out.value


def solve_static(G, h, c, stream=None):
    """sfft_solve_static: G c = h with the library's static scratch array (no allocation); G (n, n), h (n,), c (n,)
    are the caller's CUDA float64 tensors, c is written and returned.  Blocks until done."""
    lib = load_library()
    n = int(h.shape[0])
    _dev_f64(G, (n, n), "G"); _dev_f64(h, (n,), "h"); _dev_f64(c, (n,), "c")
    st = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = lib.sfft_solve_static(G.data_ptr(), h.data_ptr(), c.data_ptr(), n, st)
    if rc:
        raise SfftError(rc, "sfft_solve_static", lib.sfft_solve_static_last_error().decode())
    return c


def _dev_f64(t, shape, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous CUDA float64 tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return t.data_ptr()


def _dev_mask(m, shape):
    if m is None:
        return None
    if not (isinstance(m, torch.Tensor) and m.is_cuda and m.dtype == torch.uint8 and m.is_contiguous()):
        raise TypeError("mask: need a contiguous CUDA uint8 tensor")
    if tuple(m.shape) != tuple(shape):
        raise ValueError("mask: shape mismatch")
    return m.data_ptr()


class SfftPlan:
    """sfft_plan_create(nx, ny, L, DK, DB) and the calls on it; same names as the C ABI."""

    FP32_SPECTRA = 1   # SFFT_PLAN_FP32_SPECTRA: the reduced-memory mode (spectra stored as complex64)

    def __init__(self, nx, ny, L, DK, DB, stream=None, flags=0):
        if not torch.cuda.is_available():
            raise RuntimeError("libsfft needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        rc = self._lib.sfft_plan_create_ex(ctypes.byref(self._h), nx, ny, L, DK, DB, int(flags))
        if rc:
            self._h = None
            raise SfftError(rc, "sfft_plan_create_ex" if flags else "sfft_plan_create")
        self.flags = int(flags)
        self.nx, self.ny, self.L, self.DK, self.DB = nx, ny, L, DK, DB
        self.shape = (ny, nx)
        self.n = self._lib.sfft_num_unknowns(self._h)
        self._keep = []
        self.set_stream(stream if stream is not None else torch.cuda.current_stream())

    # -- life cycle ---------------------------------------------------------------------
    def set_stream(self, stream):
        self._stream = stream
        self._ck(self._lib.sfft_plan_set_stream(self._h, ctypes.c_void_p(stream.cuda_stream)), "sfft_plan_set_stream")

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.sfft_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _ck(self, rc, where):
        if rc:
            raise SfftError(rc, where, self._lib.sfft_last_error(self._h).decode())

    @property
    def workspace_bytes(self):
        return self._lib.sfft_workspace_bytes(self._h)

    @property
    def launch_count(self):
        return self._lib.sfft_launch_count(self._h)

    # -- single pair ----------------------------------------------------------------------
    def build_system(self, S, R, mask=None):
        sp, rp, mp = _dev_f64(S, self.shape, "S"), _dev_f64(R, self.shape, "R"), _dev_mask(mask, self.shape)
        self._keep = [S, R, mask]  # the plan keeps the pointers until subtract
        self._ck(self._lib.sfft_build_system(self._h, sp, rp, mp), "sfft_build_system")

    def solve(self):
        self._ck(self._lib.sfft_solve(self._h), "sfft_solve")

    def set_constant_ratio(self, on=True):
        """Plan mode: every solve (single, batched, host path) under the constant-ratio constraint (f4)."""
        self._ck(self._lib.sfft_set_constant_ratio(self._h, 1 if on else 0), "sfft_set_constant_ratio")

    def solve_constant_ratio(self):
        """sfft_solve under the constant-photometric-ratio constraint (f4); see sfft_solve_constant_ratio."""
        self._ck(self._lib.sfft_solve_constant_ratio(self._h), "sfft_solve_constant_ratio")

    def subtract(self, D=None, coeffs=None):
        if D is None:
            D = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        if coeffs is None:
            coeffs = torch.empty(self.n, dtype=torch.float64, device="cuda")
        self._ck(self._lib.sfft_subtract(self._h, _dev_f64(D, self.shape, "D"), _dev_f64(coeffs, (self.n,), "coeffs")),
                 "sfft_subtract")
        return D, coeffs

    def subtract_with(self, coeffs_in, S=None, D=None):
        if D is None:
            D = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        sp = _dev_f64(S, self.shape, "S") if S is not None else None
        self._ck(self._lib.sfft_subtract_with(self._h, sp, _dev_f64(coeffs_in, (self.n,), "coeffs_in"),
                                              _dev_f64(D, self.shape, "D")), "sfft_subtract_with")
        return D

    # -- f2: cross-convolution with a PSF stamp --------------------------------
    def convolve_stamp(self, img, stamp, out=None):
        """out = img (*) stamp (L x L taps, circular at the native grid); see sfft_convolve_stamp in include/sfft.h."""
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        self._ck(self._lib.sfft_convolve_stamp(self._h, _dev_f64(img, self.shape, "img"),
                                               _dev_f64(stamp, (self.L, self.L), "stamp"),
                                               _dev_f64(out, self.shape, "out")), "sfft_convolve_stamp")
        return out

    def cross_convolve(self, S, R, psf_S, psf_R):
        """Pipeline step 5: (S (*) psf_R, R (*) psf_S)."""
        return self.convolve_stamp(S, psf_R), self.convolve_stamp(R, psf_S)

    # -- f3: alignment onto the science grid ------------------------------------
    def resample_affine(self, img, M, method=3, fill=0.0, out=None):
        """out(x, y) = img interpolated at (M0 x + M1 y + M2, M3 x + M4 y + M5); see sfft_resample_affine."""
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        Mc = (ctypes.c_double * 6)(*[float(m) for m in M])
        self._ck(self._lib.sfft_resample_affine(self._h, _dev_f64(img, self.shape, "img"), Mc, int(method), float(fill),
                                                _dev_f64(out, self.shape, "out")), "sfft_resample_affine")
        return out

    def resample_affine_mask(self, mask, M, fill=0, out=None):
        """Nearest-neighbour resampling of a uint8 mask with the same geometry; see sfft_resample_affine_mask."""
        if out is None:
            out = torch.empty(self.shape, dtype=torch.uint8, device="cuda")
        Mc = (ctypes.c_double * 6)(*[float(m) for m in M])
        self._ck(self._lib.sfft_resample_affine_mask(self._h, _dev_mask(mask, self.shape), Mc, int(fill),
                                                     _dev_mask(out, self.shape)), "sfft_resample_affine_mask")
        return out

    # -- f1: decorrelation kernel ----------------------------------------------
    def local_kernel(self, x, y, coeffs=None, out=None):
        """K(u, v; x, y) as an L x L stamp; coeffs None = the plan's solution.  See sfft_local_kernel."""
        if out is None:
            out = torch.empty((self.L, self.L), dtype=torch.float64, device="cuda")
        cptr = None if coeffs is None else _dev_f64(coeffs, (self.n,), "coeffs")
        self._ck(self._lib.sfft_local_kernel(self._h, cptr, float(x), float(y),
                                             _dev_f64(out, (self.L, self.L), "out")), "sfft_local_kernel")
        return out

    def decorrelation_stamp(self, K, psf_S, psf_R, var_S, var_R, N, out=None):
        """The L x L crop of the decorrelation kernel (L the plan's); see sfft_decorrelation_stamp."""
        Lk, Lp = int(K.shape[0]), int(psf_S.shape[0])
        if out is None:
            out = torch.empty((self.L, self.L), dtype=torch.float64, device="cuda")
        self._ck(self._lib.sfft_decorrelation_stamp(
            self._h, _dev_f64(K, (Lk, Lk), "K"), Lk, _dev_f64(psf_S, (Lp, Lp), "psf_S"),
            _dev_f64(psf_R, (Lp, Lp), "psf_R"), Lp, float(var_S), float(var_R), int(N),
            _dev_f64(out, (self.L, self.L), "out")), "sfft_decorrelation_stamp")
        return out

    # -- batched --------------------------------------------------------------------------
    def set_template(self, R, mask=None):
        rp, mp = _dev_f64(R, self.shape, "R"), _dev_mask(mask, self.shape)
        self._keep = [R, mask]
        self._ck(self._lib.sfft_set_template(self._h, rp, mp), "sfft_set_template")

    def subtract_batch(self, S_list, D_list=None, coeffs=None):
        B = len(S_list)
        if D_list is None:
            D_list = [torch.empty(self.shape, dtype=torch.float64, device="cuda") for _ in range(B)]
        if coeffs is None:
            coeffs = torch.empty((B, self.n), dtype=torch.float64, device="cuda")
        Sp = (ctypes.c_void_p * B)(*[_dev_f64(s, self.shape, "S[b]") for s in S_list])
        Dp = (ctypes.c_void_p * B)(*[_dev_f64(d, self.shape, "D[b]") for d in D_list])
        self._ck(self._lib.sfft_subtract_batch(self._h, Sp, B, Dp, _dev_f64(coeffs, (B, self.n), "coeffs")),
                 "sfft_subtract_batch")
        return D_list, coeffs

    # -- host buffers (end to end) ----------------------------------------------------------
    def difference_host(self, S_host, R_host, mask_host=None, D_host=None, coeffs_host=None):
        """S_host, R_host: CPU float64 tensors (pinned for full copy speed).  Synchronises."""
        for t, nm in ((S_host, "S_host"), (R_host, "R_host")):
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != self.shape:
                raise TypeError(f"{nm}: need a contiguous CPU float64 tensor of shape {self.shape}")
        if D_host is None:
            D_host = torch.empty(self.shape, dtype=torch.float64).pin_memory()
        if coeffs_host is None:
            coeffs_host = torch.empty(self.n, dtype=torch.float64)
        mp = mask_host.data_ptr() if mask_host is not None else None
        self._ck(self._lib.sfft_difference_host(self._h, S_host.data_ptr(), R_host.data_ptr(), mp,
                                                D_host.data_ptr(), coeffs_host.data_ptr()), "sfft_difference_host")
        return D_host, coeffs_host

    def difference_host_batch(self, R_host, S_hosts, mask_host=None, D_hosts=None, coeffs_host=None):
        """One template, B science images, all CPU float64 tensors (pinned for the copies to overlap).  Synchronises."""
        B = len(S_hosts)
        for t, nm in [(R_host, "R_host")] + [(s, "S_hosts[b]") for s in S_hosts]:
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != self.shape:
                raise TypeError(f"{nm}: need a contiguous CPU float64 tensor of shape {self.shape}")
        if D_hosts is None:
            D_hosts = [torch.empty(self.shape, dtype=torch.float64).pin_memory() for _ in range(B)]
        if coeffs_host is None:
            coeffs_host = torch.empty((B, self.n), dtype=torch.float64)
        Sp = (ctypes.c_void_p * B)(*[s.data_ptr() for s in S_hosts])
        Dp = (ctypes.c_void_p * B)(*[d.data_ptr() for d in D_hosts])
        mp = mask_host.data_ptr() if mask_host is not None else None
        self._ck(self._lib.sfft_difference_host_batch(self._h, R_host.data_ptr(), mp, Sp, B, Dp, coeffs_host.data_ptr()),
                 "sfft_difference_host_batch")
        return D_hosts, coeffs_host

    # -- introspection ---------------------------------------------------------------------
    def sync_status(self):
        self._ck(self._lib.sfft_sync_status(self._h), "sfft_sync_status")

    def get_system(self, want_h=True):
        G = torch.empty((self.n, self.n), dtype=torch.float64, device="cuda")
        h = torch.empty(self.n, dtype=torch.float64, device="cuda") if want_h else None
        self._ck(self._lib.sfft_get_system(self._h, G.data_ptr(), h.data_ptr() if want_h else None), "sfft_get_system")
        return G, h

    def enable_timings(self, on=True):
        """on: False/0 = off, True/1 = per stage, 2 = per kernel launch."""
        self._ck(self._lib.sfft_enable_timings(self._h, int(on)), "sfft_enable_timings")

    def kernel_timings(self):
        """[(kernel name, ms), ...] of every launch since enable_timings(2), in launch order."""
        out = []
        name, ms = ctypes.c_char_p(), ctypes.c_float()
        for i in range(self._lib.sfft_kernel_timing_count(self._h)):
            self._ck(self._lib.sfft_kernel_timing_get(self._h, i, ctypes.byref(name), ctypes.byref(ms)),
                     "sfft_kernel_timing_get")
            out.append((name.value.decode(), float(ms.value)))
        return out

    def get_timings(self):
        ms = (ctypes.c_float * len(STAGES))()
        self._ck(self._lib.sfft_get_timings(self._h, ms, len(STAGES)), "sfft_get_timings")
        return dict(zip(STAGES, [float(v) for v in ms]))

    def debug_read(self, which, idx=0):
        import numpy as np
        dims = np.zeros(2)
        self._ck(self._lib.sfft_debug_read(self._h, 7, 0, dims.ctypes.data_as(ctypes.c_void_p), 16), "sfft_debug_read")
        Mx, My = int(dims[0]), int(dims[1])
        if which == 7:
            return Mx, My
        w, L = (self.L - 1) // 2, self.L
        NK, NB = (self.DK + 1) * (self.DK + 2) // 2, (self.DB + 1) * (self.DB + 2) // 2
        shapes = {0: ((My, Mx // 2 + 1), np.complex128), 1: ((My, Mx // 2 + 1), np.complex128),
                  2: ((4 * w + 1, 4 * w + 1), np.float64), 3: ((L, L), np.float64),
                  4: ((NK, NB, L, L), np.float64), 5: ((NB, NB), np.float64), 6: ((NB,), np.float64),
                  8: ((Mx // 2, My), np.complex128)}
        shp, dt = shapes[which]
        out = np.zeros(shp, dtype=dt)
        self._ck(self._lib.sfft_debug_read(self._h, which, idx, out.ctypes.data_as(ctypes.c_void_p), out.nbytes),
                 "sfft_debug_read")
        return out
