"""ctypes binding of oracle/sfft_oracle.c (plain C, FP64, OpenMP) -- test infrastructure.

The shared object is compiled on the machine that runs it (``-march=native``), into a
file whose name carries a hash of the source and of the CPU flags, so a binary built
on one box is never executed on another.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sfft_oracle.c"
_lib = None

OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_NOT_SPD = 0, -1, -2, -5


class OracleError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"oracle {where} failed with status {code}")
        self.code = code


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    h = hashlib.sha1()
    h.update(_SRC.read_bytes())
    h.update(flags.encode())
    return h.hexdigest()[:12]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O3 -march=native -fopenmp).  Building the checker
    is not using it: __graft_entry__.build() calls this too."""
    out = _HERE / f"_sfft_oracle_{_cpu_tag()}.so"
    if out.exists() and not force:
        return out
    tmp = out.with_suffix(f".{os.getpid()}.tmp")
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-std=c11", "-fPIC", "-shared",
           "-o", str(tmp), str(_SRC), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(str(build()))
    dp = ctypes.POINTER(ctypes.c_double)
    u8p = ctypes.POINTER(ctypes.c_uint8)
    ip = ctypes.POINTER(ctypes.c_int)
    ci = ctypes.c_int
    lib.oracle_num_poly.argtypes = [ci]
    lib.oracle_num_unknowns.argtypes = [ci, ci, ci]
    lib.oracle_poly_index.argtypes = [ci, ip, ip]
    lib.oracle_poly_index.restype = None
    lib.oracle_coord.argtypes = [ci, ci]
    lib.oracle_coord.restype = ctypes.c_double
    lib.oracle_weighted_image.argtypes = [dp, u8p, ci, ci, ci, ci, dp]
    lib.oracle_weighted_image.restype = None
    lib.oracle_poly_image.argtypes = [ci, ci, ci, ci, dp]
    lib.oracle_poly_image.restype = None
    lib.oracle_lag_sum.argtypes = [dp, dp, ci, ci, ci, ci]
    lib.oracle_lag_sum.restype = ctypes.c_double
    lib.oracle_build_system.argtypes = [dp, dp, u8p, ci, ci, ci, ci, ci, dp, dp]
    lib.oracle_build_system_dense.argtypes = [dp, dp, u8p, ci, ci, ci, ci, ci, dp, dp]
    lib.oracle_design_matrix.argtypes = [dp, u8p, ci, ci, ci, ci, ci, dp]
    lib.oracle_solve.argtypes = [dp, dp, ci, dp, dp]
    lib.oracle_subtract.argtypes = [dp, dp, ci, ci, ci, ci, ci, dp, dp]
    lib.oracle_subtract_at.argtypes = [dp, dp, ci, ci, ci, ci, ci, dp, ip, ip, ci, dp]
    lib.oracle_system_entry.argtypes = [dp, dp, u8p, ci, ci, ci, ci, ci, ci, ci, dp, dp]
    _lib = lib
    return lib


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _img(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 2:
        raise ValueError("image must be 2-D (ny, nx)")
    return a


def _mask(m, shape):
    if m is None:
        return None, None
    m = np.ascontiguousarray(m, dtype=np.uint8)
    if m.shape != shape:
        raise ValueError("mask shape mismatch")
    return m, m.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


def num_threads() -> int:
    """Threads the OpenMP runtime will use (what bench.py reports as `cores`)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def num_poly(deg: int) -> int:
    return _load().oracle_num_poly(deg)


def num_unknowns(L: int, DK: int, DB: int) -> int:
    return _load().oracle_num_unknowns(L, DK, DB)


def poly_index(t: int):
    i, j = ctypes.c_int(), ctypes.c_int()
    _load().oracle_poly_index(t, ctypes.byref(i), ctypes.byref(j))
    return i.value, j.value


def coord(x: int, n: int) -> float:
    return _load().oracle_coord(x, n)


def weighted_image(img, mask, i, j):
    img = _img(img)
    m, mp = _mask(mask, img.shape)
    out = np.empty_like(img)
    _load().oracle_weighted_image(_d(img), mp, img.shape[1], img.shape[0], i, j, _d(out))
    return out


def poly_image(nx, ny, p, q):
    out = np.empty((ny, nx))
    _load().oracle_poly_image(nx, ny, p, q, _d(out))
    return out


def lag_sum(a, b, du, dv) -> float:
    a, b = _img(a), _img(b)
    assert a.shape == b.shape
    return _load().oracle_lag_sum(_d(a), _d(b), a.shape[1], a.shape[0], du, dv)


def build_system(S, R, mask, L, DK, DB, dense=False):
    S, R = _img(S), _img(R)
    assert S.shape == R.shape
    m, mp = _mask(mask, S.shape)
    n = num_unknowns(L, DK, DB)
    G = np.zeros((n, n))
    h = np.zeros(n)
    fn = _load().oracle_build_system_dense if dense else _load().oracle_build_system
    rc = fn(_d(S), _d(R), mp, S.shape[1], S.shape[0], L, DK, DB, _d(G), _d(h))
    if rc:
        raise OracleError(rc, "build_system")
    return G, h


def build_system_dense(S, R, mask, L, DK, DB):
    return build_system(S, R, mask, L, DK, DB, dense=True)


def design_matrix(R, mask, L, DK, DB):
    R = _img(R)
    m, mp = _mask(mask, R.shape)
    n = num_unknowns(L, DK, DB)
    A = np.zeros((R.size, n))
    rc = _load().oracle_design_matrix(_d(R), mp, R.shape[1], R.shape[0], L, DK, DB, _d(A))
    if rc:
        raise OracleError(rc, "design_matrix")
    return A


def solve(G, h, return_factor=False):
    G = np.ascontiguousarray(G, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float64)
    n = h.shape[0]
    c = np.zeros(n)
    Lf = np.zeros((n, n)) if return_factor else None
    rc = _load().oracle_solve(_d(G), _d(h), n, _d(c), _d(Lf) if return_factor else None)
    if rc:
        raise OracleError(rc, "solve")
    return (c, Lf) if return_factor else c


def subtract(S, R, L, DK, DB, c):
    S, R = _img(S), _img(R)
    c = np.ascontiguousarray(c, dtype=np.float64)
    D = np.empty_like(S)
    rc = _load().oracle_subtract(_d(S), _d(R), S.shape[1], S.shape[0], L, DK, DB, _d(c), _d(D))
    if rc:
        raise OracleError(rc, "subtract")
    return D


def subtract_at(S, R, L, DK, DB, c, xs, ys):
    S, R = _img(S), _img(R)
    c = np.ascontiguousarray(c, dtype=np.float64)
    xs = np.ascontiguousarray(xs, dtype=np.int32)
    ys = np.ascontiguousarray(ys, dtype=np.int32)
    out = np.empty(xs.shape[0])
    ip = ctypes.POINTER(ctypes.c_int)
    rc = _load().oracle_subtract_at(_d(S), _d(R), S.shape[1], S.shape[0], L, DK, DB, _d(c),
                                    xs.ctypes.data_as(ip), ys.ctypes.data_as(ip), xs.shape[0], _d(out))
    if rc:
        raise OracleError(rc, "subtract_at")
    return out


def system_entry(S, R, mask, L, DK, DB, row, col, work=None):
    """G[row, col] (col >= 0) or h[row] (col < 0) by its direct-sum definition."""
    S, R = _img(S), _img(R)
    m, mp = _mask(mask, S.shape)
    if work is None:
        work = np.empty(3 * S.size)
    out = ctypes.c_double()
    rc = _load().oracle_system_entry(_d(S), _d(R), mp, S.shape[1], S.shape[0], L, DK, DB,
                                     int(row), int(col), _d(work), ctypes.byref(out))
    if rc:
        raise OracleError(rc, "system_entry")
    return out.value


# ---------------------------------------------------------------------------------------------------
# f2 -- cross-convolution with a PSF stamp (pipeline step 5: "Cross-convolve the template
# PSF with the science image, and the science PSF with the template").
# The paper gives no formula; the operation is the textbook discrete convolution
#     out(x, y) = sum_{u,v} stamp(u, v) * img((x - u) mod nx, (y - v) mod ny),   |u|, |v| <= w = (P-1)/2,
# with the same boundary as the subtraction (reading C6: circular at the native nx x ny) and the same
# tap layout as the kernel coefficients: stamp[(v + w) * P + (u + w)].  Plain numpy, FP64: one shifted
# copy of the image per tap, summed in the order (v, u) ascending -- no FFT, no blocking.
# ---------------------------------------------------------------------------------------------------
def convolve_stamp(img, stamp):
    img = np.ascontiguousarray(img, dtype=np.float64)
    stamp = np.ascontiguousarray(stamp, dtype=np.float64)
    P = stamp.shape[0]
    if stamp.ndim != 2 or stamp.shape[1] != P or P % 2 != 1:
        raise ValueError("stamp must be P x P with P odd")
    w = (P - 1) // 2
    out = np.zeros_like(img)
    for v in range(-w, w + 1):
        for u in range(-w, w + 1):
            # np.roll(img, (v, u))[y, x] = img[(y - v) mod ny, (x - u) mod nx]
            out += stamp[v + w, u + w] * np.roll(img, (v, u), axis=(0, 1))
    return out


def convolve_stamp_at(img, stamp, xs, ys):
    """The same sum at sampled output pixels (for full-size frames), one pixel at a time."""
    img = np.ascontiguousarray(img, dtype=np.float64)
    stamp = np.ascontiguousarray(stamp, dtype=np.float64)
    ny, nx = img.shape
    P = stamp.shape[0]
    w = (P - 1) // 2
    offs = np.arange(-w, w + 1)
    out = np.empty(len(xs))
    for k, (x, y) in enumerate(zip(xs, ys)):
        rows = (int(y) - offs) % ny          # v ascending
        cols = (int(x) - offs) % nx          # u ascending
        out[k] = float(np.sum(stamp * img[np.ix_(rows, cols)]))
    return out
