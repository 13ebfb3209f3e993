"""ctypes front of the fp64 CPU oracle (oracle/marchenko_oracle.cpp) — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
Argument marshalling only; every number comes from the C++ file.  It imports nothing from the CUDA
package (paper_2106_04649_b200.binding / csrc) and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "marchenko_oracle.cpp"
# ORACLE_SANITIZE=1 builds and loads an AddressSanitizer + UBSan copy instead (run the pins under
# LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0; profiles/sanitizers_r2.md)
_SAN = os.environ.get("ORACLE_SANITIZE", "0") not in ("", "0")
_LIB = _HERE / ("libmarchenko_oracle_san.so" if _SAN else "libmarchenko_oracle.so")
_lib = None


def build(force: bool = False) -> Path:
    """g++ -O2 -fopenmp; no fast-math, no FFT library, nothing but libstdc++/libgomp."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SAN \
            else ["-O3", "-mavx2"]
        cmd = ["g++", *opt, "-fopenmp", "-std=c++17", "-shared", "-fPIC",
               "-ffp-contract=off", str(_SRC), "-o", str(_LIB)]
        subprocess.check_call(cmd)
    return _LIB


_F32 = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_F64 = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_I32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.orc_num_threads.restype = C.c_int
        L.orc_band.restype = C.c_int
        L.orc_band.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.orc_weights.argtypes = [C.c_int, C.c_double, _F64]
        L.orc_band_kernel.argtypes = [C.c_int, C.c_int, C.c_int, _F64]
        L.orc_apply_band.argtypes = [C.c_int, _F64, _F64, _F64]
        L.orc_window.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int, _F32, _I32]
        L.orc_theta.restype = C.c_int
        L.orc_theta.argtypes = [C.c_int, C.c_int, C.c_int]
        L.orc_synthesis.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _F64, _F32, C.c_int, _F64, C.c_int,
                                    C.c_int, _F64]
        L.orc_marchenko.restype = C.c_int
        L.orc_marchenko.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int,
                                    _F32, C.c_int, _F32, _F32, C.c_int] + [C.c_void_p] * 8
        L.orc_marchenko_geom.restype = C.c_int
        L.orc_marchenko_geom.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _F64, _I32, C.c_double, C.c_double, C.c_int,
                                         _F32, C.c_int, _F32, _F32, C.c_int] + [C.c_void_p] * 8
        L.orc_init_subset.argtypes = [C.c_int, C.c_int, _F32] + [C.c_void_p] * 5
        L.orc_step_subset.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _F64, _F32, C.c_int, _F64, _I32, C.c_int,
                                      C.c_int, C.c_int, _F64] + [C.c_void_p] * 5
        L.orc_finals_subset.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _F64, _F32, C.c_int, _F64, _F64, _F64,
                                        _F64, _F64, _F64, C.c_int, C.c_int] + [C.c_void_p] * 3
        L.orc_image.argtypes = [C.c_int, C.c_int, C.c_double, _F64, C.c_int, _F64, _F64, _F64]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def band(nt: int, dt: float, fmin: float, fmax: float):
    """(klo, khi, nb) of the band B (reading G8)."""
    lo, hi = C.c_int(), C.c_int()
    nb = lib().orc_band(nt, dt, fmin, fmax, C.byref(lo), C.byref(hi))
    return lo.value, hi.value, nb


def weights(n: int, dx: float) -> np.ndarray:
    w = np.empty(n, dtype=np.float64)
    lib().orc_weights(n, dx, w)
    return w


def band_kernel(nt: int, klo: int, khi: int) -> np.ndarray:
    b = np.empty(nt, dtype=np.float64)
    lib().orc_band_kernel(nt, klo, khi, b)
    return b


def apply_band(b: np.ndarray, x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    lib().orc_apply_band(len(x), np.ascontiguousarray(b, dtype=np.float64), x, y)
    return y


def window(td: np.ndarray, nt: int, dt: float, eps: int) -> np.ndarray:
    """h[...] int32 window half-widths from fp32 traveltimes (O3)."""
    td = np.ascontiguousarray(td, dtype=np.float32)
    h = np.empty(td.shape, dtype=np.int32)
    lib().orc_window(td.size, nt, dt, eps, td.reshape(-1), h.reshape(-1))
    return h


def theta(nt: int, h: int) -> np.ndarray:
    L = lib()
    return np.array([L.orc_theta(nt, int(h), j) for j in range(nt)], dtype=np.float64)


def synthesis(R: np.ndarray, N: np.ndarray, dt: float, w: np.ndarray, klo: int, khi: int) -> np.ndarray:
    """S[f][r][:] = P_B{dt sum_s w[s] R[s][r] (*) N[f][s]} (O5a).  R: [nshot][nrout][nt] fp32, N: [nfoc][nshot][nt]."""
    R = np.ascontiguousarray(R, dtype=np.float32)
    N = np.ascontiguousarray(N, dtype=np.float64)
    nshot, nrout, nt = R.shape
    nfoc = N.shape[0]
    assert N.shape == (nfoc, nshot, nt)
    S = np.empty((nfoc, nrout, nt), dtype=np.float64)
    lib().orc_synthesis(nshot, nrout, nt, dt, np.ascontiguousarray(w, dtype=np.float64), R, nfoc, N, klo, khi, S)
    return S


def marchenko(R: np.ndarray, Gd: np.ndarray, td: np.ndarray, dt: float, dx: float, fmin: float, fmax: float,
              niter: int, eps: int = 8, keep_iters: bool = True, want=("f1plus", "f1min", "f2", "pmin", "G", "Gplus",
                                                                        "Gminus")):
    """The whole scheme (O4..O6).  Returns a dict of float64 arrays [nfoc][n][nt] (+ 'N_iters' [niter][nfoc][n][nt])."""
    R = np.ascontiguousarray(R, dtype=np.float32)
    Gd = np.ascontiguousarray(Gd, dtype=np.float32)
    td = np.ascontiguousarray(td, dtype=np.float32)
    n, n2, nt = R.shape
    assert n == n2
    nfoc = Gd.shape[0]
    assert Gd.shape == (nfoc, n, nt) and td.shape == (nfoc, n)
    out = {}
    names = ["f1plus", "f1min", "f2", "pmin", "G", "Gplus", "Gminus"]
    ptrs = []
    if keep_iters:
        out["N_iters"] = np.empty((niter, nfoc, n, nt), dtype=np.float64)
        ptrs.append(out["N_iters"].ctypes.data_as(C.c_void_p))
    else:
        ptrs.append(None)
    for nm in names:
        if nm in want:
            out[nm] = np.empty((nfoc, n, nt), dtype=np.float64)
            ptrs.append(out[nm].ctypes.data_as(C.c_void_p))
        else:
            ptrs.append(None)
    rc = lib().orc_marchenko(n, nt, dt, dx, fmin, fmax, eps, R.reshape(-1), nfoc, Gd.reshape(-1), td.reshape(-1),
                             niter, *ptrs)
    assert rc == 0
    return out


def marchenko_geom(R, Gd, td, dt, w, rec_of_shot, fmin, fmax, niter, eps=8, want=("f1plus", "f1min", "f2", "pmin", "G", "Gplus", "Gminus")):
    """The scheme for sources and receivers that are not co-located one to one (orc_marchenko_geom; NEXT-4).
    R: [nshot][nrec][nt]; Gd [nfoc][nrec][nt], td [nfoc][nrec] on the receiver grid; w [nshot] quadrature weights of the
    shot grid; rec_of_shot [nshot] int (receiver co-located with each shot, or -1).  Outputs on the receiver grid."""
    R = np.ascontiguousarray(R, dtype=np.float32)
    Gd = np.ascontiguousarray(Gd, dtype=np.float32)
    td = np.ascontiguousarray(td, dtype=np.float32)
    nshot, nrec, nt = R.shape
    nfoc = Gd.shape[0]
    assert Gd.shape == (nfoc, nrec, nt) and td.shape == (nfoc, nrec)
    w = np.ascontiguousarray(w, dtype=np.float64)
    ros = np.ascontiguousarray(rec_of_shot, dtype=np.int32)
    assert w.shape == (nshot,) and ros.shape == (nshot,)
    out = {"N_iters": np.empty((niter, nfoc, nrec, nt), dtype=np.float64)}
    ptrs = [out["N_iters"].ctypes.data_as(C.c_void_p)]
    for nm in ("f1plus", "f1min", "f2", "pmin", "G", "Gplus", "Gminus"):
        if nm in want:
            out[nm] = np.empty((nfoc, nrec, nt), dtype=np.float64)
            ptrs.append(out[nm].ctypes.data_as(C.c_void_p))
        else:
            ptrs.append(None)
    rc = lib().orc_marchenko_geom(nshot, nrec, nt, dt, w, ros, fmin, fmax, eps, R.reshape(-1), nfoc, Gd.reshape(-1), td.reshape(-1),
                                  niter, *ptrs)
    assert rc == 0
    return out


def _opt(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class SubsetChain:
    """The oracle restricted to a subset of output receivers (SURVEY.md §8(c) "single step"): every step takes the
    previous iterate at EVERY source position (supplied by the caller) and advances the subset accumulators with
    orc_step_subset; finals() is orc_finals_subset.  R_sub: [nshot][nrout][nt] fp32; td_sub: [nfoc][nrout] fp32."""

    def __init__(self, R_sub, td_sub, Gd_sub, dt, dx, fmin, fmax, eps=8):
        self.R = np.ascontiguousarray(R_sub, dtype=np.float32)
        self.nshot, self.nrout, self.nt = self.R.shape
        self.dt = float(dt)
        self.w = weights(self.nshot, dx)
        self.klo, self.khi, self.nb = band(self.nt, dt, fmin, fmax)
        self.h = window(td_sub, self.nt, dt, eps)
        self.nfoc = self.h.shape[0]
        assert self.h.shape == (self.nfoc, self.nrout)
        Gd_sub = np.ascontiguousarray(Gd_sub, dtype=np.float32)
        assert Gd_sub.shape == (self.nfoc, self.nrout, self.nt)
        # O4 on the subset (orc_init_subset): f1plus = f2 = T G_d; f1min = pmin = 0   [PAPER.md:19, 67, 74-75]
        shape = (self.nfoc, self.nrout, self.nt)
        self.f1plus, self.f2, self.f1min, self.pmin = (np.empty(shape, dtype=np.float64) for _ in range(4))
        lib().orc_init_subset(self.nfoc * self.nrout, self.nt, Gd_sub.reshape(-1), None, _opt(self.f1plus), _opt(self.f2),
                              _opt(self.f1min), _opt(self.pmin))
        self.it = 0

    def step(self, N_prev_all):
        """N_prev_all: [nfoc][nshot][nt]; returns the new iterate on the subset, float64 [nfoc][nrout][nt]."""
        N_prev_all = np.ascontiguousarray(N_prev_all, dtype=np.float64)
        assert N_prev_all.shape == (self.nfoc, self.nshot, self.nt)
        Nn = np.empty((self.nfoc, self.nrout, self.nt), dtype=np.float64)
        lib().orc_step_subset(self.nshot, self.nrout, self.nt, self.dt, self.w, self.R.reshape(-1), self.nfoc,
                              N_prev_all.reshape(-1), self.h.reshape(-1), self.klo, self.khi, self.it, Nn.reshape(-1),
                              None, _opt(self.pmin), _opt(self.f2), _opt(self.f1plus), _opt(self.f1min))
        self.it += 1
        return Nn

    def finals(self, f1plus_all, f1min_all, want=("G", "Gplus", "Gminus")):
        f1plus_all = np.ascontiguousarray(f1plus_all, dtype=np.float64)
        f1min_all = np.ascontiguousarray(f1min_all, dtype=np.float64)
        out = {nm: np.empty_like(self.f2) for nm in want}
        lib().orc_finals_subset(self.nshot, self.nrout, self.nt, self.dt, self.w, self.R.reshape(-1), self.nfoc,
                                f1plus_all.reshape(-1), f1min_all.reshape(-1), self.f1plus.reshape(-1),
                                self.f1min.reshape(-1), self.f2.reshape(-1), self.pmin.reshape(-1), self.klo, self.khi,
                                _opt(out.get("G")), _opt(out.get("Gplus")), _opt(out.get("Gminus")))
        return out


def init_field(Gd):
    """N_{-1} = T G_d as float64 (orc_init_subset; O4)."""
    Gd = np.ascontiguousarray(Gd, dtype=np.float32)
    out = np.empty(Gd.shape, dtype=np.float64)
    lib().orc_init_subset(int(np.prod(Gd.shape[:-1])), Gd.shape[-1], Gd.reshape(-1), _opt(out), None, None, None, None)
    return out


def image(Gminus, f1plus, dt, dx):
    """image[f] = dt sum_r w[r] sum_j G^-[f][r][(nt-j)%nt] f1plus[f][r][j]  (NEXT-1)."""
    Gminus = np.ascontiguousarray(Gminus, dtype=np.float64)
    f1plus = np.ascontiguousarray(f1plus, dtype=np.float64)
    nfoc, n, nt = Gminus.shape
    out = np.empty(nfoc, dtype=np.float64)
    lib().orc_image(n, nt, dt, weights(n, dx), nfoc, Gminus.reshape(-1), f1plus.reshape(-1), out)
    return out
