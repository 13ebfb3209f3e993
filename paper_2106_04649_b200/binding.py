"""Thin ctypes binding of libmk.so (include/mk.h) — same names, argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of
libmk.  There is no CPU fallback: if the library is missing or no CUDA device is present, loading or
`Marchenko(...)` raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libmk.so"

MK_OK, MK_ERR_INVALID_ARG, MK_ERR_STATE, MK_ERR_OOM, MK_ERR_CUDA = 0, -1, -2, -3, -4
MK_OPT_EPS_SAMPLES, MK_OPT_REGIME, MK_OPT_TIMING, MK_OPT_FFT_PATH, MK_OPT_FUSED_FINALS, MK_OPT_RHAT_FORMAT, MK_OPT_TUNE, MK_OPT_RHAT_LAYOUT = 1, 2, 3, 4, 5, 6, 7, 8
(MK_INFO_NB, MK_INFO_KLO, MK_INFO_KHI, MK_INFO_RHAT_BYTES, MK_INFO_RHAT_BYTES_PADDED, MK_INFO_LD_SHOT,
 MK_INFO_SHOTS_LOADED, MK_INFO_SYN_LAUNCHES, MK_INFO_SYN_MS_TOTAL, MK_INFO_SYN_RESET, MK_INFO_KERNEL_LAUNCHES,
 MK_INFO_REGIME_USED, MK_INFO_DEVICE_BYTES, MK_INFO_RESIDENT_ROWS, MK_INFO_WINDOW_ROWS, MK_INFO_H2D_BYTES, MK_INFO_RHAT_BYTES_STORED, MK_INFO_RHAT_LAYOUT, MK_INFO_SYN_COUNT) = range(1, 20)
REGIME_AUTO, REGIME_GEMV, REGIME_GEMM_FFMA, REGIME_GEMM_TF32X3 = 0, 1, 2, 3

# every symbol include/mk.h declares
SYMBOLS = ("mk_create", "mk_destroy", "mk_set_stream", "mk_set_option", "mk_get_info", "mk_load_R", "mk_load_R_host",
           "mk_run", "mk_run_host", "mk_begin", "mk_step", "mk_finish", "mk_synthesis", "mk_image", "mk_last_error",
           "mk_version", "mk_create_sharded", "mk_operand", "mk_operand_exchanged", "mk_finish_prepare", "mk_finish_complete",
           "mk_operand_reserve", "mk_operand_attach", "mk_step_contract", "mk_step_post", "mk_ipc_export", "mk_ipc_open", "mk_ipc_close",
           "mk_set_geometry", "mk_create_streamed", "mk_sync_create", "mk_sync_flags", "mk_sync_attach", "mk_sync_barrier", "mk_load_R_rows", "mk_image_static")
MK_FIELD_GMINUS, MK_FIELD_GPLUS = 1, 2
MK_IMAGE_STATIC_MAX_PARTIALS = 16384   # doubles in the static scratch array of mk_image_static


class mk_outputs(C.Structure):
    _fields_ = [(nm, C.c_void_p) for nm in ("N_last", "f1plus", "f1min", "G", "Gplus", "Gminus")]


OUTPUT_FIELDS = tuple(nm for nm, _ in mk_outputs._fields_)


class mk_operand_view(C.Structure):
    _fields_ = [("plane", C.c_void_p * 2)] + [(nm, C.c_int) for nm in ("nplanes", "nb", "rows_per_bin", "rows_per_rec", "row_floats",
                                                                         "row0", "nrows")]


class MkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmk error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """Loads libmk.so (raises if it has not been built: `python -m paper_2106_04649_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise FileNotFoundError(f"{LIB_PATH} is missing — build it with `python -m paper_2106_04649_b200.build` "
                                "(there is no CPU fallback)")
    L = C.CDLL(str(LIB_PATH))
    vp, ci, cd = C.c_void_p, C.c_int, C.c_double
    L.mk_create.argtypes = [C.POINTER(vp), ci, ci, ci, cd, cd, cd, cd]
    L.mk_destroy.argtypes = [vp]
    L.mk_set_stream.argtypes = [vp, vp]
    L.mk_set_option.argtypes = [vp, ci, cd]
    L.mk_get_info.argtypes = [vp, ci, C.POINTER(cd)]
    L.mk_set_geometry.argtypes = [vp, vp, vp]
    L.mk_load_R.argtypes = [vp, vp, ci, ci]
    L.mk_load_R_host.argtypes = [vp, vp, ci, ci]
    L.mk_load_R_rows.argtypes = [vp, vp, ci, ci]
    L.mk_run.argtypes = [vp, vp, vp, ci, ci, C.POINTER(mk_outputs)]
    L.mk_run_host.argtypes = [vp, vp, vp, ci, ci, C.POINTER(mk_outputs)]
    L.mk_begin.argtypes = [vp, vp, vp, ci]
    L.mk_step.argtypes = [vp, vp]
    L.mk_step_contract.argtypes = [vp]
    L.mk_step_post.argtypes = [vp, vp]
    L.mk_finish.argtypes = [vp, C.POINTER(mk_outputs)]
    L.mk_synthesis.argtypes = [vp, vp, vp, ci]
    L.mk_image.argtypes = [vp, vp, vp]
    L.mk_image_static.argtypes = [vp, vp, vp, vp, ci]
    L.mk_create_sharded.argtypes = [C.POINTER(vp), ci, ci, ci, cd, cd, cd, cd, ci, ci]
    L.mk_create_streamed.argtypes = [C.POINTER(vp), ci, ci, ci, cd, cd, cd, cd, ci, ci]
    L.mk_operand.argtypes = [vp, ci, C.POINTER(mk_operand_view)]
    L.mk_operand_exchanged.argtypes = [vp, ci]
    L.mk_finish_prepare.argtypes = [vp, ci]
    L.mk_operand_reserve.argtypes = [vp, ci]
    L.mk_operand_attach.argtypes = [vp, ci, ci, C.POINTER(mk_operand_view)]
    L.mk_ipc_export.argtypes = [vp, C.c_char_p]
    L.mk_ipc_open.argtypes = [C.c_char_p, C.POINTER(vp)]
    L.mk_ipc_close.argtypes = [vp]
    L.mk_sync_create.argtypes = [vp, ci, ci]
    L.mk_sync_flags.argtypes = [vp, C.POINTER(vp)]
    L.mk_sync_attach.argtypes = [vp, C.POINTER(vp)]
    L.mk_sync_barrier.argtypes = [vp]
    L.mk_finish_complete.argtypes = [vp, ci, vp]
    L.mk_last_error.argtypes = [vp]
    L.mk_last_error.restype = C.c_char_p
    L.mk_version.restype = C.c_char_p
    for nm in SYMBOLS:
        if nm not in ("mk_last_error", "mk_version"):
            getattr(L, nm).restype = ci
    _lib = L
    return L


def _dev_ptr(t, dtype=None, numel=None):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"expected {numel} elements, got {t.numel()}")
    return C.c_void_p(t.data_ptr())


def _host_ptr(a, numel=None):
    """numpy array or CPU torch tensor (float32, contiguous) -> pointer."""
    import numpy as np
    import torch
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or not a.is_contiguous() or a.dtype != torch.float32:
            raise TypeError("expected a contiguous float32 CPU tensor")
        n, p = a.numel(), a.data_ptr()
    else:
        if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous):
            raise TypeError("expected a C-contiguous float32 numpy array")
        n, p = a.size, a.ctypes.data
    if numel is not None and n != numel:
        raise ValueError(f"expected {numel} elements, got {n}")
    return C.c_void_p(p)


class Marchenko:
    """One context = one reflection response resident in HBM (mk_create .. mk_destroy)."""

    def __init__(self, nshot, nrec, nt, dt, dx, fmin, fmax, stream=None, rows=None, streamed=None):
        """rows = (row0, nrows): a row-sharded context that owns these receiver rows of R^ (mk_create_sharded).
        streamed = (resident_rows, window_rows): out-of-core R^, the other rows in pinned host memory (mk_create_streamed)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libmk needs a CUDA device (there is no CPU fallback)")
        self._L = load()
        self._h = C.c_void_p()
        self.nshot, self.nrec, self.nt = nshot, nrec, nt
        self.rows = (0, nrec) if rows is None else (int(rows[0]), int(rows[1]))
        if streamed is not None:
            if rows is not None:
                raise ValueError("row sharding and out-of-core streaming cannot be combined")
            rc = self._L.mk_create_streamed(C.byref(self._h), nshot, nrec, nt, dt, dx, fmin, fmax, int(streamed[0]), int(streamed[1]))
        else:
            rc = self._L.mk_create_sharded(C.byref(self._h), nshot, nrec, nt, dt, dx, fmin, fmax, self.rows[0], self.rows[1])
        if rc != MK_OK:
            msg = self._L.mk_last_error(self._h).decode() if self._h else "mk_create failed"
            if self._h:
                self._L.mk_destroy(self._h)
                self._h = C.c_void_p()
            raise MkError(rc, msg)
        self.set_stream(torch.cuda.current_stream().cuda_stream if stream is None else stream)

    # -- plumbing
    def _check(self, rc):
        if rc != MK_OK:
            raise MkError(rc, self._L.mk_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.mk_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_stream(self, cuda_stream):
        self._check(self._L.mk_set_stream(self._h, C.c_void_p(cuda_stream)))

    def set_option(self, key, value):
        self._check(self._L.mk_set_option(self._h, key, float(value)))

    def get_info(self, key) -> float:
        v = C.c_double()
        self._check(self._L.mk_get_info(self._h, key, C.byref(v)))
        return v.value

    def _outs(self, outs, ptr, numel):
        o = mk_outputs()
        for nm, t in (outs or {}).items():
            if nm not in OUTPUT_FIELDS:
                raise KeyError(nm)
            setattr(o, nm, ptr(t, numel=numel).value if t is not None else None)
        return o

    # -- the calls of include/mk.h
    def set_geometry(self, rec_of_shot=None, weights=None):
        """rec_of_shot: int array [nshot] (receiver co-located with each shot, -1 = none) or None; weights: float array
        [nshot] (quadrature weights of the shot grid) or None.  Before the first load_R."""
        import numpy as np
        ros = None if rec_of_shot is None else np.ascontiguousarray(rec_of_shot, dtype=np.int32)
        w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32)
        if ros is not None and ros.shape != (self.nshot,):
            raise ValueError("rec_of_shot must have nshot entries")
        if w is not None and w.shape != (self.nshot,):
            raise ValueError("weights must have nshot entries")
        self._check(self._L.mk_set_geometry(self._h, None if ros is None else C.c_void_p(ros.ctypes.data),
                                            None if w is None else C.c_void_p(w.ctypes.data)))

    def load_R(self, d_R_time, shot0=0):
        import torch
        nshots = d_R_time.shape[0]
        self._check(self._L.mk_load_R(self._h, _dev_ptr(d_R_time, torch.float32, nshots * self.nrec * self.nt), shot0, nshots))

    def load_R_rows(self, d_R_rows, shot0=0):
        """d_R_rows: [nshots][rows of this context][nt] (the receiver rows a row-sharded context owns, nothing else)."""
        import torch
        nshots, nrows = d_R_rows.shape[0], d_R_rows.shape[1]
        self._check(self._L.mk_load_R_rows(self._h, _dev_ptr(d_R_rows, torch.float32, nshots * nrows * self.nt), shot0, nshots))

    def load_R_host(self, h_R_time, shot0=0):
        nshots = h_R_time.shape[0]
        self._check(self._L.mk_load_R_host(self._h, _host_ptr(h_R_time, nshots * self.nrec * self.nt), shot0, nshots))

    def run(self, d_Gd, d_td, niter, outs):
        import torch
        nfoc = d_Gd.shape[0]
        self._nfoc = nfoc
        numel = nfoc * self.nrec * self.nt
        o = self._outs(outs, lambda t, numel: _dev_ptr(t, torch.float32, numel), numel)
        self._check(self._L.mk_run(self._h, _dev_ptr(d_Gd, torch.float32, numel), _dev_ptr(d_td, torch.float32, nfoc * self.nrec),
                                   nfoc, niter, C.byref(o)))

    def run_host(self, h_Gd, h_td, niter, outs):
        nfoc = h_Gd.shape[0]
        self._nfoc = nfoc
        numel = nfoc * self.nrec * self.nt
        o = self._outs(outs, lambda t, numel: _host_ptr(t, numel), numel)
        self._check(self._L.mk_run_host(self._h, _host_ptr(h_Gd, numel), _host_ptr(h_td, nfoc * self.nrec), nfoc, niter, C.byref(o)))

    def begin(self, d_Gd, d_td):
        import torch
        nfoc = d_Gd.shape[0]
        self._nfoc = nfoc
        self._check(self._L.mk_begin(self._h, _dev_ptr(d_Gd, torch.float32, nfoc * self.nrec * self.nt),
                                     _dev_ptr(d_td, torch.float32, nfoc * self.nrec), nfoc))

    def step(self, d_N_i=None):
        import torch
        self._check(self._L.mk_step(self._h, _dev_ptr(d_N_i, torch.float32, self._nfoc * self.nrec * self.nt) if d_N_i is not None else None))

    def step_contract(self):
        self._check(self._L.mk_step_contract(self._h))

    def step_post(self, d_N_i=None):
        import torch
        self._check(self._L.mk_step_post(self._h, _dev_ptr(d_N_i, torch.float32, self._nfoc * self.nrec * self.nt) if d_N_i is not None else None))

    def finish(self, outs):
        import torch
        numel = self._nfoc * self.nrec * self.nt
        o = self._outs(outs, lambda t, numel: _dev_ptr(t, torch.float32, numel), numel)
        self._check(self._L.mk_finish(self._h, C.byref(o)))

    def synthesis(self, d_N_in, d_S_out):
        import torch
        nfoc = d_N_in.shape[0]
        numel = nfoc * self.nrec * self.nt
        self._check(self._L.mk_synthesis(self._h, _dev_ptr(d_N_in, torch.float32, numel), _dev_ptr(d_S_out, torch.float32, numel), nfoc))

    # -- row sharding
    def operand(self, slot):
        """Torch views (no copy) of the operand planes of `slot`, each [nb][rows_per_bin][row_floats] fp32, and the view struct."""
        import torch
        v = mk_operand_view()
        self._check(self._L.mk_operand(self._h, slot, C.byref(v)))
        planes = []
        for p in range(v.nplanes):
            shape = (v.nb, v.rows_per_bin, v.row_floats)
            holder = type("_DevArray", (), {"__cuda_array_interface__": {"shape": shape, "typestr": "<f4", "data": (int(v.plane[p]), False),
                                                                        "version": 3, "strides": None}})()
            planes.append(torch.as_tensor(holder, device="cuda"))
        return planes, v

    def operand_reserve(self, nfoc):
        self._nfoc = nfoc
        self._check(self._L.mk_operand_reserve(self._h, nfoc))

    def operand_view(self, slot):
        v = mk_operand_view()
        self._check(self._L.mk_operand(self._h, slot, C.byref(v)))
        return v

    def operand_attach(self, slot, views):
        """views: mk_operand_view structs of the peers' operands of the same slot (pointers valid in this process)."""
        arr = (mk_operand_view * max(len(views), 1))(*views)
        self._check(self._L.mk_operand_attach(self._h, slot, len(views), arr))

    def operand_exchanged(self, slot):
        self._check(self._L.mk_operand_exchanged(self._h, slot))

    # ---- stream-ordered barrier between the ranks of a row-sharded run (include/mk.h mk_sync_*)
    def sync_create(self, rank, world):
        self._check(self._L.mk_sync_create(self._h, rank, world))

    def sync_flags(self) -> int:
        p = C.c_void_p()
        self._check(self._L.mk_sync_flags(self._h, C.byref(p)))
        return int(p.value)

    def sync_attach(self, flags_of_rank):
        """flags_of_rank: one device pointer (int) per rank, valid in this process; the own rank's entry may be None."""
        arr = (C.c_void_p * len(flags_of_rank))(*[C.c_void_p(p) if p else C.c_void_p() for p in flags_of_rank])
        self._check(self._L.mk_sync_attach(self._h, arr))

    def sync_barrier(self):
        self._check(self._L.mk_sync_barrier(self._h))

    def finish_prepare(self, field):
        self._check(self._L.mk_finish_prepare(self._h, field))

    def finish_complete(self, field, d_out):
        import torch
        self._check(self._L.mk_finish_complete(self._h, field, _dev_ptr(d_out, torch.float32, self._nfoc * self.nrec * self.nt)))

    def image(self, d_Gminus, d_image):
        import torch
        self._check(self._L.mk_image(self._h, _dev_ptr(d_Gminus, torch.float32, self._nfoc * self.nrec * self.nt),
                                     _dev_ptr(d_image, torch.float32, self._nfoc)))

    def image_static(self, d_Gminus, d_f1plus, d_image):
        """mk_image_static: the image of two explicit fields [nfoc][nrec][nt] -> d_image [nfoc], with the kernels' scratch in
        a static device array (no cudaMalloc / cudaFree in the call); nfoc is d_image's length.  Needs no run."""
        import torch
        nfoc = int(d_image.numel())
        self._check(self._L.mk_image_static(self._h, _dev_ptr(d_Gminus, torch.float32, nfoc * self.nrec * self.nt),
                                            _dev_ptr(d_f1plus, torch.float32, nfoc * self.nrec * self.nt),
                                            _dev_ptr(d_image, torch.float32, nfoc), nfoc))


def ipc_export(ptr: int) -> bytes:
    buf = C.create_string_buffer(64)
    rc = load().mk_ipc_export(C.c_void_p(ptr), buf)
    if rc != MK_OK:
        raise MkError(rc, "cudaIpcGetMemHandle failed")
    return buf.raw


def ipc_open(handle: bytes) -> int:
    p = C.c_void_p()
    rc = load().mk_ipc_open(C.c_char_p(handle), C.byref(p))
    if rc != MK_OK:
        raise MkError(rc, "cudaIpcOpenMemHandle failed")
    return p.value


def ipc_close(ptr: int) -> None:
    load().mk_ipc_close(C.c_void_p(ptr))


def version() -> str:
    return load().mk_version().decode()
