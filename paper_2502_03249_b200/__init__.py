"""Thin ctypes binding of libqcd_b200.so (include/qcd.h): argument marshalling only.

Every step of the path (layout permutation, Dslash, M, reductions, CG loop) runs in the CUDA
kernels of the library; PyTorch appears only as the owner of device memory and of the stream.
There is no CPU fallback: if the shared object is missing, or no sm_100 device is present,
calls raise.

    ctx = Context((16, 16, 16, 16), precision=64)
    U = ctx.field(QCD_GAUGE).upload(U_host)            # complex128 [V,4,3,3]
    b = ctx.field(QCD_SPINOR_EVEN).upload(b_host)      # complex128 [V,3]
    x = ctx.field(QCD_SPINOR_EVEN)
    info = ctx.qcd_cg_solve(U, b, x, m=0.05, tol=1e-10, maxiter=10000)
    x_host = x.download()
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from .build import LIB_PATH

QCD_OK, QCD_EINVAL, QCD_ENOMEM, QCD_ECUDA, QCD_ENOTCONVERGED, QCD_EBREAKDOWN = range(6)
QCD_SPINOR_EVEN, QCD_SPINOR_ODD, QCD_SPINOR_FULL, QCD_GAUGE, QCD_GAUGE_2ROW, QCD_COLOUR_MATRIX = range(6)
QCD_MAX_RHS = 8
QCD_K_DSLASH, QCD_K_DSLASH_EPI, QCD_K_UPDATE_XR, QCD_K_UPDATE_P, QCD_K_MISC = range(5)
QCD_RE_DOT_STATIC_MAX_REALS = 50331648      # include/qcd.h: one 64^4 half-field

# every symbol include/qcd.h declares
SYMBOLS = [
    "qcd_strerror", "qcd_last_error", "qcd_init", "qcd_finalize", "qcd_field_bytes",
    "qcd_workspace_bytes", "qcd_field_alloc", "qcd_field_free", "qcd_field_upload",
    "qcd_field_download", "qcd_set_workspace", "qcd_dslash_eo", "qcd_dslash_oe", "qcd_apply_M",
    "qcd_cg_solve", "qcd_cg_begin", "qcd_cg_iterate", "qcd_cg_poll", "qcd_cg_finish",
    "qcd_cg_solve_host", "qcd_profile_enable", "qcd_profile_read", "qcd_launch_count",
    "qcd_set_dslash_variant", "qcd_set_traversal_chunk", "qcd_set_cg_loop", "qcd_last_cg_loop", "qcd_last_cg_cluster", "qcd_set_cg_cluster", "qcd_cg_timeline_enable", "qcd_cg_timeline_read", "qcd_re_dot", "qcd_re_dot_static", "qcd_stream_read", "qcd_stream_read_resident", "qcd_stream_mix", "qcd_stream_bulk", "qcd_cg_history",
    # variants and mixed precision
    "qcd_gauge_compress", "qcd_gauge_fix_temporal", "qcd_gauge_set_temporal_unit", "qcd_spinor_rotate",
    "qcd_workspace_bytes_multi", "qcd_dslash_eo_multi", "qcd_dslash_oe_multi", "qcd_cg_solve_multi",
    "qcd_cg_begin_multi", "qcd_cg_finish_multi", "qcd_field_convert", "qcd_cg_solve_mixed",
]


class qcd_cg_info(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("converged", ctypes.c_int), ("rel_resid", ctypes.c_double),
                ("bnorm2", ctypes.c_double), ("seconds", ctypes.c_double)]


class qcd_mixed_info(ctypes.Structure):
    _fields_ = [("converged", ctypes.c_int), ("outer", ctypes.c_int), ("inner_iters", ctypes.c_int),
                ("m_applications_fp64", ctypes.c_int), ("true_resid", ctypes.c_double), ("seconds", ctypes.c_double)]


class QcdError(RuntimeError):
    def __init__(self, status: int, where: str, msg: str):
        super().__init__(f"{where}: status {status} ({msg})")
        self.status = status


_LIB = None


def load_library() -> ctypes.CDLL:
    """dlopen libqcd_b200.so; raises if it has not been built (python -m paper_2502_03249_b200.build)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2502_03249_b200.build` "
                           "(there is no fallback path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    P = ctypes.POINTER
    sig = {
        "qcd_strerror": (ctypes.c_char_p, [ci]),
        "qcd_last_error": (ctypes.c_char_p, [vp]),
        "qcd_init": (ci, [P(vp), P(ci), ci, vp]),
        "qcd_finalize": (ci, [vp]),
        "qcd_field_bytes": (sz, [vp, ci]),
        "qcd_workspace_bytes": (sz, [vp]),
        "qcd_field_alloc": (ci, [vp, ci, vp, sz, P(vp)]),
        "qcd_field_free": (ci, [vp]),
        "qcd_field_upload": (ci, [vp, vp]),
        "qcd_field_download": (ci, [vp, vp]),
        "qcd_set_workspace": (ci, [vp, vp, sz]),
        "qcd_dslash_eo": (ci, [vp, vp, vp, vp]),
        "qcd_dslash_oe": (ci, [vp, vp, vp, vp]),
        "qcd_apply_M": (ci, [vp, vp, vp, vp, cd]),
        "qcd_cg_solve": (ci, [vp, vp, vp, vp, cd, cd, ci, P(qcd_cg_info)]),
        "qcd_cg_begin": (ci, [vp, vp, vp, vp, cd, cd, ci]),
        "qcd_cg_iterate": (ci, [vp, ci]),
        "qcd_cg_poll": (ci, [vp, P(ci), P(ci), P(cd)]),
        "qcd_cg_finish": (ci, [vp, P(qcd_cg_info)]),
        "qcd_cg_solve_host": (ci, [vp, vp, vp, vp, vp, vp, cd, cd, ci, P(qcd_cg_info)]),
        "qcd_profile_enable": (ci, [vp, ci]),
        "qcd_profile_read": (ci, [vp, ci, P(ci), P(cd)]),
        "qcd_launch_count": (ctypes.c_longlong, [vp]),
        "qcd_set_dslash_variant": (ci, [vp, ci]),
        "qcd_set_traversal_chunk": (ci, [vp, ci]),
        "qcd_set_cg_loop": (ci, [vp, ci]),
        "qcd_last_cg_loop": (ci, [vp]),
        "qcd_last_cg_cluster": (ci, [vp]),
        "qcd_set_cg_cluster": (ci, [vp, ci]),
        "qcd_cg_timeline_enable": (ci, [vp, ci]),
        "qcd_cg_timeline_read": (ci, [vp, P(ctypes.c_ulonglong), ci, P(ci)]),
        "qcd_re_dot": (ci, [vp, vp, vp, P(cd)]),
        "qcd_re_dot_static": (ci, [vp, vp, sz, ci, vp, vp, ctypes.c_char_p, sz]),
        "qcd_stream_read": (ci, [vp, vp, ci, P(cd)]),
        "qcd_stream_read_resident": (ci, [vp, vp, ci, P(cd)]),
        "qcd_stream_mix": (ci, [vp, vp, vp, ci, ci, ci, P(cd)]),
        "qcd_stream_bulk": (ci, [vp, vp, ci, ci, ci, ci, ci, ci, P(cd)]),
        "qcd_cg_history": (ci, [vp, ci, P(cd), ci, P(ci)]),
        "qcd_gauge_compress": (ci, [vp, vp, vp]),
        "qcd_gauge_fix_temporal": (ci, [vp, vp, vp, vp]),
        "qcd_gauge_set_temporal_unit": (ci, [vp, ci]),
        "qcd_spinor_rotate": (ci, [vp, vp, vp, vp, ci]),
        "qcd_workspace_bytes_multi": (sz, [vp, ci]),
        "qcd_dslash_eo_multi": (ci, [vp, vp, ci, P(vp), P(vp)]),
        "qcd_dslash_oe_multi": (ci, [vp, vp, ci, P(vp), P(vp)]),
        "qcd_cg_solve_multi": (ci, [vp, vp, ci, P(vp), P(vp), cd, cd, ci, P(qcd_cg_info)]),
        "qcd_cg_begin_multi": (ci, [vp, vp, ci, P(vp), P(vp), cd, cd, ci]),
        "qcd_cg_finish_multi": (ci, [vp, P(qcd_cg_info)]),
        "qcd_field_convert": (ci, [vp, vp]),
        "qcd_cg_solve_mixed": (ci, [vp, vp, vp, vp, vp, vp, vp, vp, cd, cd, cd, ci, ci, P(qcd_mixed_info)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _LIB = lib
    return lib


def qcd_re_dot_static(a_dev: int, b_dev: int, n_reals: int, precision: int, cuda_stream: int, result_dev: int) -> None:
    """The allocation-free dot product (include/qcd.h): device addresses in, one double written at result_dev on
    `cuda_stream`; asynchronous.  No context, no cudaMalloc; n_reals <= QCD_RE_DOT_STATIC_MAX_REALS."""
    lib = load_library()
    err = ctypes.create_string_buffer(512)
    s = lib.qcd_re_dot_static(ctypes.c_void_p(a_dev), ctypes.c_void_p(b_dev), n_reals, precision,
                              ctypes.c_void_p(cuda_stream), ctypes.c_void_p(result_dev), err, len(err))
    if s != QCD_OK:
        raise QcdError(s, "qcd_re_dot_static", err.value.decode())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2502_03249_b200 needs a CUDA device (sm_100); there is no CPU fallback")
    return torch


class Field:
    """A caller-owned torch uint8 device buffer bound to a qcd_field descriptor."""

    def __init__(self, ctx: "Context", kind: int, buf=None):
        """buf: an existing uint8 device tensor to bind (e.g. the links of another context on the same
        lattice and precision: qcd_field_alloc only binds, so descriptors may share memory)."""
        torch = _torch()
        self.ctx, self.kind = ctx, kind
        self.nbytes = ctx.qcd_field_bytes(kind)
        if buf is None:
            buf = torch.empty(self.nbytes, dtype=torch.uint8, device=ctx.device)
        self.buf = buf
        h = ctypes.c_void_p()
        ctx._check(ctx.lib.qcd_field_alloc(ctx.handle, kind, ctypes.c_void_p(self.buf.data_ptr()), self.nbytes,
                                            ctypes.byref(h)), "qcd_field_alloc")
        self.handle = h

    def host_shape(self):
        v = self.ctx.volume
        if self.kind in (QCD_GAUGE, QCD_GAUGE_2ROW):
            return (v, 4, 3, 3)
        return (v, 3, 3) if self.kind == QCD_COLOUR_MATRIX else (v, 3)

    def upload(self, host: np.ndarray) -> "Field":
        """qcd_field_upload: host array in the canonical layout, complex dtype of the context precision."""
        a = np.ascontiguousarray(host, dtype=self.ctx.cdtype)
        if a.shape != self.host_shape():
            raise ValueError(f"expected host shape {self.host_shape()}, got {a.shape}")
        self.ctx._check(self.ctx.lib.qcd_field_upload(self.handle, a.ctypes.data_as(ctypes.c_void_p)), "qcd_field_upload")
        return self

    def download(self, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.empty(self.host_shape(), dtype=self.ctx.cdtype)
        assert out.flags.c_contiguous and out.dtype == self.ctx.cdtype and out.shape == self.host_shape()
        self.ctx._check(self.ctx.lib.qcd_field_download(self.handle, out.ctypes.data_as(ctypes.c_void_p)), "qcd_field_download")
        return out

    def free(self):
        if self.handle:
            self.ctx.lib.qcd_field_free(self.handle)
            self.handle = None
        self.buf = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """qcd_ctx plus the torch-owned workspace.  Methods carry the C names and marshal only."""

    def __init__(self, dims, precision: int = 64, stream=None, device="cuda:0", workspace: bool = True, nrhs: int = 1):
        torch = _torch()
        self.lib = load_library()
        self.dims = tuple(int(d) for d in dims)
        self.precision = int(precision)
        self.cdtype = np.complex128 if self.precision == 64 else np.complex64
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.handle = ctypes.c_void_p()
        d = (ctypes.c_int * 4)(*self.dims)
        st = self.lib.qcd_init(ctypes.byref(self.handle), d, self.precision, ctypes.c_void_p(self.stream.cuda_stream))
        if st != QCD_OK:
            self.handle = None
            raise QcdError(st, "qcd_init", self.lib.qcd_last_error(None).decode())
        self.volume = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self.ws = None
        if workspace:
            self.ws = torch.empty(self.qcd_workspace_bytes_multi(nrhs), dtype=torch.uint8, device=self.device)
            self._check(self.lib.qcd_set_workspace(self.handle, ctypes.c_void_p(self.ws.data_ptr()), self.ws.numel()),
                        "qcd_set_workspace")

    # ---- helpers -------------------------------------------------------------------------
    def _check(self, st: int, where: str, ok=(QCD_OK,)):
        if st not in ok:
            raise QcdError(st, where, self.lib.qcd_last_error(self.handle).decode())
        return st

    def field(self, kind: int, buf=None) -> Field:
        return Field(self, kind, buf)

    def close(self):
        if self.handle:
            self.lib.qcd_finalize(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C calls ---------------------------------------------------------------------
    def qcd_field_bytes(self, kind: int) -> int:
        return int(self.lib.qcd_field_bytes(self.handle, kind))

    def qcd_workspace_bytes(self) -> int:
        return int(self.lib.qcd_workspace_bytes(self.handle))

    def qcd_dslash_eo(self, U: Field, out_even: Field, in_odd: Field):
        self._check(self.lib.qcd_dslash_eo(self.handle, U.handle, out_even.handle, in_odd.handle), "qcd_dslash_eo")

    def qcd_dslash_oe(self, U: Field, out_odd: Field, in_even: Field):
        self._check(self.lib.qcd_dslash_oe(self.handle, U.handle, out_odd.handle, in_even.handle), "qcd_dslash_oe")

    def qcd_apply_M(self, U: Field, out_even: Field, in_even: Field, m: float):
        self._check(self.lib.qcd_apply_M(self.handle, U.handle, out_even.handle, in_even.handle, float(m)), "qcd_apply_M")

    @staticmethod
    def _info(i: qcd_cg_info, status: int) -> dict:
        return dict(status=status, iters=i.iters, converged=bool(i.converged), rel_resid=i.rel_resid,
                    bnorm2=i.bnorm2, seconds=i.seconds)

    _CG_OK = (QCD_OK, QCD_ENOTCONVERGED, QCD_EBREAKDOWN)

    def qcd_cg_solve(self, U: Field, b: Field, x: Field, m: float, tol: float, maxiter: int) -> dict:
        i = qcd_cg_info()
        st = self._check(self.lib.qcd_cg_solve(self.handle, U.handle, b.handle, x.handle, float(m), float(tol),
                                               int(maxiter), ctypes.byref(i)), "qcd_cg_solve", self._CG_OK)
        return self._info(i, st)

    def qcd_cg_begin(self, U: Field, b: Field, x: Field, m: float, tol: float, maxiter: int):
        self._check(self.lib.qcd_cg_begin(self.handle, U.handle, b.handle, x.handle, float(m), float(tol), int(maxiter)),
                    "qcd_cg_begin")

    def qcd_cg_iterate(self, n: int):
        self._check(self.lib.qcd_cg_iterate(self.handle, int(n)), "qcd_cg_iterate")

    def qcd_cg_poll(self):
        st, it, rr = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
        self._check(self.lib.qcd_cg_poll(self.handle, ctypes.byref(st), ctypes.byref(it), ctypes.byref(rr)), "qcd_cg_poll")
        return st.value, it.value, rr.value

    def qcd_cg_finish(self) -> dict:
        i = qcd_cg_info()
        st = self._check(self.lib.qcd_cg_finish(self.handle, ctypes.byref(i)), "qcd_cg_finish", self._CG_OK)
        return self._info(i, st)

    def qcd_cg_solve_host(self, U: Field, b_dev: Field, x_dev: Field, b_host_ptr: int, x_host_ptr: int,
                          m: float, tol: float, maxiter: int) -> dict:
        """b_host_ptr / x_host_ptr: host addresses (e.g. pinned torch tensors' data_ptr()) of canonical spinors."""
        i = qcd_cg_info()
        st = self._check(self.lib.qcd_cg_solve_host(self.handle, U.handle, b_dev.handle, x_dev.handle,
                                                    ctypes.c_void_p(b_host_ptr), ctypes.c_void_p(x_host_ptr),
                                                    float(m), float(tol), int(maxiter), ctypes.byref(i)),
                         "qcd_cg_solve_host", self._CG_OK)
        return self._info(i, st)

    def qcd_cg_history(self, rhs: int = 0, cap: int = 16384) -> np.ndarray:
        """rr_k / bb after k = 1 .. iters M applications of the most recent solve (numpy float64)."""
        out = np.zeros(int(cap), dtype=np.float64)
        n = ctypes.c_int()
        self._check(self.lib.qcd_cg_history(self.handle, int(rhs), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(cap),
                                                 ctypes.byref(n)),
                    "qcd_cg_history")
        return out[: n.value].copy()

    def qcd_profile_enable(self, on: bool):
        self._check(self.lib.qcd_profile_enable(self.handle, 1 if on else 0), "qcd_profile_enable")

    def qcd_profile_read(self, which: int):
        n, ms = ctypes.c_int(), ctypes.c_double()
        self._check(self.lib.qcd_profile_read(self.handle, int(which), ctypes.byref(n), ctypes.byref(ms)), "qcd_profile_read")
        return n.value, ms.value

    def qcd_launch_count(self) -> int:
        return int(self.lib.qcd_launch_count(self.handle))

    def qcd_set_dslash_variant(self, variant: int):
        self._check(self.lib.qcd_set_dslash_variant(self.handle, int(variant)), "qcd_set_dslash_variant")

    def qcd_set_traversal_chunk(self, width: int):
        self._check(self.lib.qcd_set_traversal_chunk(self.handle, int(width)), "qcd_set_traversal_chunk")

    def qcd_set_cg_loop(self, mode: int):
        self._check(self.lib.qcd_set_cg_loop(self.handle, int(mode)), "qcd_set_cg_loop")

    def qcd_last_cg_loop(self) -> int:
        return int(self.lib.qcd_last_cg_loop(self.handle))

    def qcd_last_cg_cluster(self) -> int:
        return int(self.lib.qcd_last_cg_cluster(self.handle))

    def qcd_set_cg_cluster(self, on: bool):
        self._check(self.lib.qcd_set_cg_cluster(self.handle, 1 if on else 0), "qcd_set_cg_cluster")

    def qcd_cg_timeline_enable(self, on: bool):
        self._check(self.lib.qcd_cg_timeline_enable(self.handle, 1 if on else 0), "qcd_cg_timeline_enable")

    def qcd_cg_timeline_read(self, cap_iters: int = 64) -> np.ndarray:
        """uint64 [2][n][9] %globaltimer stamps (block 0, last block) of the iterations that ran (n <= cap_iters <= 64)."""
        cap = min(int(cap_iters), 64)
        out = np.zeros((2, cap, 9), dtype=np.uint64)
        n = ctypes.c_int()
        self._check(self.lib.qcd_cg_timeline_read(self.handle, out.ctypes.data_as(ctypes.POINTER(ctypes.c_ulonglong)), cap,
                                                  ctypes.byref(n)), "qcd_cg_timeline_read")
        return out[:, : n.value, :].copy()

    def qcd_re_dot(self, a: Field, b: Field) -> float:
        r = ctypes.c_double()
        self._check(self.lib.qcd_re_dot(self.handle, a.handle, b.handle, ctypes.byref(r)), "qcd_re_dot")
        return r.value

    def qcd_stream_read(self, f: Field, reps: int) -> float:
        ms = ctypes.c_double()
        self._check(self.lib.qcd_stream_read(self.handle, f.handle, int(reps), ctypes.byref(ms)), "qcd_stream_read")
        return ms.value

    def qcd_stream_read_resident(self, f: Field, passes: int) -> float:
        ms = ctypes.c_double()
        self._check(self.lib.qcd_stream_read_resident(self.handle, f.handle, int(passes), ctypes.byref(ms)), "qcd_stream_read_resident")
        return ms.value

    def qcd_stream_mix(self, src: Field, dst: Field, read_planes: int, write_planes: int, reps: int) -> float:
        ms = ctypes.c_double()
        self._check(self.lib.qcd_stream_mix(self.handle, src.handle, dst.handle, int(read_planes), int(write_planes), int(reps),
                                            ctypes.byref(ms)), "qcd_stream_mix")
        return ms.value

    def qcd_stream_bulk(self, src: Field, rows: int, copies: int, hops: int, stages: int, producers: int, reps: int) -> float:
        ms = ctypes.c_double()
        self._check(self.lib.qcd_stream_bulk(self.handle, src.handle, int(rows), int(copies), int(hops), int(stages), int(producers), int(reps),
                                             ctypes.byref(ms)), "qcd_stream_bulk")
        return ms.value

    # ---- variants -------------------------------------------------------
    @staticmethod
    def _handles(fields):
        return (ctypes.c_void_p * len(fields))(*[f.handle.value for f in fields])

    def qcd_workspace_bytes_multi(self, n: int) -> int:
        return int(self.lib.qcd_workspace_bytes_multi(self.handle, int(n)))

    def qcd_gauge_compress(self, U: Field, U12: Field):
        self._check(self.lib.qcd_gauge_compress(self.handle, U.handle, U12.handle), "qcd_gauge_compress")

    def qcd_gauge_fix_temporal(self, U: Field, U_fixed: Field, g: Field):
        self._check(self.lib.qcd_gauge_fix_temporal(self.handle, U.handle, U_fixed.handle, g.handle), "qcd_gauge_fix_temporal")

    def qcd_gauge_set_temporal_unit(self, U: Field, on: bool):
        self._check(self.lib.qcd_gauge_set_temporal_unit(U.handle, 1 if on else 0), "qcd_gauge_set_temporal_unit")

    def qcd_spinor_rotate(self, g: Field, out: Field, in_: Field, dagger: bool = False):
        self._check(self.lib.qcd_spinor_rotate(self.handle, g.handle, out.handle, in_.handle, 1 if dagger else 0), "qcd_spinor_rotate")

    def qcd_dslash_eo_multi(self, U: Field, out_even, in_odd):
        self._check(self.lib.qcd_dslash_eo_multi(self.handle, U.handle, len(out_even), self._handles(out_even),
                                                 self._handles(in_odd)), "qcd_dslash_eo_multi")

    def qcd_dslash_oe_multi(self, U: Field, out_odd, in_even):
        self._check(self.lib.qcd_dslash_oe_multi(self.handle, U.handle, len(out_odd), self._handles(out_odd),
                                                 self._handles(in_even)), "qcd_dslash_oe_multi")

    def qcd_cg_solve_multi(self, U: Field, b, x, m: float, tol: float, maxiter: int):
        n = len(b)
        infos = (qcd_cg_info * n)()
        st = self._check(self.lib.qcd_cg_solve_multi(self.handle, U.handle, n, self._handles(b), self._handles(x),
                                                     float(m), float(tol), int(maxiter), infos), "qcd_cg_solve_multi", self._CG_OK)
        return [self._info(infos[i], st) for i in range(n)]

    def qcd_cg_begin_multi(self, U: Field, b, x, m: float, tol: float, maxiter: int):
        self._multi_n = len(b)
        self._check(self.lib.qcd_cg_begin_multi(self.handle, U.handle, len(b), self._handles(b), self._handles(x),
                                                float(m), float(tol), int(maxiter)), "qcd_cg_begin_multi")

    def qcd_cg_finish_multi(self):
        n = self._multi_n
        infos = (qcd_cg_info * n)()
        st = self._check(self.lib.qcd_cg_finish_multi(self.handle, infos), "qcd_cg_finish_multi", self._CG_OK)
        return [self._info(infos[i], st) for i in range(n)]

    def qcd_field_convert(self, dst: Field, src: Field):
        """dst and src belong to two contexts of different precision on the same lattice and stream."""
        dst.ctx._check(self.lib.qcd_field_convert(dst.handle, src.handle), "qcd_field_convert")

    def qcd_cg_solve_mixed(self, ctx32: "Context", U64: Field, U32: Field, b: Field, x: Field, rhs32: Field, e32: Field,
                           m: float, tol: float, inner_tol: float, maxiter: int, max_outer: int = 50) -> dict:
        i = qcd_mixed_info()
        st = self._check(self.lib.qcd_cg_solve_mixed(self.handle, ctx32.handle, U64.handle, U32.handle, b.handle, x.handle,
                                                     rhs32.handle, e32.handle, float(m), float(tol), float(inner_tol),
                                                     int(maxiter), int(max_outer), ctypes.byref(i)),
                         "qcd_cg_solve_mixed", self._CG_OK)
        return dict(status=st, converged=bool(i.converged), outer=i.outer, inner_iters=i.inner_iters,
                    m_applications_fp64=i.m_applications_fp64, true_resid=i.true_resid, seconds=i.seconds)
