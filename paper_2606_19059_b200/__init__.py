"""B200-native spectral Ewald for the triply periodic Stokeslet sum (arXiv 2606.19059).

Thin ctypes binding over the C-ABI in include/se.h (libse_b200.so, built in-tree by
`python -m paper_2606_19059_b200.build`).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  PyTorch supplies device memory and streams.
There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libse_b200.so"

SE_FP64, SE_FP32 = 0, 1
SE_WINDOW_GAUSSIAN, SE_WINDOW_KAISER_BESSEL = 0, 1
WINDOWS = {"gaussian": SE_WINDOW_GAUSSIAN, "kb": SE_WINDOW_KAISER_BESSEL}
SE_BUF_TARGETS = 16
STAGES = ("sort", "p2p", "p2g", "fft", "scale", "ifft", "g2p", "sum")
(SE_STAGE_SORT, SE_STAGE_P2P, SE_STAGE_P2G, SE_STAGE_FFT, SE_STAGE_SCALE, SE_STAGE_IFFT,
 SE_STAGE_G2P, SE_STAGE_SUM) = range(8)
SE_NSTAGES = 8
(SE_BUF_UN, SE_BUF_UF, SE_BUF_GRID, SE_BUF_SPEC, SE_BUF_PERM_NEAR, SE_BUF_PERM_GRID,
 SE_BUF_CELL_START, SE_BUF_BIN_START) = range(8)

EXPORTS = ("se_plan_create", "se_plan_create_ex", "se_plan_create_tol", "se_select_params", "se_eval",
           "se_eval_targets", "se_set_targets", "se_eval_host", "se_plan_destroy", "se_strerror",
           "se_plan_info", "se_eval_stage", "se_buffer_read", "se_buffer_write",
           "se_set_profiling", "se_stage_ms", "se_last_launch_count", "se_measure_peak", "se_count_pairs", "se_scale_block",
           "se_scale_noalloc")


class SeInfo(C.Structure):
    _fields_ = [("N", C.c_int64), ("M", C.c_int), ("P", C.c_int), ("precision", C.c_int),
                ("L", C.c_double), ("xi", C.c_double), ("rc", C.c_double), ("h", C.c_double),
                ("m", C.c_double), ("eta", C.c_double), ("a", C.c_double), ("cw", C.c_double),
                ("ncell", C.c_int), ("nbin", C.c_int), ("grid_mode", C.c_int), ("nbins_total", C.c_int),
                ("nchunk", C.c_int), ("nmodes", C.c_int64),
                ("workspace_bytes", C.c_size_t), ("Nt", C.c_int64), ("window", C.c_int), ("nu", C.c_int),
                ("kb_beta", C.c_double), ("Mx", C.c_int), ("px0", C.c_int), ("fft_fused", C.c_int), ("fft_threads", C.c_int), ("fft_planes_own", C.c_int)]


class SePlanDesc(C.Structure):
    _fields_ = [("N", C.c_int64), ("Nt", C.c_int64), ("L", C.c_double), ("xi", C.c_double), ("rc", C.c_double),
                ("M", C.c_int), ("P", C.c_int), ("precision", C.c_int), ("window", C.c_int),
                ("Mx", C.c_int), ("px0", C.c_int), ("Nown", C.c_int64)]


class SeParams(C.Structure):
    _fields_ = [("rc", C.c_double), ("xi", C.c_double), ("M", C.c_int), ("P", C.c_int),
                ("EN", C.c_double), ("EF", C.c_double), ("Ew", C.c_double), ("s", C.c_double),
                ("model_ms", C.c_double)]


class SeError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().se_strerror(status).decode() if status >= 0 else "?"
        super().__init__(f"{where}: {msg} (se_status {status})")


_lib = None


def lib() -> C.CDLL:
    """Load libse_b200.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2606_19059_b200.build` "
                "(nvcc, sm_100a).  This package has no CPU or PyTorch fallback.")
        L = C.CDLL(str(LIB_PATH))
        vp, i64, dbl, i32 = C.c_void_p, C.c_int64, C.c_double, C.c_int
        L.se_plan_create.argtypes = [C.POINTER(vp), i64, dbl, dbl, dbl, i32, i32, i32]
        L.se_plan_create_ex.argtypes = [C.POINTER(vp), C.POINTER(SePlanDesc)]
        L.se_plan_create_tol.argtypes = [C.POINTER(vp), i64, i64, dbl, dbl, i32, i32, C.POINTER(SeParams)]
        L.se_select_params.argtypes = [i64, dbl, dbl, i32, i32, C.POINTER(SeParams)]
        L.se_eval.argtypes = [vp, vp, vp, vp, vp]
        L.se_eval_targets.argtypes = [vp, vp, vp, vp, vp, vp]
        L.se_set_targets.argtypes = [vp, vp]
        L.se_measure_peak.argtypes = [i32, i32, C.POINTER(dbl)]
        L.se_count_pairs.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
        L.se_scale_block.argtypes = [vp, vp, i32, i32, vp]
        L.se_scale_noalloc.argtypes = [vp, i32, i32, dbl, dbl, i32, i32, i32, vp]
        L.se_eval_host.argtypes = [vp, vp, vp, vp, vp]
        L.se_plan_destroy.argtypes = [vp]
        L.se_strerror.argtypes = [i32]
        L.se_strerror.restype = C.c_char_p
        L.se_plan_info.argtypes = [vp, C.POINTER(SeInfo)]
        L.se_eval_stage.argtypes = [vp, i32, vp, vp, vp, vp]
        L.se_buffer_read.argtypes = [vp, i32, vp, C.c_size_t, C.POINTER(C.c_size_t), vp]
        L.se_buffer_write.argtypes = [vp, i32, vp, C.c_size_t, vp]
        L.se_set_profiling.argtypes = [vp, i32]
        L.se_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.se_last_launch_count.argtypes = [vp, C.POINTER(i32)]
        for name in EXPORTS:
            if name != "se_strerror":
                getattr(L, name).restype = i32
        _lib = L
    return _lib


def _check(status: int, where: str):
    if status != 0:
        raise SeError(status, where)


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def scale_noalloc(spec, M, P, L, xi, precision="fp64", ky0=0, nky=None, stream=None):
    """se_scale_noalloc: K4 of a Gaussian-window plan (M, P, L, xi) in place on a complex block [3, M, nky, M // 2 + 1], without
    a plan and without any allocation (the multiplier table sits in a fixed 64 KB device array of the library: M <= 4096;
    calls that overlap on the GPU race on it)."""
    import torch
    nky = M if nky is None else nky
    cdt = torch.complex128 if precision == "fp64" else torch.complex64
    if not (spec.is_cuda and spec.is_contiguous() and spec.dtype == cdt and
            tuple(spec.shape) == (3, int(M), int(nky), int(M) // 2 + 1)):
        raise ValueError("scale_noalloc: need a contiguous CUDA complex tensor [3, M, nky, M // 2 + 1] of the given precision")
    _check(lib().se_scale_noalloc(C.c_void_p(spec.data_ptr()), int(M), int(P), float(L), float(xi), {"fp64": SE_FP64, "fp32": SE_FP32}[precision],
                                  int(ky0), int(nky), _stream_ptr(stream)), "se_scale_noalloc")
    return spec


def select_params(N, L, eps, window="gaussian", precision="fp64") -> SeParams:
    """se_select_params: (rc, xi, M, P) from a tolerance (host arithmetic only, no GPU needed)."""
    out = SeParams()
    _check(lib().se_select_params(int(N), float(L), float(eps), WINDOWS[window],
                                  {"fp64": SE_FP64, "fp32": SE_FP32}[precision], C.byref(out)), "se_select_params")
    return out


def measure_peak(which, reps=5) -> float:
    """se_measure_peak: TFLOP/s of a register-only chain, which = "fp64" | "fp64_tensor" | "fp32"; TB/s of a read + write
    stream for which = "hbm"."""
    v = C.c_double()
    _check(lib().se_measure_peak({"fp64": 0, "fp64_tensor": 1, "fp32": 2, "hbm": 3}[which], int(reps), C.byref(v)),
           "se_measure_peak")
    return v.value


class Plan:
    """se_plan_create[_ex|_tol] / se_eval / se_plan_destroy with torch tensors for memory."""

    def __init__(self, N, L, xi=None, rc=None, M=None, P=None, precision="fp64", window="gaussian", Nt=0, eps=None,
                 Mx=0, px0=0, Nown=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_19059_b200 needs a CUDA device (no CPU fallback)")
        self._h = C.c_void_p()
        self.precision = precision
        self.dtype = torch.float64 if precision == "fp64" else torch.float32
        prec = {"fp64": SE_FP64, "fp32": SE_FP32}[precision]
        win = WINDOWS[window]
        self.chosen = None
        if eps is not None:                                   # parameters from a tolerance
            self.chosen = SeParams()
            _check(lib().se_plan_create_tol(C.byref(self._h), int(N), int(Nt), float(L), float(eps), win, prec,
                                            C.byref(self.chosen)), "se_plan_create_tol")
            M, P = self.chosen.M, self.chosen.P
        elif win == SE_WINDOW_GAUSSIAN and not Nt and not Mx:
            _check(lib().se_plan_create(C.byref(self._h), int(N), float(L), float(xi), float(rc), int(M), int(P), prec),
                   "se_plan_create")
        else:
            d = SePlanDesc(int(N), int(Nt), float(L), float(xi), float(rc), int(M), int(P), prec, win, int(Mx), int(px0), int(Nown))
            _check(lib().se_plan_create_ex(C.byref(self._h), C.byref(d)), "se_plan_create_ex")
        self.N, self.M, self.P, self.Nt = int(N), int(M), int(P), int(Nt)
        self.Mx, self.px0 = (int(Mx), int(px0)) if Mx else (int(M), 0)       # slab plans (se.h se_plan_desc)
        self.Nown = int(Nown)

    # -- lifetime -----------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().se_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    # -- helpers --------------------------------------------------------------------------
    def _dev(self, t, name, n=None):
        if t is None:
            return C.c_void_p()
        n = self.N if n is None else n
        if not (t.is_cuda and t.is_contiguous() and t.dtype == self.dtype):
            raise ValueError(f"{name}: need a contiguous CUDA tensor of dtype {self.dtype}")
        if t.numel() != 3 * n:
            raise ValueError(f"{name}: need {n} x 3 = {3 * n} elements, got {t.numel()}")
        return C.c_void_p(t.data_ptr())

    def info(self) -> SeInfo:
        out = SeInfo()
        _check(lib().se_plan_info(self._h, C.byref(out)), "se_plan_info")
        return out

    # -- evaluation -------------------------------------------------------------------------
    def eval(self, x, f, u=None, stream=None):
        import torch
        if u is None:
            u = torch.empty((self.N, 3), dtype=self.dtype, device=x.device)
        _check(lib().se_eval(self._h, self._dev(x, "x"), self._dev(f, "f"), self._dev(u, "u"), _stream_ptr(stream)),
               "se_eval")
        return u

    def eval_targets(self, xs, f, xt, ut=None, stream=None):
        """Plans with Nt > 0: u at the Nt targets xt from the N sources (xs, f)."""
        import torch
        if ut is None:
            ut = torch.empty((self.Nt, 3), dtype=self.dtype, device=xs.device)
        _check(lib().se_eval_targets(self._h, self._dev(xs, "xs"), self._dev(f, "f"), self._dev(xt, "xt", self.Nt),
                                     self._dev(ut, "ut", self.Nt), _stream_ptr(stream)), "se_eval_targets")
        return ut

    def set_targets(self, xt):
        _check(lib().se_set_targets(self._h, self._dev(xt, "xt", self.Nt)), "se_set_targets")

    def eval_host(self, x_host, f_host, u_host, stream=None):
        """x_host, f_host, u_host: CPU tensors (ideally pinned); async on the stream."""
        for t in (x_host, f_host, u_host):
            if t.is_cuda or not t.is_contiguous() or t.dtype != self.dtype or t.numel() != 3 * self.N:
                raise ValueError("eval_host: need contiguous CPU tensors N x 3 of the plan's dtype")
        _check(lib().se_eval_host(self._h, C.c_void_p(x_host.data_ptr()), C.c_void_p(f_host.data_ptr()),
                                  C.c_void_p(u_host.data_ptr()), _stream_ptr(stream)), "se_eval_host")
        return u_host

    def stage(self, stage, x=None, f=None, u=None, stream=None):
        if isinstance(stage, str):
            stage = STAGES.index(stage)
        # the sum stage of a slab plan with ghost sources (Nown = Nt) takes the strengths of the owned points only
        nf = self.Nt if (self.Nown and stage == STAGES.index("sum")) else self.N
        _check(lib().se_eval_stage(self._h, int(stage), self._dev(x, "x"), self._dev(f, "f", nf),
                                   self._dev(u, "u", self.Nt or self.N), _stream_ptr(stream)), f"se_eval_stage({stage})")

    # -- buffers ------------------------------------------------------------------------------
    def _buf_shape(self, which):
        import torch
        tg = bool(which & SE_BUF_TARGETS)
        which &= ~SE_BUF_TARGETS
        N, M = (self.Nt if tg else self.N), self.M
        i = self.info()
        if which in (SE_BUF_UN, SE_BUF_UF):
            return (self.Nt or self.N, 3), self.dtype
        if which == SE_BUF_GRID:
            return (3, self.Mx, M, M), self.dtype
        if which == SE_BUF_SPEC:
            return (3, M, M, M // 2 + 1, 2), self.dtype
        if which in (SE_BUF_PERM_NEAR, SE_BUF_PERM_GRID):
            return (N,), torch.int32
        if which == SE_BUF_CELL_START:
            return (i.ncell ** 3 + 1,), torch.int32
        if which == SE_BUF_BIN_START:
            return (i.nbins_total + 1,), torch.int32
        raise ValueError(which)

    def read(self, which, stream=None):
        import torch
        shape, dt = self._buf_shape(which)
        out = torch.empty(shape, dtype=dt, device="cuda")
        nbytes = out.numel() * out.element_size()
        _check(lib().se_buffer_read(self._h, which, C.c_void_p(out.data_ptr()), nbytes, None, _stream_ptr(stream)),
               "se_buffer_read")
        return out

    def write(self, which, t, stream=None):
        shape, dt = self._buf_shape(which)
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise ValueError("write: need a contiguous CUDA tensor of the buffer's dtype")
        nbytes = t.numel() * t.element_size()
        _check(lib().se_buffer_write(self._h, which, C.c_void_p(t.data_ptr()), nbytes, _stream_ptr(stream)),
               "se_buffer_write")

    # -- timing ---------------------------------------------------------------------------------
    def scale_block(self, spec, ky0, nky, stream=None):
        """K4 in place on a complex block [3, M, nky, M // 2 + 1] of the spectrum (modes ky0 <= i_y < ky0 + nky)."""
        import torch
        cdt = torch.complex128 if self.precision == "fp64" else torch.complex64
        if not (spec.is_cuda and spec.is_contiguous() and spec.dtype == cdt and
                tuple(spec.shape) == (3, self.M, int(nky), self.M // 2 + 1)):
            raise ValueError("scale_block: need a contiguous CUDA complex tensor [3, M, nky, M // 2 + 1] of the plan's precision")
        _check(lib().se_scale_block(self._h, C.c_void_p(spec.data_ptr()), int(ky0), int(nky), _stream_ptr(stream)),
               "se_scale_block")
        return spec

    def set_profiling(self, on: bool):
        _check(lib().se_set_profiling(self._h, int(bool(on))), "se_set_profiling")

    def stage_ms(self):
        arr = (C.c_float * SE_NSTAGES)()
        _check(lib().se_stage_ms(self._h, arr), "se_stage_ms")
        return dict(zip(STAGES, [float(v) for v in arr]))

    def count_pairs(self):
        """se_count_pairs: (candidates, in-range pairs) of the last sorted point sets."""
        a, b = C.c_int64(), C.c_int64()
        _check(lib().se_count_pairs(self._h, C.byref(a), C.byref(b)), "se_count_pairs")
        return a.value, b.value

    def launch_count(self) -> int:
        n = C.c_int()
        _check(lib().se_last_launch_count(self._h, C.byref(n)), "se_last_launch_count")
        return n.value
