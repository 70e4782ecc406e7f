"""ctypes binding of libsfft.so (include/sfft.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for
device memory and streams only.  There is NO CPU fallback: if the library is missing or no CUDA
device is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_NAME = "libsfft.so"

# every symbol include/sfft.h declares (tests check the built library exports all of them)
EXPORTED_SYMBOLS = [
    "sfft_plan_create", "sfft_plan_destroy", "sfft_num_coeffs", "sfft_workspace_bytes",
    "sfft_status_string", "sfft_build_system", "sfft_build_system_exact", "sfft_solve", "sfft_subtract", "sfft_subtract_prepare",
    "sfft_probe_fp64", "sfft_last_launch_count", "sfft_plan_fused", "sfft_plan_set_solve_ctas", "sfft_version",
    "sfft_profile_enable", "sfft_profile_read", "sfft_median_combine", "sfft_aperture_stats", "sfft_resample_affine", "sfft_resample_mask_affine",
    "sfft_cut_stamps", "sfft_multi_template_difference", "sfft_multi_template_difference_plans", "sfft_solve_static",
]

SOLVE_STATIC_MAX_N = 768   # SFFT_SOLVE_STATIC_MAX_N (include/sfft.h)

STAGE_NAMES = ["build.row_fwd", "build.col_fwd", "build.cross_KK", "build.cross_KS",
               "build.lag_gather", "solve", "subtract.row_fwd", "subtract.mix", "subtract.row_inv",
               "build.kb_sparse"]


class SfftError(RuntimeError):
    def __init__(self, code: int, where: str, text: str):
        super().__init__(f"{where}: {text} (sfft_status {code})")
        self.code = code


def lib_path() -> str:
    return os.path.join(_HERE, _LIB_NAME)


_lib = None


def load_library():
    """dlopen the in-tree libsfft.so and declare the prototypes.  Raises if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
            "(there is no CPU fallback for the SFFT hot path)")
    lib = ctypes.CDLL(path)
    vp, i32, dbl_p = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)
    lib.sfft_plan_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32, i32, i32]
    lib.sfft_plan_create.restype = i32
    lib.sfft_plan_destroy.argtypes = [vp]
    lib.sfft_plan_destroy.restype = i32
    lib.sfft_num_coeffs.argtypes = [vp]
    lib.sfft_num_coeffs.restype = i32
    lib.sfft_workspace_bytes.argtypes = [vp]
    lib.sfft_workspace_bytes.restype = ctypes.c_size_t
    lib.sfft_status_string.argtypes = [i32]
    lib.sfft_status_string.restype = ctypes.c_char_p
    lib.sfft_build_system.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.sfft_build_system.restype = i32
    lib.sfft_solve.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.sfft_solve.restype = i32
    lib.sfft_solve_static.argtypes = [vp, vp, i32, vp, vp, vp]
    lib.sfft_solve_static.restype = i32
    lib.sfft_subtract.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.sfft_subtract.restype = i32
    lib.sfft_probe_fp64.argtypes = [i32, i32, dbl_p, dbl_p, vp]
    lib.sfft_probe_fp64.restype = i32
    lib.sfft_last_launch_count.argtypes = [vp, i32]
    lib.sfft_last_launch_count.restype = i32
    lib.sfft_build_system_exact.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.sfft_build_system_exact.restype = i32
    lib.sfft_subtract_prepare.argtypes = [vp, vp, vp]
    lib.sfft_subtract_prepare.restype = i32
    lib.sfft_plan_fused.argtypes = [vp]
    lib.sfft_plan_fused.restype = i32
    lib.sfft_plan_set_solve_ctas.argtypes = [vp, i32]
    lib.sfft_plan_set_solve_ctas.restype = i32
    lib.sfft_median_combine.argtypes = [vp, vp, i32, ctypes.c_size_t, vp, vp]
    lib.sfft_median_combine.restype = i32
    lib.sfft_cut_stamps.argtypes = [vp, vp, vp, i32, i32, vp, vp, i32, i32, vp, vp]
    lib.sfft_cut_stamps.restype = i32
    lib.sfft_multi_template_difference.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp]
    lib.sfft_multi_template_difference.restype = i32
    lib.sfft_multi_template_difference_plans.argtypes = [vp, i32, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp]
    lib.sfft_multi_template_difference_plans.restype = i32
    lib.sfft_aperture_stats.argtypes = [vp, vp, i32, i32, vp, vp, i32, ctypes.c_double, vp, vp, vp]
    lib.sfft_aperture_stats.restype = i32
    lib.sfft_resample_affine.argtypes = [vp, i32, i32, vp, i32, vp, i32, i32, vp, vp]
    lib.sfft_resample_affine.restype = i32
    lib.sfft_resample_mask_affine.argtypes = [vp, i32, i32, vp, i32, ctypes.c_double, vp, i32, i32, vp]
    lib.sfft_resample_mask_affine.restype = i32
    lib.sfft_profile_enable.argtypes = [vp, i32]
    lib.sfft_profile_enable.restype = i32
    lib.sfft_profile_read.argtypes = [vp, i32, dbl_p, ctypes.POINTER(i32), i32]
    lib.sfft_profile_read.restype = i32
    lib.sfft_version.argtypes = []
    lib.sfft_version.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(lib, code: int, where: str):
    if code != 0:
        raise SfftError(code, where, lib.sfft_status_string(code).decode())


def _stream_handle(stream) -> Optional[int]:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _dev_ptr(t, dtype, numel, name):
    import torch
    if t is None:
        return ctypes.c_void_p(0)
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor (device memory is the caller's)")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise ValueError(f"{name}: need contiguous {dtype} with {numel} elements, got "
                         f"{t.dtype} {tuple(t.shape)} contiguous={t.is_contiguous()}")
    return ctypes.c_void_p(t.data_ptr())


class SfftPlan:
    """sfft_plan_create / sfft_build_system / sfft_solve / sfft_subtract with torch CUDA tensors.

    All methods only enqueue work on the given (default: current) torch stream.
    """

    def __init__(self, H: int, W: int, w: int, DK: int, DB: int):
        self._lib = load_library()
        self._p = ctypes.c_void_p(0)
        _check(self._lib, self._lib.sfft_plan_create(ctypes.byref(self._p), H, W, w, DK, DB),
               "sfft_plan_create")
        self.H, self.W, self.w, self.DK, self.DB = H, W, w, DK, DB
        self.N = self._lib.sfft_num_coeffs(self._p)

    # -- lifetime
    def close(self):
        if getattr(self, "_p", None) is not None and self._p.value:
            self._lib.sfft_plan_destroy(self._p)
            self._p = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def workspace_bytes(self) -> int:
        return int(self._lib.sfft_workspace_bytes(self._p))

    # -- the four hot calls
    def build_system(self, R, S, mask, A=None, b=None, stream=None):
        import torch
        P = self.H * self.W
        if A is None:
            A = torch.empty((self.N, self.N), dtype=torch.float64, device=R.device)
        if b is None:
            b = torch.empty(self.N, dtype=torch.float64, device=R.device)
        _check(self._lib, self._lib.sfft_build_system(
            self._p, _dev_ptr(R, torch.float64, P, "R"), _dev_ptr(S, torch.float64, P, "S"),
            _dev_ptr(mask, torch.uint8, P, "mask"), _dev_ptr(A, torch.float64, self.N * self.N, "A"),
            _dev_ptr(b, torch.float64, self.N, "b"), _stream_handle(stream)), "sfft_build_system")
        return A, b

    def build_system_exact(self, R, S, mask, A=None, b=None, stream=None):
        """sfft_build_system_exact: the normal equations of the literal objective (masked pixels
        dropped from the sum, images used unmasked)."""
        import torch
        P = self.H * self.W
        if A is None:
            A = torch.empty((self.N, self.N), dtype=torch.float64, device=R.device)
        if b is None:
            b = torch.empty(self.N, dtype=torch.float64, device=R.device)
        _check(self._lib, self._lib.sfft_build_system_exact(
            self._p, _dev_ptr(R, torch.float64, P, "R"), _dev_ptr(S, torch.float64, P, "S"),
            _dev_ptr(mask, torch.uint8, P, "mask"), _dev_ptr(A, torch.float64, self.N * self.N, "A"),
            _dev_ptr(b, torch.float64, self.N, "b"), _stream_handle(stream)), "sfft_build_system_exact")
        return A, b

    def solve(self, A, b, coeffs=None, info=None, stream=None):
        import torch
        if coeffs is None:
            coeffs = torch.empty(self.N, dtype=torch.float64, device=A.device)
        if info is None:
            info = torch.zeros(1, dtype=torch.int32, device=A.device)
        _check(self._lib, self._lib.sfft_solve(
            self._p, _dev_ptr(A, torch.float64, self.N * self.N, "A"),
            _dev_ptr(b, torch.float64, self.N, "b"), _dev_ptr(coeffs, torch.float64, self.N, "coeffs"),
            _dev_ptr(info, torch.int32, 1, "info"), _stream_handle(stream)), "sfft_solve")
        return coeffs, info

    def subtract(self, R, S, coeffs, D=None, stream=None):
        import torch
        P = self.H * self.W
        if D is None:
            D = torch.empty((self.H, self.W), dtype=torch.float64, device=R.device)
        _check(self._lib, self._lib.sfft_subtract(
            self._p, _dev_ptr(R, torch.float64, P, "R"), _dev_ptr(S, torch.float64, P, "S"),
            _dev_ptr(coeffs, torch.float64, self.N, "coeffs"), _dev_ptr(D, torch.float64, P, "D"),
            _stream_handle(stream)), "sfft_subtract")
        return D

    def subtract_prepare(self, R, stream=None):
        """sfft_subtract_prepare: start the coefficient-independent stage of the next subtract(R, ...)
        on the plan's side stream (overlaps the solve).  R must stay ALIVE and unmodified until that
        subtract has been enqueued: the side stream is not known to torch's caching allocator, so a
        dropped R could be handed out again while the side stream still reads it."""
        import torch
        _check(self._lib, self._lib.sfft_subtract_prepare(
            self._p, _dev_ptr(R, torch.float64, self.H * self.W, "R"), _stream_handle(stream)), "sfft_subtract_prepare")

    def multi_template_difference(self, Rs, S, mask, scales, stream=None, helpers=()):
        """sfft_multi_template_difference: S against every template of Rs with one
        common mask, then the median of the scaled differences.  Returns (out, Dk, coeffs, info) with
        Dk [n, H, W], coeffs [n, N], info [n].  helpers: further SfftPlan objects of the same
        configuration; template k then runs on plan k % (1 + len(helpers))
        (sfft_multi_template_difference_plans), bitwise the same results."""
        import torch
        n, P = len(Rs), self.H * self.W
        dev = S.device
        ptrs = (ctypes.c_void_p * n)(*[_dev_ptr(R, torch.float64, P, f"Rs[{k}]").value for k, R in enumerate(Rs)])
        sc = (ctypes.c_double * n)(*[float(x) for x in scales])
        Dk = torch.empty((n, self.H, self.W), dtype=torch.float64, device=dev)
        coeffs = torch.empty((n, self.N), dtype=torch.float64, device=dev)
        info = torch.zeros(n, dtype=torch.int32, device=dev)
        out = torch.empty((self.H, self.W), dtype=torch.float64, device=dev)
        plans = [self, *helpers]
        pl = (ctypes.c_void_p * len(plans))(*[q._p for q in plans])
        _check(self._lib, self._lib.sfft_multi_template_difference_plans(
            pl, len(plans), ptrs, _dev_ptr(S, torch.float64, P, "S"), _dev_ptr(mask, torch.uint8, P, "mask"), sc, n,
            _dev_ptr(Dk, torch.float64, n * P, "Dk"), _dev_ptr(coeffs, torch.float64, n * self.N, "coeffs"),
            _dev_ptr(info, torch.int32, n, "info"), _dev_ptr(out, torch.float64, P, "out"),
            _stream_handle(stream)), "sfft_multi_template_difference_plans")
        return out, Dk, coeffs, info

    def difference(self, R, S, mask, stream=None):
        """One pass of the whole hot path: build -> (subtract_prepare) -> solve -> subtract."""
        A, b = self.build_system(R, S, mask, stream=stream)
        self.subtract_prepare(R, stream=stream)
        c, info = self.solve(A, b, stream=stream)
        D = self.subtract(R, S, c, stream=stream)
        return A, b, c, info, D

    def difference_host_async(self, R_host, S_host, mask_host, stream=None, D_host=None, c_host=None):
        """End-to-end call with HOST buffers: H2D copies of R, S, mask, the hot path (build -> solve ->
        subtract) and D2H copies of D, the coefficients and `info`, ALL enqueued on one stream (default:
        the current one); nothing synchronises.  Returns (D_host, c_host, info_host, done) with `done` a
        CUDA event recorded after the last copy: the host tensors are valid once it has completed.
        Pinned host tensors make the copies asynchronous; the plan keeps its device staging buffers and,
        unless D_host / c_host are given, its pinned result buffers between calls (so a second call on
        the same plan overwrites the first call's results).  Copies and marshalling only."""
        import torch
        st = torch.cuda.current_stream() if stream is None else stream
        dev = torch.device("cuda", torch.cuda.current_device())
        sg = getattr(self, "_stage", None)
        if sg is None:
            sg = dict(
                R=torch.empty((self.H, self.W), dtype=torch.float64, device=dev),
                S=torch.empty((self.H, self.W), dtype=torch.float64, device=dev),
                M=torch.empty((self.H, self.W), dtype=torch.uint8, device=dev),
                A=torch.empty((self.N, self.N), dtype=torch.float64, device=dev),
                b=torch.empty(self.N, dtype=torch.float64, device=dev),
                c=torch.empty(self.N, dtype=torch.float64, device=dev),
                info=torch.zeros(1, dtype=torch.int32, device=dev),
                D=torch.empty((self.H, self.W), dtype=torch.float64, device=dev),
                Dh=torch.empty((self.H, self.W), dtype=torch.float64).pin_memory(),
                ch=torch.empty(self.N, dtype=torch.float64).pin_memory(),
                ih=torch.zeros(1, dtype=torch.int32).pin_memory())
            self._stage = sg
        Dh = sg["Dh"] if D_host is None else D_host
        ch = sg["ch"] if c_host is None else c_host
        with torch.cuda.stream(st):
            sg["R"].copy_(R_host.reshape(self.H, self.W), non_blocking=True)
            sg["S"].copy_(S_host.reshape(self.H, self.W), non_blocking=True)
            M = None
            if mask_host is not None:
                sg["M"].copy_(mask_host.reshape(self.H, self.W), non_blocking=True)
                M = sg["M"]
            self.build_system(sg["R"], sg["S"], M, sg["A"], sg["b"], stream=st)
            self.solve(sg["A"], sg["b"], sg["c"], sg["info"], stream=st)
            self.subtract(sg["R"], sg["S"], sg["c"], sg["D"], stream=st)
            Dh.copy_(sg["D"], non_blocking=True)
            ch.copy_(sg["c"], non_blocking=True)
            sg["ih"].copy_(sg["info"], non_blocking=True)
            done = torch.cuda.Event()
            done.record(st)
        return Dh, ch, sg["ih"], done

    def difference_host(self, R_host, S_host, mask_host, stream=None):
        """difference_host_async, then wait for its event: (D, coeffs, info) as host tensors."""
        Dh, ch, ih, done = self.difference_host_async(R_host, S_host, mask_host, stream=stream)
        done.synchronize()
        return Dh, ch, ih

    @staticmethod
    def host_bytes_per_call(H, W, N, with_mask=True):
        """(h2d, d2h) bytes difference_host moves per call, counted from the tensors it copies."""
        return 2 * H * W * 8 + (H * W if with_mask else 0), H * W * 8 + N * 8 + 4

    # -- diagnostics
    def last_launch_count(self, which: int) -> int:
        return int(self._lib.sfft_last_launch_count(self._p, which))

    def set_solve_ctas(self, max_ctas: int) -> None:
        """sfft_plan_set_solve_ctas: cap the Cholesky kernel's grid (0 = one CTA per SM)."""
        _check(self._lib, self._lib.sfft_plan_set_solve_ctas(self._p, int(max_ctas)), "sfft_plan_set_solve_ctas")

    @property
    def fused(self) -> bool:
        """True if the plan runs the fused column-FFT + cross-spectra kernel (sfft_plan_fused)."""
        return int(self._lib.sfft_plan_fused(self._p)) == 1

    def profile_enable(self, on: bool = True):
        _check(self._lib, self._lib.sfft_profile_enable(self._p, 1 if on else 0), "sfft_profile_enable")

    def profile_read(self, reset: bool = True):
        """{stage name: (total_ms, count)} accumulated since the last reset (synchronises)."""
        out = {}
        for i, name in enumerate(STAGE_NAMES):
            ms, cnt = ctypes.c_double(0), ctypes.c_int(0)
            _check(self._lib, self._lib.sfft_profile_read(self._p, i, ctypes.byref(ms), ctypes.byref(cnt),
                                                          1 if reset else 0), "sfft_profile_read")
            out[name] = (ms.value, cnt.value)
        return out


def solve_static(A, b, coeffs=None, info=None, stream=None):
    """sfft_solve_static: A c = b without a plan and without any device allocation inside the library (the
    workspace is a static array shared by every call on the device: calls that overlap on the GPU race).
    N = len(b) <= SOLVE_STATIC_MAX_N.  The output tensors created here when coeffs / info are None are the
    caller-side allocations; pass preallocated ones from code that must not allocate at all."""
    import torch
    lib = load_library()
    N = int(b.numel())
    if coeffs is None:
        coeffs = torch.empty(N, dtype=torch.float64, device=A.device)
    if info is None:
        info = torch.zeros(1, dtype=torch.int32, device=A.device)
    _check(lib, lib.sfft_solve_static(
        _dev_ptr(A, torch.float64, N * N, "A"), _dev_ptr(b, torch.float64, N, "b"), N,
        _dev_ptr(coeffs, torch.float64, N, "coeffs"), _dev_ptr(info, torch.int32, 1, "info"),
        _stream_handle(stream)), "sfft_solve_static")
    return coeffs, info


def probe_fp64(kind: int = 0, iters: int = 4096, stream=None):
    """Measured fp64 peak (TFLOP/s) of the DFMA (kind 0) or DMMA (kind 1) pipe."""
    lib = load_library()
    tf, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(lib, lib.sfft_probe_fp64(kind, iters, ctypes.byref(tf), ctypes.byref(ms),
                                    _stream_handle(stream)), "sfft_probe_fp64")
    return tf.value, ms.value


def median_combine(Ds, scales, out=None, stream=None):
    """sfft_median_combine: out = median_k(scales[k] * Ds[k]) per pixel.  Ds: CUDA
    float64 tensors of one shape.  Argument marshalling only."""
    import torch
    lib = load_library()
    n = len(Ds)
    assert n == len(scales) and n >= 1
    for D in Ds:
        assert D.is_cuda and D.dtype == torch.float64 and D.is_contiguous() and D.shape == Ds[0].shape
    if out is None:
        out = torch.empty_like(Ds[0])
    ptrs = (ctypes.c_void_p * n)(*[D.data_ptr() for D in Ds])
    sc = (ctypes.c_double * n)(*[float(s) for s in scales])
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib, lib.sfft_median_combine(ptrs, sc, n, Ds[0].numel(), out.data_ptr(), st.cuda_stream), "sfft_median_combine")
    return out


def aperture_stats(D, mask, xs, ys, radius, stream=None):
    """sfft_aperture_stats: fluxes at the given positions and (count, mean, sigma) of the kept ones
    (PAPER.md:164).  D: CUDA float64 [H,W]; mask: CUDA uint8 or None; xs, ys: CUDA float64 [n]."""
    import torch
    lib = load_library()
    H, W = D.shape
    n = xs.numel()
    assert D.is_cuda and D.dtype == torch.float64 and D.is_contiguous()
    assert xs.is_cuda and ys.is_cuda and xs.dtype == torch.float64 and ys.dtype == torch.float64 and ys.numel() == n
    flux = torch.empty(n, dtype=torch.float64, device=D.device)
    stats = torch.empty(3, dtype=torch.float64, device=D.device)
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib, lib.sfft_aperture_stats(D.data_ptr(), 0 if mask is None else mask.data_ptr(), H, W, xs.data_ptr(),
                                        ys.data_ptr(), n, float(radius), flux.data_ptr(), stats.data_ptr(),
                                        st.cuda_stream), "sfft_aperture_stats")
    return flux, stats


def cut_stamps(S, R, D, xs, ys, size, stream=None):
    """sfft_cut_stamps: [n, 3, size, size] (science, template, difference) stamps centred on the
    positions.  S, R, D: CUDA float64 [H, W]; xs, ys: CUDA float64 [n]."""
    import torch
    lib = load_library()
    H, W = S.shape
    n = xs.numel()
    out = torch.empty((n, 3, size, size), dtype=torch.float64, device=S.device)
    _check(lib, lib.sfft_cut_stamps(_dev_ptr(S, torch.float64, H * W, "S"), _dev_ptr(R, torch.float64, H * W, "R"),
                                    _dev_ptr(D, torch.float64, H * W, "D"), H, W, _dev_ptr(xs, torch.float64, n, "xs"),
                                    _dev_ptr(ys, torch.float64, n, "ys"), n, int(size),
                                    _dev_ptr(out, torch.float64, out.numel(), "out"), _stream_handle(stream)),
           "sfft_cut_stamps")
    return out


def resample_affine(img, M, Hout, Wout, a=3, out=None, outside=None, stream=None):
    """sfft_resample_affine: (out, outside) of a CUDA float64 image through the affine map M (6 floats)."""
    import torch
    lib = load_library()
    assert img.is_cuda and img.dtype == torch.float64 and img.is_contiguous() and img.dim() == 2
    if out is None:
        out = torch.empty((Hout, Wout), dtype=torch.float64, device=img.device)
    if outside is None:
        outside = torch.empty((Hout, Wout), dtype=torch.uint8, device=img.device)
    assert out.shape == (Hout, Wout) and out.dtype == torch.float64 and out.is_contiguous()
    assert outside.shape == (Hout, Wout) and outside.dtype == torch.uint8 and outside.is_contiguous()
    Mc = (ctypes.c_double * 6)(*[float(v) for v in M])
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib, lib.sfft_resample_affine(img.data_ptr(), img.shape[0], img.shape[1], Mc, int(a), out.data_ptr(),
                                         Hout, Wout, outside.data_ptr(), st.cuda_stream), "sfft_resample_affine")
    return out, outside


def resample_mask_affine(mask, M, Hout, Wout, a=3, threshold=0.3, stream=None):
    """sfft_resample_mask_affine: resampled data-quality mask, 2 = bad, 1 = good."""
    import torch
    lib = load_library()
    assert mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous() and mask.dim() == 2
    out = torch.empty((Hout, Wout), dtype=torch.uint8, device=mask.device)
    Mc = (ctypes.c_double * 6)(*[float(v) for v in M])
    st = torch.cuda.current_stream() if stream is None else stream
    _check(lib, lib.sfft_resample_mask_affine(mask.data_ptr(), mask.shape[0], mask.shape[1], Mc, int(a),
                                              float(threshold), out.data_ptr(), Hout, Wout, st.cuda_stream),
           "sfft_resample_mask_affine")
    return out
