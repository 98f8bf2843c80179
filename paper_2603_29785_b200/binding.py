"""ctypes binding of libqtam.so (include/qtam.h).  Argument marshalling only: every step of the
transform runs in the CUDA kernels.  PyTorch is used for device memory and streams.

There is no CPU fallback: if the library is missing it is built (nvcc), and if no CUDA device is
present the compute calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libqtam.so")
_lib = None

QTAM_F32, QTAM_F64 = 0, 1
STATUS = {0: "ok", 1: "invalid argument", 2: "unsupported", 3: "alloc", 4: "cuda", 5: "empty frame", 6: "too large"}
CLUSTER_NOALLOC_MAX_PIXELS = 1 << 20      # QTAM_CLUSTER_NOALLOC_MAX_PIXELS of include/qtam.h

SYMBOLS = ["qtam_plan_create", "qtam_plan_create_host", "qtam_plan_destroy", "qtam_plan_info",
           "qtam_plan_rows", "qtam_plan_window", "qtam_plan_frame", "qtam_forward", "qtam_inverse",
           "qtam_dense", "qtam_dense_invert", "qtam_threshold_rowmedian", "qtam_forward_threshold", "qtam_plane_metric", "qtam_gather_plane", "qtam_max_plane_coeffs", "qtam_remodulate", "qtam_instantaneous_frequency", "qtam_last_launch_count", "qtam_status_string",
           "qtam_profile_enable", "qtam_profile_read", "qtam_output_length", "qtam_forward_length", "qtam_inverse_length",
           "qtam_resample", "qtam_plane_pixels", "qtam_cluster", "qtam_mask", "qtam_cluster_noalloc"]


class QtamError(RuntimeError):
    def __init__(self, code, where):
        super().__init__(f"{where}: status {code} ({STATUS.get(code, '?')})")
        self.code = code


class Options(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("window", C.c_int), ("clamp_mode", C.c_int),
                ("clamp_overlap", C.c_double), ("max_window_bins", C.c_int64),
                ("cover_floor", C.c_double), ("rows_are_bins_per_octave", C.c_int),
                ("max_batch", C.c_int), ("window_param", C.c_double),
                ("freqs", C.POINTER(C.c_double)), ("n_freqs", C.c_int), ("tile_length", C.c_int64), ("epsilon", C.c_double),
                ("plane_window", C.POINTER(C.c_int)), ("plane_window_param", C.POINTER(C.c_double)),
                ("out_length", C.c_int64)]


WINDOWS = {"bisquare": 0, "hann": 1, "kaiser": 2, "tukey": 3, "planck": 4}


class Row(C.Structure):
    _fields_ = [("plane", C.c_int), ("row", C.c_int), ("q", C.c_double), ("f_request", C.c_double),
                ("f_center", C.c_double), ("kc", C.c_int64), ("dk", C.c_int64), ("L", C.c_int64),
                ("M", C.c_int64), ("offset", C.c_int64), ("norm", C.c_double)]


class Info(C.Structure):
    _fields_ = [("n_planes", C.c_int), ("n_rows", C.c_int), ("n", C.c_int64), ("n_bins", C.c_int64),
                ("coeffs_per_segment", C.c_int64), ("sum_L", C.c_int64), ("cover_lo", C.c_int64),
                ("cover_hi", C.c_int64), ("holes", C.c_int64), ("frame_A", C.c_double),
                ("frame_B", C.c_double), ("workspace_bytes", C.c_size_t)]


class KernelStat(C.Structure):
    _fields_ = [("name", C.c_char * 48), ("launches", C.c_int), ("ms", C.c_double),
                ("algo_bytes", C.c_double), ("design_bytes", C.c_double)]


def lib():
    """Loads libqtam.so (building it in-tree first if it is missing)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            from . import build as _b
            _b.build()
        L = C.CDLL(_LIBPATH)
        vp, dp = C.c_void_p, C.POINTER(C.c_double)
        create_args = [C.POINTER(vp), C.c_double, C.c_int64, dp, C.c_int, C.c_double, C.c_double,
                       C.c_double, C.c_int, C.POINTER(Options)]
        L.qtam_plan_create.argtypes = create_args
        L.qtam_plan_create_host.argtypes = create_args
        L.qtam_plan_destroy.argtypes = [vp]
        L.qtam_plan_info.argtypes = [vp, C.POINTER(Info)]
        L.qtam_plan_rows.argtypes = [vp, C.POINTER(Row), C.c_int]
        L.qtam_plan_window.argtypes = [vp, C.c_int, dp]
        L.qtam_plan_frame.argtypes = [vp, C.c_int, dp, C.POINTER(C.c_uint8)]
        L.qtam_forward.argtypes = [vp, vp, C.c_int, vp, vp]
        L.qtam_inverse.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.qtam_dense.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp]
        L.qtam_threshold_rowmedian.argtypes = [vp, vp, C.c_int, C.c_double, vp]
        L.qtam_forward_threshold.argtypes = [vp, vp, C.c_int, C.c_double, vp, vp]
        L.qtam_plane_metric.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp, vp]
        L.qtam_remodulate.argtypes = [vp, vp, C.c_int, vp, vp]
        L.qtam_dense_invert.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.qtam_gather_plane.argtypes = [vp, vp, C.c_int, vp, vp, vp]
        L.qtam_max_plane_coeffs.argtypes = [vp]
        L.qtam_max_plane_coeffs.restype = C.c_int64
        L.qtam_instantaneous_frequency.argtypes = [vp, vp, C.c_int, vp, vp]
        L.qtam_last_launch_count.argtypes = [vp]
        L.qtam_last_launch_count.restype = C.c_int
        L.qtam_status_string.argtypes = [C.c_int]
        L.qtam_status_string.restype = C.c_char_p
        L.qtam_profile_enable.argtypes = [vp, C.c_int, C.c_int]
        L.qtam_profile_read.argtypes = [vp, C.POINTER(KernelStat), C.c_int]
        L.qtam_profile_read.restype = C.c_int
        L.qtam_output_length.argtypes = [vp, C.c_int]
        L.qtam_output_length.restype = C.c_int64
        L.qtam_forward_length.argtypes = [vp, vp, C.c_int, vp, vp]
        L.qtam_inverse_length.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.qtam_resample.argtypes = [vp, vp, C.c_int, C.c_int, vp, vp]
        L.qtam_plane_pixels.argtypes = [vp, C.c_int]
        L.qtam_plane_pixels.restype = C.c_int64
        L.qtam_cluster.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp, vp]
        L.qtam_mask.argtypes = [vp, vp, C.c_int, C.c_int, vp, C.c_int, vp, vp]
        L.qtam_cluster_noalloc.argtypes = [C.c_int, vp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp, vp]
        _lib = L
    return _lib


def _check(code, where):
    if code != 0:
        raise QtamError(code, where)


def cluster_noalloc(img, segment_stride, batch, rows, samples, min_area, labels, count):
    """qtam_cluster_noalloc: the labelling of Plan.cluster for a caller that may not allocate device memory (no plan,
    no cudaMalloc inside the library: its one piece of scratch is a fixed 4 MiB array inside libqtam.so, shared by all
    calls on a GPU, so keep them on one stream).  Every tensor is the caller's, this wrapper creates none: `img` a
    CUDA complex64 / complex128 tensor (or a view starting at a plane's first coefficient), segment b at
    img.data_ptr() + b * segment_stride elements; `labels` int32 with batch * rows * samples elements and `count`
    int32 with batch elements are overwritten.  batch * rows * samples <= CLUSTER_NOALLOC_MAX_PIXELS, else QtamError
    with code 6 ('too large').  Runs on torch's current stream; make the first call per device at start-up."""
    import torch
    if not (img.is_cuda and labels.is_cuda and count.is_cuda):
        raise ValueError("qtam_cluster_noalloc: img, labels and count must be CUDA tensors")
    if img.dtype not in (torch.complex64, torch.complex128):
        raise ValueError(f"img: dtype {img.dtype}, expected complex64 or complex128")
    if labels.dtype != torch.int32 or count.dtype != torch.int32 or not labels.is_contiguous() or not count.is_contiguous():
        raise ValueError("labels and count must be contiguous int32 tensors")
    batch, rows, samples = int(batch), int(rows), int(samples)
    if batch < 0 or rows < 1 or samples < 1:
        raise ValueError("batch >= 0, rows >= 1 and samples >= 1 expected")
    if labels.numel() != batch * rows * samples or count.numel() != batch:
        raise ValueError("labels needs batch * rows * samples elements and count needs batch")
    if batch > 0 and img.storage_offset() + (batch - 1) * int(segment_stride) + rows * samples > img.untyped_storage().nbytes() // img.element_size():
        raise ValueError("img: the last segment's image ends beyond the tensor's storage")
    _check(lib().qtam_cluster_noalloc(QTAM_F32 if img.dtype == torch.complex64 else QTAM_F64, img.data_ptr(),
                                      int(segment_stride), batch, rows, samples, int(min_area), labels.data_ptr(),
                                      count.data_ptr(), C.c_void_p(torch.cuda.current_stream().cuda_stream)),
           "qtam_cluster_noalloc")
    return labels, count


class Plan:
    """qtam_plan_create(fs, N, Q list, fmin, fmax, row spacing, dtype, options)."""

    def __init__(self, fs, N, Q, fmin, fmax, spacing, dtype="f32", max_batch=1, clamp_mode=1,
                 clamp_overlap=1.0, max_window_bins=0, cover_floor=1e-2, rows_are_bins_per_octave=0,
                 host_only=False, window="bisquare", window_param=0.0, freqs=None, tile_length=0, epsilon=0.0,
                 out_length=0, plane_windows=None):
        L = lib()
        self._h = C.c_void_p()
        self.dtype = dtype
        q = np.ascontiguousarray(Q, dtype=np.float64)
        fr = None if freqs is None else np.ascontiguousarray(freqs, dtype=np.float64)
        pw = pp = None
        if plane_windows is not None:       # [(family, parameter)] per plane: a composite filter bank
            if len(plane_windows) != q.size:
                raise ValueError("plane_windows: one (family, parameter) per entry of Q")
            pw = np.ascontiguousarray([WINDOWS[w] for w, _ in plane_windows], dtype=np.int32)
            pp = np.ascontiguousarray([float(a) for _, a in plane_windows], dtype=np.float64)
        opt = Options(C.sizeof(Options), WINDOWS[window], clamp_mode, clamp_overlap, max_window_bins,
                      cover_floor, rows_are_bins_per_octave, max_batch, float(window_param),
                      None if fr is None else fr.ctypes.data_as(C.POINTER(C.c_double)),
                      0 if fr is None else fr.size, int(tile_length), float(epsilon),
                      None if pw is None else pw.ctypes.data_as(C.POINTER(C.c_int)),
                      None if pp is None else pp.ctypes.data_as(C.POINTER(C.c_double)),
                      {"standard": -1, "minimal": -2}.get(out_length, out_length))
        fn = L.qtam_plan_create_host if host_only else L.qtam_plan_create
        code = fn(C.byref(self._h), float(fs), int(N), q.ctypes.data_as(C.POINTER(C.c_double)), q.size,
                  float(fmin), float(fmax), float(spacing), QTAM_F64 if dtype == "f64" else QTAM_F32,
                  C.byref(opt))
        if code != 0:
            self._h = None
            raise QtamError(code, "qtam_plan_create")
        self.max_batch = max_batch
        info = Info()
        _check(L.qtam_plan_info(self._h, C.byref(info)), "qtam_plan_info")
        self.info = info
        self.N, self.n_bins = int(info.n), int(info.n_bins)
        self.n_rows, self.n_planes = int(info.n_rows), int(info.n_planes)
        self.ctot = int(info.coeffs_per_segment)
        rows = (Row * self.n_rows)()
        _check(L.qtam_plan_rows(self._h, rows, self.n_rows), "qtam_plan_rows")
        self.rows = list(rows)

    def close(self):
        if getattr(self, "_h", None):
            lib().qtam_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: the module globals may already be gone
            pass

    # ---- host tables -------------------------------------------------------------------------------
    def window(self, k):
        out = np.empty(int(self.rows[k].L), dtype=np.float64)
        _check(lib().qtam_plan_window(self._h, k, out.ctypes.data_as(C.POINTER(C.c_double))), "qtam_plan_window")
        return out

    def frame(self, plane=-1):
        P = np.empty(self.n_bins, dtype=np.float64)
        cov = np.empty(self.n_bins, dtype=np.uint8)
        _check(lib().qtam_plan_frame(self._h, plane, P.ctypes.data_as(C.POINTER(C.c_double)),
                                     cov.ctypes.data_as(C.POINTER(C.c_uint8))), "qtam_plan_frame")
        return P, cov.astype(bool)

    def row_slice(self, k):
        r = self.rows[k]
        return slice(int(r.offset), int(r.offset + r.M))

    # ---- device calls (torch tensors on the GPU; stream = torch's current stream) -----------------
    def _torch(self):
        import torch
        return torch

    def _rdt(self):
        t = self._torch()
        return t.float64 if self.dtype == "f64" else t.float32

    def _cdt(self):
        t = self._torch()
        return t.complex128 if self.dtype == "f64" else t.complex64

    def _stream(self):
        return C.c_void_p(self._torch().cuda.current_stream().cuda_stream)

    # argument checks: explicit errors (an `assert` disappears under python -O, and a mis-sized tensor would
    # become an out-of-bounds device write inside the library)
    def _need(self, t, dtype, what, numel=None, last=None):
        if not (hasattr(t, "is_cuda") and t.is_cuda):
            raise ValueError(f"{what}: expected a CUDA tensor")
        if t.dtype != dtype:
            raise ValueError(f"{what}: dtype {t.dtype}, expected {dtype}")
        if not t.is_contiguous():
            raise ValueError(f"{what}: must be contiguous")
        if last is not None and (t.dim() < 1 or t.shape[-1] != last):
            raise ValueError(f"{what}: last dimension {tuple(t.shape)}, expected {last}")
        if numel is not None and t.numel() != numel:
            raise ValueError(f"{what}: {t.numel()} elements, expected {numel}")

    def _batch(self, t, per_segment, what):
        if per_segment <= 0 or t.numel() % per_segment != 0:
            raise ValueError(f"{what}: {t.numel()} elements is not a multiple of {per_segment}")
        b = t.numel() // per_segment
        if b > self.max_batch:
            raise QtamError(1, f"{what}: batch {b} exceeds the plan's max_batch {self.max_batch}")
        return b

    def forward(self, x, out=None):
        t = self._torch()
        self._need(x, self._rdt(), "x", last=self.N)
        batch = self._batch(x, self.N, "x")
        if out is None:
            out = t.empty((batch, self.ctot), dtype=self._cdt(), device=x.device)
        self._need(out, self._cdt(), "out", numel=batch * self.ctot)
        _check(lib().qtam_forward(self._h, x.data_ptr(), batch, out.data_ptr(), self._stream()), "qtam_forward")
        return out

    def inverse(self, coef, plane=-1, out=None):
        t = self._torch()
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        if out is None:
            out = t.empty((batch, self.N), dtype=self._rdt(), device=coef.device)
        self._need(out, self._rdt(), "out", numel=batch * self.N)
        _check(lib().qtam_inverse(self._h, coef.data_ptr(), batch, plane, out.data_ptr(), self._stream()), "qtam_inverse")
        return out

    def dense(self, x, row_begin=0, row_end=None, out=None):
        t = self._torch()
        row_end = self.n_rows if row_end is None else row_end
        if not (0 <= row_begin <= row_end <= self.n_rows):
            raise ValueError(f"row range [{row_begin}, {row_end}) outside [0, {self.n_rows})")
        self._need(x, self._rdt(), "x", last=self.N)
        batch = self._batch(x, self.N, "x")
        if out is None:
            out = t.empty((batch, row_end - row_begin, self.N), dtype=self._cdt(), device=x.device)
        self._need(out, self._cdt(), "out", numel=batch * (row_end - row_begin) * self.N)
        _check(lib().qtam_dense(self._h, x.data_ptr(), batch, row_begin, row_end, out.data_ptr(), self._stream()), "qtam_dense")
        return out

    def forward_threshold(self, x, kappa=3.0, out=None):
        """forward + row-median threshold in one call (fused for float plans)"""
        t = self._torch()
        self._need(x, self._rdt(), "x", last=self.N)
        batch = self._batch(x, self.N, "x")
        if out is None:
            out = t.empty((batch, self.ctot), dtype=self._cdt(), device=x.device)
        self._need(out, self._cdt(), "out", numel=batch * self.ctot)
        _check(lib().qtam_forward_threshold(self._h, x.data_ptr(), batch, float(kappa), out.data_ptr(), self._stream()),
               "qtam_forward_threshold")
        return out

    def dense_invert(self, tile, row):
        """x[batch][N] from one dense tile per segment (Eq. 13); the plan needs epsilon > 0"""
        t = self._torch()
        self._need(tile, self._cdt(), "tile", last=self.N)
        batch = self._batch(tile, self.N, "tile")
        out = t.empty((batch, self.N), dtype=self._rdt(), device=tile.device)
        _check(lib().qtam_dense_invert(self._h, tile.data_ptr(), batch, int(row), out.data_ptr(), self._stream()),
               "qtam_dense_invert")
        return out

    def output_length(self, mode=0):
        """the plan's uniform output length (mode 0), the 'standard' N/2 + 1 (-1) or the 'minimal' one (-2)"""
        return int(lib().qtam_output_length(self._h, {"standard": -1, "minimal": -2}.get(mode, mode)))

    def forward_length(self, x):
        """[batch][rows][n] image at the plan's uniform output length (the paper's output-resolution option)"""
        t = self._torch()
        n = self.output_length()
        if n <= 0:
            raise ValueError("the plan was created without out_length")
        self._need(x, self._rdt(), "x", last=self.N)
        batch = self._batch(x, self.N, "x")
        out = t.empty((batch, self.n_rows, n), dtype=self._cdt(), device=x.device)
        _check(lib().qtam_forward_length(self._h, x.data_ptr(), batch, out.data_ptr(), self._stream()), "qtam_forward_length")
        return out

    def inverse_length(self, img, plane=-1):
        t = self._torch()
        n = self.output_length()
        if n <= 0:
            raise ValueError("the plan was created without out_length")
        self._need(img, self._cdt(), "img", last=n)
        batch = self._batch(img, self.n_rows * n, "img")
        out = t.empty((batch, self.N), dtype=self._rdt(), device=img.device)
        _check(lib().qtam_inverse_length(self._h, img.data_ptr(), batch, plane, out.data_ptr(), self._stream()),
               "qtam_inverse_length")
        return out

    def resample(self, img, to_standard=True):
        """between the plan's length and the standard N/2 + 1 (Fig. 3 of the paper); exact for band-limited rows"""
        t = self._torch()
        n, ns = self.output_length(), self.output_length(-1)
        n_in, n_out = (n, ns) if to_standard else (ns, n)
        if n <= 0:
            raise ValueError("the plan was created without out_length")
        self._need(img, self._cdt(), "img", last=n_in)
        batch = self._batch(img, self.n_rows * n_in, "img")
        out = t.empty((batch, self.n_rows, n_out), dtype=self._cdt(), device=img.device)
        _check(lib().qtam_resample(self._h, img.data_ptr(), batch, 1 if to_standard else 0, out.data_ptr(), self._stream()),
               "qtam_resample")
        return out

    def cluster(self, coef, plane, min_area=1):
        """(labels[batch][R*M] int32, count[batch] int32): connected clusters of the non-zero coefficients of one
        Q-plane (uniform-tile layout; threshold first), PAPER.md:208"""
        t = self._torch()
        npx = int(lib().qtam_plane_pixels(self._h, int(plane)))
        if npx <= 0:
            raise ValueError("qtam_cluster needs a plan in the uniform-tile layout (tile_length != 0)")
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        labels = t.empty((batch, npx), dtype=t.int32, device=coef.device)
        count = t.empty((batch,), dtype=t.int32, device=coef.device)
        _check(lib().qtam_cluster(self._h, coef.data_ptr(), batch, int(plane), int(min_area), labels.data_ptr(),
                                  count.data_ptr(), self._stream()), "qtam_cluster")
        return labels, count

    def mask(self, coef, plane, labels, label=0, out=None):
        """the binary mask of one cluster (label > 0) or of all kept clusters (0) applied to the coefficients"""
        t = self._torch()
        npx = int(lib().qtam_plane_pixels(self._h, int(plane)))
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        self._need(labels, t.int32, "labels", numel=batch * npx)
        if out is None:
            out = t.empty_like(coef)
        self._need(out, self._cdt(), "out", numel=batch * self.ctot)
        _check(lib().qtam_mask(self._h, coef.data_ptr(), batch, int(plane), labels.data_ptr(), int(label), out.data_ptr(),
                               self._stream()), "qtam_mask")
        return out

    def threshold_rowmedian(self, coef, kappa=3.0):
        """in place"""
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        _check(lib().qtam_threshold_rowmedian(self._h, coef.data_ptr(), batch, float(kappa), self._stream()),
               "qtam_threshold_rowmedian")
        return coef

    def remodulate(self, coef, out=None):
        """decimated envelopes -> samples of the dense tiles (Eq. 10a); out may be coef (in place)"""
        t = self._torch()
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        if out is None:
            out = t.empty_like(coef)
        self._need(out, self._cdt(), "out", numel=batch * self.ctot)
        _check(lib().qtam_remodulate(self._h, coef.data_ptr(), batch, out.data_ptr(), self._stream()), "qtam_remodulate")
        return out

    def instantaneous_frequency(self, coef):
        """[batch][ctot] real, Hz: circular forward difference of the unwrapped baseband phase plus the carrier"""
        t = self._torch()
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        out = t.empty((batch, self.ctot), dtype=self._rdt(), device=coef.device)
        _check(lib().qtam_instantaneous_frequency(self._h, coef.data_ptr(), batch, out.data_ptr(), self._stream()),
               "qtam_instantaneous_frequency")
        return out

    def gather_plane(self, coef, best):
        """[batch][max plane size]: plane best[b] of every segment, zero padded (optimal-selection mode)"""
        t = self._torch()
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        self._need(best, t.int32, "best", numel=batch)
        out = t.empty((batch, int(lib().qtam_max_plane_coeffs(self._h))), dtype=self._cdt(), device=coef.device)
        _check(lib().qtam_gather_plane(self._h, coef.data_ptr(), batch, best.data_ptr(), out.data_ptr(), self._stream()),
               "qtam_gather_plane")
        return out

    def plane_metric(self, coef, metric="energy"):
        """(values[batch][n_planes], best[batch] int32) of the multi-Q scan's plane selection"""
        t = self._torch()
        self._need(coef, self._cdt(), "coef")
        batch = self._batch(coef, self.ctot, "coef")
        if metric not in ("energy", "peak"):
            raise ValueError(f"metric {metric!r}: expected 'energy' or 'peak'")
        vals = t.empty((batch, self.n_planes), dtype=self._rdt(), device=coef.device)
        best = t.empty((batch,), dtype=t.int32, device=coef.device)
        _check(lib().qtam_plane_metric(self._h, coef.data_ptr(), batch, {"energy": 0, "peak": 1}[metric],
                                       vals.data_ptr(), best.data_ptr(), self._stream()), "qtam_plane_metric")
        return vals, best

    def last_launch_count(self):
        return int(lib().qtam_last_launch_count(self._h))

    def profile_enable(self, on=True, max_launches=4096):
        _check(lib().qtam_profile_enable(self._h, 1 if on else 0, max_launches), "qtam_profile_enable")

    def profile_read(self):
        """[{name, launches, ms, algo_bytes, design_bytes}] since the last read (waits for the recorded events)"""
        buf = (KernelStat * 32)()
        n = lib().qtam_profile_read(self._h, buf, 32)
        if n < 0:
            raise QtamError(4, "qtam_profile_read")
        return [dict(name=buf[i].name.decode(), launches=int(buf[i].launches), ms=float(buf[i].ms),
                     algo_bytes=float(buf[i].algo_bytes), design_bytes=float(buf[i].design_bytes)) for i in range(n)]

    # ---- host-buffer convenience (the end-to-end path bench.py times) ------------------------------
    def forward_host(self, x_pinned, coef_pinned, d_x, d_coef):
        """H2D copy of x, forward, D2H copy of the coefficients; all on the current stream."""
        d_x.copy_(x_pinned, non_blocking=True)
        self.forward(d_x, out=d_coef)
        coef_pinned.copy_(d_coef, non_blocking=True)
