"""ctypes binding of the CPU oracle (oracle/libqtam_ref.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  Argument marshalling only; all arithmetic is in qtam_ref.cpp.
"""
import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
if _HERE not in sys.path:
    sys.path.insert(0, _HERE)
import build as _build  # noqa: E402  (oracle/build.py)

_lib = None


class Options(C.Structure):
    _fields_ = [("window", C.c_int), ("clamp_mode", C.c_int), ("clamp_overlap", C.c_double),
                ("max_window_bins", C.c_int64), ("cover_floor", C.c_double),
                ("rows_are_bins_per_octave", C.c_int), ("window_param", C.c_double),
                ("freqs", C.POINTER(C.c_double)), ("n_freqs", C.c_int), ("tile_length", C.c_int64), ("epsilon", C.c_double),
                ("plane_window", C.POINTER(C.c_int)), ("plane_window_param", C.POINTER(C.c_double))]


WINDOWS = {"bisquare": 0, "hann": 1, "kaiser": 2, "tukey": 3, "planck": 4}


class Row(C.Structure):
    _fields_ = [("plane", C.c_int), ("row", C.c_int), ("q", C.c_double), ("f_request", C.c_double),
                ("f_center", C.c_double), ("kc", C.c_int64), ("dk", C.c_int64), ("L", C.c_int64),
                ("M", C.c_int64), ("offset", C.c_int64), ("norm", C.c_double)]


class Info(C.Structure):
    _fields_ = [("n_planes", C.c_int), ("n_rows", C.c_int), ("n", C.c_int64), ("n_bins", C.c_int64),
                ("coeffs_per_segment", C.c_int64), ("sum_L", C.c_int64), ("cover_lo", C.c_int64),
                ("cover_hi", C.c_int64), ("holes", C.c_int64), ("cover_count", C.c_int64),
                ("frame_A", C.c_double), ("frame_B", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        vp, dp, fp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_float)
        _lib.qtam_ref_plan_create.argtypes = [C.POINTER(vp), C.c_double, C.c_int64, dp, C.c_int,
                                              C.c_double, C.c_double, C.c_double, C.POINTER(Options)]
        _lib.qtam_ref_plan_destroy.argtypes = [vp]
        _lib.qtam_ref_plan_destroy.restype = None
        _lib.qtam_ref_plan_info.argtypes = [vp, C.POINTER(Info)]
        _lib.qtam_ref_plan_rows.argtypes = [vp, C.POINTER(Row), C.c_int]
        _lib.qtam_ref_plan_window.argtypes = [vp, C.c_int, dp]
        _lib.qtam_ref_plan_frame.argtypes = [vp, C.c_int, dp, C.POINTER(C.c_uint8)]
        _lib.qtam_ref_forward.argtypes = [vp, dp, C.c_int, dp, C.c_int]
        _lib.qtam_ref_inverse.argtypes = [vp, dp, C.c_int, C.c_int, dp, C.c_int]
        _lib.qtam_ref_dense.argtypes = [vp, dp, C.c_int, C.c_int, C.c_int, dp, C.c_int]
        _lib.qtam_ref_brute_tile.argtypes = [vp, dp, C.c_int, dp]
        _lib.qtam_ref_threshold_rowmedian.argtypes = [vp, dp, C.c_int, C.c_double]
        _lib.qtam_ref_threshold_rowmedian_f32.argtypes = [vp, fp, C.c_int, C.c_float]
        _lib.qtam_ref_remodulate.argtypes = [vp, dp, C.c_int, dp]
        _lib.qtam_ref_instantaneous_frequency.argtypes = [vp, dp, C.c_int, dp]
        _lib.qtam_ref_gather_plane.argtypes = [vp, dp, C.c_int, C.POINTER(C.c_int32), dp]
        _lib.qtam_ref_dense_invert.argtypes = [vp, dp, C.c_int, C.c_int, dp]
        _lib.qtam_ref_plane_metric.argtypes = [vp, dp, C.c_int, C.c_int, dp, C.POINTER(C.c_int32)]
        _lib.qtam_ref_project_cover.argtypes = [vp, dp, C.c_int, C.c_int, dp, C.c_int]
        _lib.qtam_ref_cluster_labels.argtypes = [C.POINTER(C.c_uint8), C.c_int, C.c_int, C.c_int64, C.c_int,
                                                 C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        _lib.qtam_ref_output_length.argtypes = [vp, C.c_int]
        _lib.qtam_ref_output_length.restype = C.c_int64
        _lib.qtam_ref_forward_length.argtypes = [vp, dp, C.c_int, C.c_int64, dp, C.c_int]
        _lib.qtam_ref_inverse_length.argtypes = [vp, dp, C.c_int, C.c_int64, C.c_int, dp, C.c_int]
        _lib.qtam_ref_resample.argtypes = [vp, dp, C.c_int, C.c_int64, C.c_int64, dp]
        _lib.qtam_ref_spectrum.argtypes = [vp, dp, C.c_int, dp, C.c_int]
        _lib.qtam_ref_dft.argtypes = [dp, dp, C.c_int64, C.c_int]
        _lib.qtam_ref_fft.argtypes = [dp, dp, C.c_int64, C.c_int]
        _lib.qtam_ref_threads.restype = C.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _c2d(a):
    """complex128 array -> float64 view (interleaved)"""
    return np.ascontiguousarray(a, dtype=np.complex128).view(np.float64)


def threads():
    return int(lib().qtam_ref_threads())


def set_threads(n):
    lib().qtam_ref_set_threads(int(n))


def cluster_labels(mask, min_area=1):
    """connected components (4-connectivity, time circular) of a [batch][rows][M] mask; labels = 1 + smallest pixel
    index of the cluster, 0 for background and for clusters smaller than min_area"""
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    if m.ndim == 2:
        m = m[None]
    labels = np.zeros(m.shape, dtype=np.int32)
    count = np.zeros(m.shape[0], dtype=np.int32)
    assert lib().qtam_ref_cluster_labels(m.ctypes.data_as(C.POINTER(C.c_uint8)), m.shape[0], m.shape[1], m.shape[2],
                                         int(min_area), labels.ctypes.data_as(C.POINTER(C.c_int32)),
                                         count.ctypes.data_as(C.POINTER(C.c_int32))) == 0
    return labels, count


def dft(z, sign):
    z = np.ascontiguousarray(z, dtype=np.complex128)
    out = np.empty_like(z)
    assert lib().qtam_ref_dft(_dp(z.view(np.float64)), _dp(out.view(np.float64)), z.size, sign) == 0
    return out


def fft(z, sign):
    z = np.ascontiguousarray(z, dtype=np.complex128)
    out = np.empty_like(z)
    assert lib().qtam_ref_fft(_dp(z.view(np.float64)), _dp(out.view(np.float64)), z.size, sign) == 0
    return out


class RefPlan:
    """Oracle plan; same constructor arguments as the CUDA library's plan."""

    def __init__(self, fs, N, Q, fmin, fmax, spacing, clamp_mode=1, clamp_overlap=1.0,
                 max_window_bins=0, cover_floor=1e-2, rows_are_bins_per_octave=0,
                 window="bisquare", window_param=0.0, freqs=None, tile_length=0, epsilon=0.0, plane_windows=None):
        L = lib()
        self._h = C.c_void_p()
        q = np.ascontiguousarray(Q, dtype=np.float64)
        fr = None if freqs is None else np.ascontiguousarray(freqs, dtype=np.float64)
        pw = pp = None
        if plane_windows is not None:       # [(family, parameter)] per plane: a composite filter bank
            pw = np.ascontiguousarray([WINDOWS[w] for w, _ in plane_windows], dtype=np.int32)
            pp = np.ascontiguousarray([float(a) for _, a in plane_windows], dtype=np.float64)
            assert pw.size == len(Q)
        opt = Options(WINDOWS[window], clamp_mode, clamp_overlap, max_window_bins, cover_floor,
                      rows_are_bins_per_octave, float(window_param),
                      None if fr is None else fr.ctypes.data_as(C.POINTER(C.c_double)),
                      0 if fr is None else fr.size, int(tile_length), float(epsilon),
                      None if pw is None else pw.ctypes.data_as(C.POINTER(C.c_int)),
                      None if pp is None else pp.ctypes.data_as(C.POINTER(C.c_double)))
        rc = L.qtam_ref_plan_create(C.byref(self._h), float(fs), int(N), _dp(q), q.size,
                                    float(fmin), float(fmax), float(spacing), C.byref(opt))
        if rc != 0:
            self._h = None
            raise ValueError(f"qtam_ref_plan_create failed with code {rc}")
        info = Info()
        assert L.qtam_ref_plan_info(self._h, C.byref(info)) == 0
        self.info = info
        self.N = int(info.n)
        self.n_bins = int(info.n_bins)
        self.n_rows = int(info.n_rows)
        self.n_planes = int(info.n_planes)
        self.ctot = int(info.coeffs_per_segment)
        rows = (Row * self.n_rows)()
        assert L.qtam_ref_plan_rows(self._h, rows, self.n_rows) == 0
        self.rows = list(rows)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().qtam_ref_plan_destroy(self._h)
            self._h = None

    def window(self, k):
        out = np.empty(int(self.rows[k].L), dtype=np.float64)
        assert lib().qtam_ref_plan_window(self._h, k, _dp(out)) == 0
        return out

    def frame(self, plane=-1):
        P = np.empty(self.n_bins, dtype=np.float64)
        cov = np.empty(self.n_bins, dtype=np.uint8)
        assert lib().qtam_ref_plan_frame(self._h, plane, _dp(P),
                                         cov.ctypes.data_as(C.POINTER(C.c_uint8))) == 0
        return P, cov.astype(bool)

    def _x(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        if x.ndim == 1:
            x = x[None, :]
        assert x.shape[1] == self.N
        return x

    def forward(self, x, engine=0):
        x = self._x(x)
        out = np.empty((x.shape[0], self.ctot), dtype=np.complex128)
        assert lib().qtam_ref_forward(self._h, _dp(x), x.shape[0], _dp(out.view(np.float64)), engine) == 0
        return out

    def inverse(self, coef, plane=-1, engine=0):
        c = np.ascontiguousarray(coef, dtype=np.complex128)
        if c.ndim == 1:
            c = c[None, :]
        assert c.shape[1] == self.ctot
        out = np.empty((c.shape[0], self.N), dtype=np.float64)
        assert lib().qtam_ref_inverse(self._h, _dp(c.view(np.float64)), c.shape[0], plane, _dp(out), engine) == 0
        return out

    def dense(self, x, row_begin=0, row_end=None, engine=0):
        x = self._x(x)
        row_end = self.n_rows if row_end is None else row_end
        out = np.empty((x.shape[0], row_end - row_begin, self.N), dtype=np.complex128)
        assert lib().qtam_ref_dense(self._h, _dp(x), x.shape[0], row_begin, row_end,
                                    _dp(out.view(np.float64)), engine) == 0
        return out

    def brute_tile(self, x, k):
        x = np.ascontiguousarray(x, dtype=np.float64).reshape(-1)
        assert x.size == self.N
        out = np.empty(self.N, dtype=np.complex128)
        assert lib().qtam_ref_brute_tile(self._h, _dp(x), k, _dp(out.view(np.float64))) == 0
        return out

    def threshold(self, coef, kappa=3.0):
        c = np.array(coef, dtype=np.complex128, order="C", copy=True)
        if c.ndim == 1:
            c = c[None, :]
        assert lib().qtam_ref_threshold_rowmedian(self._h, _dp(c.view(np.float64)), c.shape[0], kappa) == 0
        return c

    def remodulate(self, coef):
        """decimated envelopes -> samples of the dense tiles T_k[n N/M_k] (Eq. 10a, identity P2)"""
        c = np.ascontiguousarray(np.atleast_2d(coef), dtype=np.complex128)
        out = np.empty_like(c)
        assert lib().qtam_ref_remodulate(self._h, _dp(c.view(np.float64)), c.shape[0], _dp(out.view(np.float64))) == 0
        return out

    def instantaneous_frequency(self, coef):
        """[batch][ctot] real: forward difference of the unwrapped baseband phase plus the carrier, in Hz"""
        c = np.ascontiguousarray(np.atleast_2d(coef), dtype=np.complex128)
        out = np.empty(c.shape, dtype=np.float64)
        assert lib().qtam_ref_instantaneous_frequency(self._h, _dp(c.view(np.float64)), c.shape[0], _dp(out)) == 0
        return out

    def plane_sizes(self):
        """coefficients per plane in the layout"""
        sizes = np.zeros(self.n_planes, dtype=np.int64)
        for r in self.rows:
            sizes[r.plane] += r.M
        return sizes

    def gather_plane(self, coef, best):
        c = np.ascontiguousarray(np.atleast_2d(coef), dtype=np.complex128)
        b = np.ascontiguousarray(best, dtype=np.int32)
        out = np.empty((c.shape[0], int(self.plane_sizes().max())), dtype=np.complex128)
        rc = lib().qtam_ref_gather_plane(self._h, _dp(c.view(np.float64)), c.shape[0],
                                         b.ctypes.data_as(C.POINTER(C.c_int32)), _dp(out.view(np.float64)))
        assert rc == 0
        return out

    def dense_invert(self, tile, row):
        """x[batch][N] from ONE dense tile per segment (Eq. 13); the plan needs epsilon > 0"""
        c = np.ascontiguousarray(np.atleast_2d(tile), dtype=np.complex128)
        out = np.empty((c.shape[0], self.N), dtype=np.float64)
        rc = lib().qtam_ref_dense_invert(self._h, _dp(c.view(np.float64)), c.shape[0], int(row), _dp(out))
        if rc != 0:
            raise ValueError(f"qtam_ref_dense_invert failed with code {rc}")
        return out

    def plane_metric(self, coef, metric="energy"):
        """(values[batch][n_planes], best[batch]) of the multi-Q scan's plane selection"""
        c = np.ascontiguousarray(np.atleast_2d(coef), dtype=np.complex128)
        vals = np.zeros((c.shape[0], self.n_planes))
        best = np.zeros(c.shape[0], dtype=np.int32)
        rc = lib().qtam_ref_plane_metric(self._h, _dp(c.view(np.float64)), c.shape[0],
                                         {"energy": 0, "peak": 1}[metric], _dp(vals),
                                         best.ctypes.data_as(C.POINTER(C.c_int32)))
        assert rc == 0
        return vals, best

    def threshold_f32(self, coef, kappa=3.0):
        c = np.array(coef, dtype=np.complex64, order="C", copy=True)
        if c.ndim == 1:
            c = c[None, :]
        ptr = c.view(np.float32).ctypes.data_as(C.POINTER(C.c_float))
        assert lib().qtam_ref_threshold_rowmedian_f32(self._h, ptr, c.shape[0], kappa) == 0
        return c

    def plane_slice(self, plane):
        rows = [r for r in self.rows if r.plane == plane]
        return slice(int(rows[0].offset), int(rows[-1].offset + rows[-1].M)), len(rows), int(rows[0].M)

    def cluster(self, coef, plane, min_area=1):
        """(labels[batch][rows][M] int32, count[batch]) of the clusters of NON-ZERO coefficients of one Q-plane in
        the uniform-tile layout: apply the row-median threshold first (the normalized threshold)."""
        c = np.atleast_2d(np.asarray(coef))
        sl, R, M = self.plane_slice(plane)
        assert all(r.M == M for r in self.rows if r.plane == plane), "uniform tile layout needed"
        mask = np.ascontiguousarray((c[:, sl] != 0).astype(np.uint8))
        return cluster_labels(mask.reshape(c.shape[0], R, M), min_area)

    def apply_mask(self, coef, plane, labels, label=0):
        """the binary mask of one cluster (label > 0) or of every kept cluster (label 0) applied to the plane's
        coefficients; everything else, the other planes included, is zero"""
        c = np.atleast_2d(np.asarray(coef))
        out = np.zeros_like(c)
        sl, R, M = self.plane_slice(plane)
        L = np.asarray(labels).reshape(c.shape[0], R * M)
        keep = (L == label) if label > 0 else (L > 0)
        out[:, sl] = np.where(keep, c[:, sl], 0)
        return out

    def output_length(self, mode):
        """'standard' (N/2 + 1) or 'minimal' (the largest window's 2 dk + 1)"""
        return int(lib().qtam_ref_output_length(self._h, {"standard": -1, "minimal": -2}[mode]))

    def forward_length(self, x, n, engine=0):
        """[batch][rows][n]: every row resampled to n time samples (A22)"""
        x = self._x(x)
        out = np.empty((x.shape[0], self.n_rows, n), dtype=np.complex128)
        assert lib().qtam_ref_forward_length(self._h, _dp(x), x.shape[0], n, _dp(out.view(np.float64)), engine) == 0
        return out

    def inverse_length(self, img, plane=-1, engine=0):
        img = np.ascontiguousarray(img, dtype=np.complex128)
        if img.ndim == 2:
            img = img[None]
        out = np.empty((img.shape[0], self.N), dtype=np.float64)
        assert lib().qtam_ref_inverse_length(self._h, _dp(img.view(np.float64)), img.shape[0], img.shape[-1], plane,
                                             _dp(out), engine) == 0
        return out

    def resample(self, img, n_out):
        img = np.ascontiguousarray(img, dtype=np.complex128)
        if img.ndim == 2:
            img = img[None]
        out = np.empty((img.shape[0], self.n_rows, n_out), dtype=np.complex128)
        assert lib().qtam_ref_resample(self._h, _dp(img.view(np.float64)), img.shape[0], img.shape[-1], n_out,
                                       _dp(out.view(np.float64))) == 0
        return out

    def project_cover(self, x, plane=-1, engine=0):
        x = self._x(x)
        out = np.empty_like(x)
        assert lib().qtam_ref_project_cover(self._h, _dp(x), x.shape[0], plane, _dp(out), engine) == 0
        return out

    def spectrum(self, x, engine=0):
        x = self._x(x)
        out = np.empty((x.shape[0], self.n_bins), dtype=np.complex128)
        assert lib().qtam_ref_spectrum(self._h, _dp(x), x.shape[0], _dp(out.view(np.float64)), engine) == 0
        return out

    def row_slice(self, k):
        r = self.rows[k]
        return slice(int(r.offset), int(r.offset + r.M))
