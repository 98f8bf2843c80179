"""CPU-side checks of libqtam: the shared library loads, exports every symbol include/qtam.h declares,
its host plan equals the oracle's plan (integers bit for bit, windows to 1 ulp), and bad arguments
are refused with status codes.  No compute call is made (no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle.qtam_ref import RefPlan
from paper_2603_29785_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "qtam.h")).read()
    declared = set(re.findall(r"\b(qtam_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations found"
    L = binding.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"libqtam.so does not export {name}"
    assert set(binding.SYMBOLS) == declared


def test_status_strings():
    L = binding.lib()
    assert L.qtam_status_string(0) == b"ok"
    assert b"argument" in L.qtam_status_string(1)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "paper6s"])
@pytest.mark.parametrize("ov", [1.0, 2.0])
def test_host_plan_equals_oracle_plan(name, ov):
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
    dt = inputs.CONFIGS[name]["dtype"]
    p = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype=dt, clamp_overlap=ov, host_only=True)
    r = RefPlan(fs, N, Q, fmin, fmax, rows, clamp_overlap=ov)
    assert (p.n_rows, p.n_planes, p.ctot, p.N, p.n_bins) == (r.n_rows, r.n_planes, r.ctot, r.N, r.n_bins)
    for a, b in zip(p.rows, r.rows):
        assert (a.plane, a.row, a.kc, a.dk, a.L, a.M, a.offset) == (b.plane, b.row, b.kc, b.dk, b.L, b.M, b.offset)
        assert a.q == b.q and a.f_request == b.f_request and a.f_center == b.f_center
        assert abs(a.norm - b.norm) <= 2e-16 * b.norm
    step = 1 if name != "cfg4" else 37
    for k in range(0, p.n_rows, step):
        wa, wb = p.window(k), r.window(k)
        assert np.max(np.abs(wa - wb)) <= np.spacing(np.max(wb))
    for plane in range(-1, p.n_planes):
        Pa, Ca = p.frame(plane)
        Pb, Cb = r.frame(plane)
        assert np.array_equal(Ca, Cb)
        assert np.max(np.abs(Pa - Pb)) <= 4 * np.spacing(np.max(Pb))
    ia, ib = p.info, r.info
    assert (ia.cover_lo, ia.cover_hi, ia.holes, ia.sum_L) == (ib.cover_lo, ib.cover_hi, ib.holes, ib.sum_L)
    assert ia.frame_A == pytest.approx(ib.frame_A, rel=1e-14) and ia.frame_B == pytest.approx(ib.frame_B, rel=1e-14)


def test_bins_per_octave_grid_matches_oracle():
    p = binding.Plan(4096.0, 4096, [6.0, 12.0], 20.0, 900.0, 8, rows_are_bins_per_octave=1, host_only=True)
    r = RefPlan(4096.0, 4096, [6.0, 12.0], 20.0, 900.0, 8, rows_are_bins_per_octave=1)
    assert p.n_rows == r.n_rows and p.ctot == r.ctot
    f = [x.f_request for x in p.rows[: p.n_rows // 2]]
    assert f[0] == 20.0 and abs(f[8] - 40.0) < 1e-12 and f[-1] <= 900.0 < f[-1] * 2 ** (1 / 8)


def test_manual_clamp_and_no_clamp():
    a = binding.Plan(4096.0, 4096, [8.0], 16.0, 512.0, 16, clamp_mode=2, max_window_bins=40, host_only=True)
    assert max(x.L for x in a.rows) == 39
    b = binding.Plan(4096.0, 4096, [8.0], 16.0, 512.0, 16, clamp_mode=0, host_only=True)
    assert max(x.L for x in b.rows) == 2 * int(np.floor(512.0 * np.sqrt(11.0) / 8.0)) + 1
    rb = RefPlan(4096.0, 4096, [8.0], 16.0, 512.0, 16, clamp_mode=0)
    assert [x.L for x in b.rows] == [x.L for x in rb.rows]


@pytest.mark.parametrize("bad", [dict(N=3000), dict(fmax=2048.0), dict(fmin=0.0), dict(fmin=-1.0),
                                 dict(Q=[3.0]), dict(fmin=1.0, Q=[64.0]), dict(spacing=1),
                                 dict(fmax=10.0), dict(N=4)])
def test_plan_create_refuses_bad_arguments(bad):
    ok = dict(fs=4096.0, N=4096, Q=[8.0], fmin=16.0, fmax=1024.0, spacing=16)
    binding.Plan(**ok, host_only=True)
    with pytest.raises(binding.QtamError) as e:
        binding.Plan(**{**ok, **bad}, host_only=True)
    assert e.value.code == 1


def test_null_and_host_only_calls_fail_loudly():
    L = binding.lib()
    assert L.qtam_plan_destroy(None) == 1
    assert L.qtam_plan_info(None, None) == 1
    p = binding.Plan(4096.0, 4096, [8.0], 16.0, 1024.0, 16, host_only=True)
    # compute calls on a host-only plan are refused: there is no CPU fallback
    assert L.qtam_forward(p._h, C.c_void_p(16), 1, C.c_void_p(16), None) == 4
    assert L.qtam_inverse(p._h, C.c_void_p(16), 1, -1, C.c_void_p(16), None) == 4
    assert L.qtam_dense(p._h, C.c_void_p(16), 1, 0, 1, C.c_void_p(16), None) == 4
    assert L.qtam_threshold_rowmedian(p._h, C.c_void_p(16), 1, 3.0, None) == 4
    rows = (binding.Row * 4)()
    assert L.qtam_plan_rows(p._h, rows, 4) == 1      # capacity too small
    assert L.qtam_plan_window(p._h, 99, None) == 1
    assert L.qtam_plan_frame(p._h, 5, None, None) == 1


def test_plan_create_without_gpu_reports_cuda_error():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.QtamError) as e:
        binding.Plan(4096.0, 4096, [8.0], 16.0, 1024.0, 16)
    assert e.value.code == 4


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_29785_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".hpp", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "qtam_ref" not in src and "import oracle" not in src and "from oracle" not in src, f


@pytest.mark.parametrize("window,par", [("hann", 0.0), ("kaiser", 6.5), ("tukey", 0.4), ("planck", 0.5)])
def test_window_families_host_plan_matches_oracle(window, par):
    """App. A, A2-A6: the library's window tables (its own evaluation, Bessel I_0 from <cmath>) against
    the oracle's (power series in long double); cover sets equal, P to a few ulp."""
    args = (4096.0, 4096, [4.0, 8.0, 16.0], 16.0, 1024.0, 32)
    p = binding.Plan(*args, dtype="f64", host_only=True, window=window, window_param=par)
    r = RefPlan(*args, window=window, window_param=par)
    assert [(a.kc, a.dk, a.M, a.offset) for a in p.rows] == [(b.kc, b.dk, b.M, b.offset) for b in r.rows]
    for k in range(p.n_rows):
        wb = r.window(k)
        assert np.max(np.abs(p.window(k) - wb)) <= 1e-14 * np.max(wb)     # cyl_bessel_i is good to a few ulp
    Pa, Ca = p.frame(-1)
    Pb, Cb = r.frame(-1)
    assert np.array_equal(Ca, Cb)
    assert np.max(np.abs(Pa - Pb)) <= 1e-14 * np.max(Pb)


def test_window_parameters_and_manual_grid_are_validated():
    args = (4096.0, 4096, [4.0, 8.0], 16.0, 1024.0, 16)
    with pytest.raises(binding.QtamError):
        binding.Plan(*args, host_only=True, window="kaiser", window_param=0.0)
    with pytest.raises(binding.QtamError):
        binding.Plan(*args, host_only=True, window="tukey", window_param=1.5)
    with pytest.raises(binding.QtamError):
        binding.Plan(4096.0, 4096, [4.0], 0.0, 0.0, 0.0, host_only=True, freqs=[50.0, 40.0, 90.0])
    freqs = [20.0, 30.0, 47.0, 80.0, 150.0, 260.0, 400.0]
    p = binding.Plan(4096.0, 4096, [4.0, 12.0], 0.0, 0.0, 0.0, host_only=True, freqs=freqs)
    r = RefPlan(4096.0, 4096, [4.0, 12.0], 0.0, 0.0, 0.0, freqs=freqs)
    assert [(a.kc, a.dk, a.M, a.offset, a.f_request) for a in p.rows] == \
           [(b.kc, b.dk, b.M, b.offset, b.f_request) for b in r.rows]


@pytest.mark.parametrize("tile_length", [-1, 4096])
def test_uniform_tile_length_host_plan_matches_oracle(tile_length):
    args = (4096.0, 4096, [4.0, 8.0, 16.0], 16.0, 1024.0, 32)
    p = binding.Plan(*args, dtype="f64", host_only=True, tile_length=tile_length)
    r = RefPlan(*args, tile_length=tile_length)
    assert [(a.kc, a.dk, a.L, a.M, a.offset) for a in p.rows] == [(b.kc, b.dk, b.L, b.M, b.offset) for b in r.rows]
    assert p.ctot == r.ctot
    with pytest.raises(binding.QtamError):
        binding.Plan(*args, host_only=True, tile_length=96)
    with pytest.raises(binding.QtamError):
        binding.Plan(*args, host_only=True, tile_length=64)


def test_output_length_modes_on_a_host_plan():
    """standard = N/2 + 1, minimal = the largest window; a length below it is refused"""
    kw = dict(dtype="f32", host_only=True)
    p = binding.Plan(4096.0, 24576, [8.0], 20.0, 1800.0, 62.0, out_length="minimal", **kw)
    lmax = max(int(r.L) for r in p.rows)
    assert p.output_length() == lmax == p.output_length("minimal") and p.output_length("standard") == 12289
    assert binding.Plan(4096.0, 24576, [8.0], 20.0, 1800.0, 62.0, out_length="standard", **kw).output_length() == 12289
    assert binding.Plan(4096.0, 24576, [8.0], 20.0, 1800.0, 62.0, out_length=lmax + 5, **kw).output_length() == lmax + 5
    assert binding.Plan(4096.0, 24576, [8.0], 20.0, 1800.0, 62.0, **kw).output_length() == 0


def test_composite_bank_host_plan_equals_oracle_plan():
    cfgs = [(8.0, "bisquare", 0.0), (8.0, "hann", 0.0), (16.0, "tukey", 0.5), (16.0, "kaiser", 6.0), (32.0, "planck", 0.4)]
    kw = dict(plane_windows=[(c[1], c[2]) for c in cfgs])
    p = binding.Plan(4096.0, 8192, [c[0] for c in cfgs], 20.0, 1800.0, 24.0, dtype="f64", host_only=True, **kw)
    r = RefPlan(4096.0, 8192, [c[0] for c in cfgs], 20.0, 1800.0, 24.0, **kw)
    assert p.ctot == r.ctot and p.n_rows == r.n_rows
    for k in range(p.n_rows):
        wa, wb = p.window(k), r.window(k)
        assert np.max(np.abs(wa - wb)) <= 1e-14 * np.max(wb)      # two independent evaluations of cos / I_0 / exp
        assert abs(p.rows[k].norm - r.rows[k].norm) <= 1e-14 * r.rows[k].norm
    for plane in range(-1, p.n_planes):
        Pa, Ca = p.frame(plane)
        Pb, Cb = r.frame(plane)
        assert np.array_equal(Ca, Cb) and np.max(np.abs(Pa - Pb)) <= 1e-13 * np.max(Pb)
    with pytest.raises(ValueError):
        binding.Plan(4096.0, 8192, [8.0, 16.0], 20.0, 1800.0, 24.0, host_only=True, plane_windows=[("hann", 0.0)])
