"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these touch the CUDA path.  Each pin is chosen so that a plausible mistake in the oracle
(dropped term, wrong sign or index, transposed operand, wrong scale) fails at least one of them.
Independent references used: brute-force circular convolution (no DFT of x), closed forms, numpy.fft
as an outside library, exact rationals for the window.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from conftest import rel_l2
from oracle.qtam_ref import RefPlan, cluster_labels, dft, fft
from paper_2603_29785_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def mk(args, **kw):
    return RefPlan(args["fs"], args["N"], args["Q"], args["fmin"], args["fmax"], args["spacing"], **kw)


@pytest.fixture(scope="module")
def plan256(small_plan_args):
    return mk(small_plan_args)


@pytest.fixture(scope="module")
def plan1k():
    # 1024 samples, three planes, clamp active on the top rows, M from 8 to 64
    return RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)


# ---- P11: the oracle's DFT engines ------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_p11_fft_vs_naive_dft(n):
    rng = np.random.default_rng(n)
    z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        a, b = dft(z, sign), fft(z, sign)
        assert rel_l2(b, a) <= 1e-13


@pytest.mark.parametrize("n", [3, 6, 12, 24, 48, 96, 192, 384, 768, 1536, 3072])
def test_p11_mixed_radix_fft_vs_naive_dft(n):
    """segment lengths 3 * 2^k (the paper's benchmark shape, 6 s at 4096 Hz = 24576 samples):
    the engine's radix-3 step against the naive sums, and at the benchmark length against an outside library"""
    rng = np.random.default_rng(n)
    z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        assert rel_l2(fft(z, sign), dft(z, sign)) <= 1e-13
    z = rng.standard_normal(24576) + 1j * rng.standard_normal(24576)
    assert rel_l2(fft(z, -1), np.fft.fft(z)) <= 1e-13


@pytest.mark.parametrize("n", [8, 12, 64, 100, 1024])
def test_naive_dft_vs_numpy_library(n):
    """C1/C2 sign and index convention against an outside library."""
    rng = np.random.default_rng(7 + n)
    z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert rel_l2(dft(z, -1), np.fft.fft(z)) <= 1e-13
    assert rel_l2(dft(z, +1), np.fft.ifft(z) * n) <= 1e-13


def test_naive_dft_delta_and_constant():
    n = 16
    e = np.zeros(n, complex); e[3] = 1
    k = np.arange(n)
    assert np.allclose(dft(e, -1), np.exp(-2j * np.pi * 3 * k / n), atol=1e-15)
    assert np.allclose(dft(np.ones(n, complex), -1), n * (k == 0), atol=1e-13)


# ---- P12: plan invariants + closed-form window ------------------------------------------------

def test_window_closed_form_golden():
    """bisquare dk=3 against exact rationals (tests/golden/bisquare_dk3.txt; Eq. 6, Eq. 5/R3)."""
    fs, N, Q, fmin, fmax, rows = inputs.plan_args("cfg1")
    p = RefPlan(fs, N, Q, fmin, fmax, rows)
    k = 2 * 32  # plane Q=16 (third), lowest row
    r = p.rows[k]
    assert (r.q, r.kc, r.dk, r.L, r.M) == (16.0, 16, 3, 7, 8)
    vals, S = {}, None
    for line in open(os.path.join(GOLD, "bisquare_dk3.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] == "S":
            S = Fraction(int(t[1]), int(t[2]))
        else:
            vals[int(t[0])] = Fraction(int(t[1]), int(t[2]))
    # the file's rationals are Eq. 6 evaluated exactly
    for j, v in vals.items():
        assert v == (1 - Fraction(j * j, 9)) ** 2
    raw = np.array([float(vals[j]) for j in range(-3, 4)])
    assert S == sum(((1 - Fraction(j * j, 9)) ** 2) ** 2 for j in range(-3, 4))
    w = p.window(k)
    expect = raw / np.sqrt(float(S))
    assert np.max(np.abs(w - expect)) <= 2e-16
    assert abs(np.sum(w * w) - 1.0) <= 1e-15


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
@pytest.mark.parametrize("ov", [1.0, 2.0])
def test_p12_plan_invariants(name, ov):
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
    p = RefPlan(fs, N, Q, fmin, fmax, rows, clamp_overlap=ov)
    T = N / fs
    off = 0
    Lmax = max(r.L for r in p.rows)
    for r in p.rows:
        assert r.L == 2 * r.dk + 1 and r.dk >= 1
        assert r.M >= r.L and r.M < 2 * r.L and (r.M & (r.M - 1)) == 0
        assert r.offset == off
        off += r.M
        assert r.kc == int(np.floor(r.f_request * T + 0.5))
        assert r.L == min(2 * int(np.floor(r.f_request * T * np.sqrt(11.0) / r.q)) + 1, Lmax)
    assert off == p.ctot
    # grid endpoints inclusive, geometric (R14)
    R = int(rows)
    assert abs(p.rows[0].f_request - fmin) < 1e-12 and abs(p.rows[R - 1].f_request - fmax) < 1e-9
    ratio = [p.rows[i + 1].f_request / p.rows[i].f_request for i in range(R - 1)]
    assert max(ratio) - min(ratio) < 1e-12
    # A7: L_max = 2*floor(ceil(ov*T*dfmax)/2)+1, dfmax = largest gap
    dfmax = max(p.rows[i + 1].f_request - p.rows[i].f_request for i in range(R - 1))
    assert Lmax == 2 * (int(np.ceil(ov * T * dfmax)) // 2) + 1
    # P recomputed from the rows equals the plan's; per-plane P sum to the joint P (C36/C51)
    Pj, Cj = p.frame(-1)
    acc = np.zeros(p.n_bins)
    accp = np.zeros((p.n_planes, p.n_bins))
    if name != "cfg4":
        for k, r in enumerate(p.rows):
            w = p.window(k)
            f = np.arange(r.kc - r.dk, r.kc + r.dk + 1)
            ok = (f >= 0) & (f < p.n_bins)
            np.add.at(acc, f[ok], w[ok] ** 2)
            np.add.at(accp[r.plane], f[ok], w[ok] ** 2)
        assert np.max(np.abs(acc - Pj)) <= 1e-15 * max(1.0, Pj.max())
    Psum = np.zeros(p.n_bins)
    cov_or = np.zeros(p.n_bins, bool)
    for pl in range(p.n_planes):
        Pp, Cp = p.frame(pl)
        Psum += Pp
        cov_or |= Cp
        if name != "cfg4":
            assert np.max(np.abs(accp[pl] - Pp)) <= 1e-15 * max(1.0, Pp.max())
    assert np.max(np.abs(Psum - Pj)) <= 4e-16 * max(1.0, Pj.max())
    assert np.array_equal(cov_or, Cj)
    assert np.all(Pj[Cj] > 0)
    i = p.info
    assert i.frame_A == Pj[Cj].min() and i.frame_B == Pj.max()
    assert i.holes == (i.cover_hi - i.cover_lo + 1) - Cj.sum()
    if ov == 2.0:
        assert i.holes == 0  # R7: overlap 2 gives hole-free frames on every configuration


def test_plan_table_sizes_match_survey():
    """SURVEY.md 8 per-config table (re-derived, not assumed)."""
    want = {"cfg1": (96, 8186, 14784), "cfg2": (144, 129464, 198272), "cfg3": (320, 103950, 170360),
            "cfg4": (480, 6767322, 10934848), "cfg5": (192, 14272, 25148)}
    for name, (K, sumL, ctot) in want.items():
        fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
        p = RefPlan(fs, N, Q, fmin, fmax, rows)
        assert (p.n_rows, p.info.sum_L, p.ctot) == (K, sumL, ctot)


def test_plan_rejects_bad_arguments():
    ok = dict(fs=256.0, N=256, Q=[4.0], fmin=8.0, fmax=100.0, spacing=6)
    RefPlan(**ok)
    RefPlan(**{**ok, **dict(N=192, fs=192.0, fmax=90.0)})          # 3 * 2^k is a segment length too
    for bad in (dict(N=300), dict(N=320), dict(N=12), dict(fmax=128.0), dict(fmin=0.0), dict(Q=[3.0]), dict(fmin=1.0, Q=[64.0])):
        with pytest.raises(ValueError):
            RefPlan(**{**ok, **bad})


# ---- P1: dense vs brute-force circular convolution --------------------------------------------

@pytest.mark.parametrize("engine", [0, 1])
def test_p1_dense_vs_bruteforce(plan256, engine):
    x = inputs.white_noise(256, 11)[0]
    D = plan256.dense(x, engine=engine)[0]
    for k in range(plan256.n_rows):
        B = plan256.brute_tile(x, k)
        assert rel_l2(D[k], B) <= 1e-12, k


def test_p1_bruteforce_tiny_n64():
    p = RefPlan(64.0, 64, [4.0], 6.0, 20.0, 4)
    x = inputs.white_noise(64, 12)[0]
    D = p.dense(x)[0]
    for k in range(p.n_rows):
        assert rel_l2(D[k], p.brute_tile(x, k)) <= 1e-12


@pytest.mark.parametrize("N", [96, 192])
def test_non_power_of_two_segment_length(N):
    """N = 3 * 2^k: the same pins as for powers of two -- P1 dense tiles
    against the brute-force circular convolution (no DFT of x), both engines; P2 against the dense tiles; P4 the
    round trip against an outside library's projection; P6 the frame-energy identity; the engines agree."""
    p = RefPlan(float(N), N, [4.0, 8.0], 5.0, 0.42 * N, 7.0)
    assert p.N == N and p.n_bins == N // 2 + 1
    x = inputs.white_noise(N, 60 + N, batch=2)
    for engine in (0, 1):
        D = p.dense(x[0], engine=engine)[0]
        for k in range(p.n_rows):
            assert rel_l2(D[k], p.brute_tile(x[0], k)) <= 1e-12, (engine, k)
    Y0, Y1 = p.forward(x, engine=0), p.forward(x, engine=1)
    assert rel_l2(Y1, Y0) <= 1e-13
    D = p.dense(x[0], engine=0)[0]
    for k, r in enumerate(p.rows):
        if N % r.M:
            continue                                   # P2 needs tau = n N / M on the sample grid
        n = np.arange(r.M)
        want = np.sqrt(N / r.M) * np.exp(-2j * np.pi * r.kc * n / r.M) * D[k][n * N // r.M]
        assert rel_l2(Y0[0, p.row_slice(k)], want) <= 1e-12, k
    X = np.fft.rfft(x, axis=-1)
    P, _ = p.frame(-1)
    tot = np.sum(np.abs(Y0) ** 2, axis=1)
    assert np.all(np.abs(tot - np.sum(np.abs(X) ** 2 * P[None, :], axis=1) / N) <= 1e-13 * tot)
    for plane in (-1, 0, 1):
        _, C = p.frame(plane)
        proj = np.fft.irfft(np.where(C[None, :], X, 0), n=N, axis=-1)
        for engine in (0, 1):
            assert rel_l2(p.inverse(Y0, plane=plane, engine=engine), proj) <= 1e-12, (plane, engine)


def test_bruteforce_atom_is_time_domain_definition():
    """the brute-force path itself, against a literal numpy evaluation of C4/C5"""
    p = RefPlan(64.0, 64, [4.0], 6.0, 20.0, 4)
    x = inputs.white_noise(64, 13)[0]
    N = 64
    n = np.arange(N)
    for k, r in enumerate(p.rows):
        w = p.window(k)
        f = np.arange(r.kc - r.dk, r.kc + r.dk + 1)
        T = np.zeros(N, complex)
        for tau in range(N):
            g = (1.0 / N) * np.sum(w[None, :] * np.exp(2j * np.pi * f[None, :] * (tau - n[:, None]) / N), axis=1)
            T[tau] = np.sum(x * g)
        assert rel_l2(p.brute_tile(x, k), T) <= 1e-12


# ---- P2 / P3: decimated coefficients vs dense tiles -------------------------------------------

@pytest.mark.parametrize("engine", [0, 1])
def test_p2_decimated_is_sampled_demodulated_dense(plan1k, engine):
    p = plan1k
    x = inputs.white_noise(p.N, 21)[0]
    Y = p.forward(x, engine=engine)[0]
    D = p.dense(x, engine=engine)[0]
    for k, r in enumerate(p.rows):
        n = np.arange(r.M)
        step = p.N // r.M
        expect = np.sqrt(p.N / r.M) * np.exp(-2j * np.pi * ((r.kc * n) % r.M) / r.M) * D[k][n * step]
        assert rel_l2(Y[p.row_slice(k)], expect) <= 1e-12, k


def test_p3_row_energy(plan1k):
    p = plan1k
    x = inputs.white_noise(p.N, 22)[0]
    Y = p.forward(x)[0]
    D = p.dense(x)[0]
    X = np.fft.rfft(x)
    for k, r in enumerate(p.rows):
        w = p.window(k)
        f = np.arange(r.kc - r.dk, r.kc + r.dk + 1)
        ok = (f >= 0) & (f < p.n_bins)
        e_spec = np.sum(np.abs(X[f[ok]] * w[ok]) ** 2) / p.N
        e_dec = np.sum(np.abs(Y[p.row_slice(k)]) ** 2)
        e_dense = np.sum(np.abs(D[k]) ** 2)
        assert abs(e_dec - e_spec) <= 1e-13 * e_spec
        assert abs(e_dense - e_spec) <= 1e-13 * e_spec


def test_forward_vs_numpy_library_construction(plan1k):
    """special case reducing to library routines: rfft, then ifft of the shifted windowed band"""
    p = plan1k
    x = inputs.white_noise(p.N, 23)[0]
    Y = p.forward(x)[0]
    X = np.fft.rfft(x)
    for k, r in enumerate(p.rows):
        w = p.window(k)
        B = np.zeros(r.M, complex)
        for j in range(-r.dk, r.dk + 1):
            if 0 <= r.kc + j < p.n_bins:
                B[j % r.M] = X[r.kc + j] * w[j + r.dk]
        expect = np.fft.ifft(B) * np.sqrt(r.M / p.N)
        assert rel_l2(Y[p.row_slice(k)], expect) <= 1e-12


# ---- P4: round trip ---------------------------------------------------------------------------

@pytest.mark.parametrize("ov", [1.0, 2.0])
@pytest.mark.parametrize("engine", [0, 1])
def test_p4_round_trip_joint_and_per_plane(ov, engine):
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12, clamp_overlap=ov)
    x = inputs.white_noise(p.N, 31, batch=2)
    Y = p.forward(x, engine=engine)
    X = np.fft.rfft(x, axis=-1)
    for plane in (-1, 0, 1, 2):
        _, C = p.frame(plane)
        proj = np.fft.irfft(np.where(C[None, :], X, 0), n=p.N, axis=-1)   # Pi_C x by an outside library
        xr = p.inverse(Y, plane=plane, engine=engine)
        assert rel_l2(xr, proj) <= 1e-12, plane
        assert rel_l2(p.project_cover(x, plane=plane, engine=engine), proj) <= 1e-12
    # Pi_C really removes something with the literal clamp, so the test is not vacuous
    assert rel_l2(proj, x) > 1e-3


def test_p4_round_trip_cfg1_fp64():
    """BASELINE config 1 (PR1 ref) at full size, round trip <= 1e-12 against Pi_C x."""
    fs, N, Q, fmin, fmax, rows = inputs.plan_args("cfg1")
    p = RefPlan(fs, N, Q, fmin, fmax, rows)
    x = inputs.make_batch("cfg1")
    Y = p.forward(x, engine=1)
    xr = p.inverse(Y, engine=1)
    _, C = p.frame(-1)
    proj = np.fft.irfft(np.where(C[None, :], np.fft.rfft(x, axis=-1), 0), n=N, axis=-1)
    assert rel_l2(xr, proj) <= 1e-12
    # white noise keeps only about half its energy in C for this plan (R9)
    assert 0.4 < np.sum(proj ** 2) / np.sum(x ** 2) < 0.65


def test_inverse_vs_numpy_library_construction(plan1k):
    p = plan1k
    rng = np.random.default_rng(33)
    Y = rng.standard_normal(p.ctot) + 1j * rng.standard_normal(p.ctot)   # arbitrary coefficients
    P, C = p.frame(-1)
    S = np.zeros(p.n_bins, complex)
    for k, r in enumerate(p.rows):
        w = p.window(k)
        Bh = np.fft.fft(Y[p.row_slice(k)]) * np.sqrt(p.N / r.M)
        for j in range(-r.dk, r.dk + 1):
            if 0 <= r.kc + j < p.n_bins:
                S[r.kc + j] += Bh[j % r.M] * w[j + r.dk]
    Xh = np.where(C, S / np.where(C, P, 1.0), 0)
    Xh[0] = Xh[0].real
    Xh[-1] = Xh[-1].real
    expect = np.fft.irfft(Xh, n=p.N)
    for engine in (0, 1):
        assert rel_l2(p.inverse(Y, engine=engine)[0], expect) <= 1e-12


# ---- P5: linearity ----------------------------------------------------------------------------

def test_p5_linearity(plan1k):
    p = plan1k
    x = inputs.white_noise(p.N, 41, batch=2)
    a, b = 0.7, -1.9
    lhs = p.forward(a * x[0] + b * x[1])[0]
    Y = p.forward(x)
    rhs = a * Y[0] + b * Y[1]
    assert rel_l2(lhs, rhs) <= 1e-13


# ---- P6: frame energy identity and bounds -----------------------------------------------------

@pytest.mark.parametrize("ov", [1.0, 2.0])
def test_p6_frame_energy(ov):
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12, clamp_overlap=ov)
    x = inputs.white_noise(p.N, 51)[0]
    P, C = p.frame(-1)
    X = np.fft.rfft(x)
    Y = p.forward(x)[0]
    total = np.sum(np.abs(Y) ** 2)
    assert abs(total - np.sum(np.abs(X) ** 2 * P) / p.N) <= 1e-13 * total
    # bounds for x = Pi_C x (no DC / Nyquist content): (A/2)|x|^2 <= sum|Y|^2 <= (B/2)|x|^2
    assert not C[0] and not C[-1]
    xc = np.fft.irfft(np.where(C, X, 0), n=p.N)
    Yc = p.forward(xc)[0]
    e = np.sum(np.abs(Yc) ** 2)
    A, B = P[C].min(), P.max()
    nx = np.sum(xc ** 2)
    assert A / 2 * nx * (1 - 1e-12) <= e <= B / 2 * nx * (1 + 1e-12)


# ---- P7: pure sinusoid closed form ------------------------------------------------------------

@pytest.mark.parametrize("k0", [40, 97, 250])
def test_p7_pure_sinusoid(plan1k, k0):
    p = plan1k
    n = np.arange(p.N)
    x = np.cos(2 * np.pi * k0 * n / p.N)
    Y = p.forward(x)[0]
    peak, best = [], -1.0
    for k, r in enumerate(p.rows):
        m = np.arange(r.M)
        d = k0 - r.kc
        if abs(d) <= r.dk:
            wv = p.window(k)[d + r.dk]
            expect = np.sqrt(p.N / r.M) * 0.5 * wv * np.exp(2j * np.pi * ((d * m) % r.M) / r.M)
        else:
            wv = 0.0
            expect = np.zeros(r.M, complex)
        assert np.max(np.abs(Y[p.row_slice(k)] - expect)) <= 1e-13 * np.sqrt(p.N), k
        peak.append(np.sum(np.abs(Y[p.row_slice(k)]) ** 2))
        best = max(best, wv)
    # the row with most energy is the one whose window is largest at k0 ("peaks in the expected row")
    kbest = int(np.argmax(peak))
    r = p.rows[kbest]
    assert abs(k0 - r.kc) <= r.dk and p.window(kbest)[k0 - r.kc + r.dk] == pytest.approx(best)


# ---- P8: shift covariance ---------------------------------------------------------------------

def test_p8_dense_shift_covariance(plan256):
    p = plan256
    x = inputs.white_noise(p.N, 61)[0]
    D = p.dense(x)[0]
    for s in (1, 5, 100):
        Ds = p.dense(np.roll(x, s))[0]
        assert rel_l2(Ds, np.roll(D, s, axis=-1)) <= 1e-13


def test_p8_decimated_shift_covariance(plan1k):
    p = plan1k
    x = inputs.white_noise(p.N, 62)[0]
    Y = p.forward(x)[0]
    for k, r in enumerate(p.rows):
        step = p.N // r.M
        for mult in (1, 3):
            s = mult * step
            Ys = p.forward(np.roll(x, s))[0][p.row_slice(k)]
            expect = np.roll(Y[p.row_slice(k)], mult) * np.exp(-2j * np.pi * ((r.kc * s) % p.N) / p.N)
            assert rel_l2(Ys, expect) <= 1e-13
        break  # one row per call keeps the CPU suite fast; the next test covers the others
    # all rows, one shift that is a multiple of every step
    s = p.N // min(r.M for r in p.rows)
    Ys = p.forward(np.roll(x, s))[0]
    for k, r in enumerate(p.rows):
        mult = s // (p.N // r.M)
        expect = np.roll(Y[p.row_slice(k)], mult) * np.exp(-2j * np.pi * ((r.kc * s) % p.N) / p.N)
        assert rel_l2(Ys[p.row_slice(k)], expect) <= 1e-13


# ---- P9: impulse symmetry ---------------------------------------------------------------------

def test_p9_impulse_real_even(plan1k):
    p = plan1k
    x = np.zeros(p.N); x[0] = 1.0
    Y = p.forward(x)[0]
    for k, r in enumerate(p.rows):
        if r.kc - r.dk < 0 or r.kc + r.dk >= p.n_bins:
            continue
        y = Y[p.row_slice(k)]
        assert np.max(np.abs(y.imag)) <= 1e-15
        assert np.max(np.abs(y.real - np.roll(y.real[::-1], 1))) <= 1e-15
        assert y.real[0] > 0 and y.real[0] == pytest.approx(np.max(np.abs(y)))


# ---- P10: white-noise variance ----------------------------------------------------------------

def test_p10_white_noise_variance(plan1k):
    p = plan1k
    nseg = 200
    x = inputs.white_noise(p.N, 71, batch=nseg)
    Y = p.forward(x, engine=1)
    for k, r in enumerate(p.rows):
        v = np.abs(Y[:, p.row_slice(k)]) ** 2
        est = v.mean() * r.M                 # E|Y|^2 = 1/M  (unit-energy window, scale R4)
        # |Y|^2 is exponential (complex Gaussian); samples within a row are correlated: about L
        # independent values per row -> sigma ~ 1/sqrt(nseg*L)
        sigma = 1.0 / np.sqrt(nseg * r.L)
        assert abs(est - 1.0) <= 4 * sigma, (k, est)


# ---- engines agree; threshold ------------------------------------------------------------------

def test_engines_agree(plan1k):
    p = plan1k
    x = inputs.white_noise(p.N, 81, batch=2)
    Y0, Y1 = p.forward(x, engine=0), p.forward(x, engine=1)
    assert rel_l2(Y1, Y0) <= 1e-13
    assert rel_l2(p.inverse(Y0, engine=1), p.inverse(Y0, engine=0)) <= 1e-13
    assert rel_l2(p.dense(x, 0, 4, engine=1), p.dense(x, 0, 4, engine=0)) <= 1e-13
    assert rel_l2(p.spectrum(x, engine=0), np.fft.rfft(x, axis=-1)) <= 1e-13
    assert rel_l2(p.spectrum(x, engine=1), np.fft.rfft(x, axis=-1)) <= 1e-13


def test_threshold_rowmedian_bruteforce(plan1k):
    p = plan1k
    rng = np.random.default_rng(91)
    Y = (rng.standard_normal((3, p.ctot)) + 1j * rng.standard_normal((3, p.ctot))) * rng.uniform(0.1, 3, (3, p.ctot))
    out = p.threshold(Y, 3.0)
    nz = 0
    for b in range(3):
        for k, r in enumerate(p.rows):
            y = Y[b, p.row_slice(k)]
            m = np.median(np.abs(y))           # numpy averages the two middle values (R11)
            keep = ~(np.abs(y) < 3.0 * m)
            assert np.array_equal(out[b, p.row_slice(k)], np.where(keep, y, 0))
            nz += keep.sum()
    assert 0 < nz < Y.size


def test_threshold_rowmedian_f32_bitwise(plan1k):
    p = plan1k
    rng = np.random.default_rng(92)
    Y = ((rng.standard_normal((2, p.ctot)) + 1j * rng.standard_normal((2, p.ctot)))).astype(np.complex64)
    out = p.threshold_f32(Y, 3.0)
    for b in range(2):
        for k, r in enumerate(p.rows):
            y = Y[b, p.row_slice(k)]
            re, im = y.real.astype(np.float32), y.imag.astype(np.float32)
            mag = np.sqrt((re * re).astype(np.float32) + (im * im).astype(np.float32)).astype(np.float32)
            s = np.sort(mag)
            m = np.float32(0.5) * np.float32(s[r.M // 2 - 1] + s[r.M // 2])
            t = np.float32(3.0) * m
            expect = np.where(mag < t, np.complex64(0), y)
            assert np.array_equal(out[b, p.row_slice(k)].view(np.uint32), expect.view(np.uint32))


# ---- window families (App. A, A2-A6) and manual grids (:303) ---------------------------

WINDOW_CASES = [("hann", 0.0), ("kaiser", 6.5), ("tukey", 0.4), ("planck", 0.5)]


@pytest.mark.parametrize("name,par", WINDOW_CASES[:3])
def test_window_families_vs_scipy(name, par):
    """A2 / A3 / A4 sampled at j/dk equal scipy's symmetric windows of length 2 dk + 1 (an outside
    library's own formulas: hann 0.5 - 0.5 cos(2 pi n/(L-1)), kaiser I0(beta sqrt(1-(2n/(L-1)-1)^2))/I0(beta),
    tukey with alpha = tapered fraction), normalised to unit energy (Eq. 5 / R3)."""
    sw = pytest.importorskip("scipy.signal.windows")
    ref = {"hann": lambda L: sw.hann(L, sym=True), "kaiser": lambda L: sw.kaiser(L, par),
           "tukey": lambda L: sw.tukey(L, par)}[name]
    p = RefPlan(1024.0, 1024, [4.0, 8.0], 16.0, 400.0, 12, window=name, window_param=par)
    for k, r in enumerate(p.rows):
        w = ref(r.L)
        assert np.abs(p.window(k) - w / np.sqrt(np.sum(w ** 2))).max() <= 1e-14


def test_planck_taper_closed_form_values():
    """A5/A6 (reading R15): with d = 1 - |u|, Z = a/d + a/(d - a): W = 1 on |u| <= 1 - a, W = 1/2 at
    d = a/2 (Z = 0), W = 1/(e^{8/3} + 1) at d = a/4 (Z = 4 - 4/3), W = 0 at |u| = 1; even, non-increasing
    in |u|.  dk = 40 and a = 1/2 put those points on the integer offsets 30 and 35."""
    p = RefPlan(1024.0, 1024, [4.0], 16.0, 400.0, 12, clamp_mode=2, max_window_bins=81,
                window="planck", window_param=0.5)
    k = [i for i, r in enumerate(p.rows) if r.dk == 40][0]
    w = p.window(k)
    raw = w / w[40]                        # centre value is 1 before normalisation
    assert np.all(raw[20:61] == 1.0)       # |j| <= 20 = dk (1 - a)
    assert abs(raw[40 + 30] - 0.5) <= 1e-15 and abs(raw[40 - 30] - 0.5) <= 1e-15
    assert abs(raw[40 + 35] - 1.0 / (np.exp(8.0 / 3.0) + 1.0)) <= 1e-15
    assert raw[0] == 0.0 and raw[80] == 0.0
    assert np.array_equal(raw, raw[::-1])
    assert np.all(np.diff(raw[40:]) <= 0)
    assert abs(np.sum(w ** 2) - 1.0) <= 1e-14      # Eq. 5 / R3


@pytest.mark.parametrize("name,par", WINDOW_CASES)
def test_window_families_round_trip_and_frame_energy(name, par):
    """P4 and P6 hold for any window: exact reconstruction on the cover set (C44-C45 :566-577) and
    sum |Y|^2 = (1/N) sum_f |X|^2 P (C36 :536, one-sided weights)."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12, window=name, window_param=par, clamp_overlap=2.0)
    x = inputs.white_noise(p.N, 61, batch=2)
    Y = p.forward(x, engine=0)
    X = np.fft.rfft(x, axis=-1)
    P, C = p.frame(-1)
    proj = np.fft.irfft(np.where(C[None, :], X, 0), n=p.N, axis=-1)
    assert rel_l2(p.inverse(Y, engine=0), proj) <= 1e-12
    for b in range(2):
        lhs = np.sum(np.abs(Y[b]) ** 2)
        rhs = np.sum(np.abs(X[b]) ** 2 * P) / p.N
        assert abs(lhs - rhs) <= 1e-12 * rhs
    # the forward against the library construction (rfft, windowed band, ifft) for this window
    for k, r in enumerate(p.rows):
        w = p.window(k)
        B = np.zeros(r.M, complex)
        for j in range(-r.dk, r.dk + 1):
            if 0 <= r.kc + j < p.n_bins:
                B[j % r.M] = X[0][r.kc + j] * w[j + r.dk]
        assert rel_l2(Y[0][p.row_slice(k)], np.fft.ifft(B) * np.sqrt(r.M / p.N)) <= 1e-12


def test_manual_frequency_grid():
    """:303 "defined ... manually, by passing a specific list of target frequencies": centre bins
    floor(f T + 1/2) (R2), clamp A7 from the largest gap of the list, round trip exact on the cover set."""
    freqs = [20.0, 30.0, 47.0, 80.0, 150.0, 260.0, 400.0]
    fs, N = 1024.0, 2048
    T = N / fs
    p = RefPlan(fs, N, [4.0, 12.0], 0.0, 0.0, 0, freqs=freqs)
    assert p.n_rows == 2 * len(freqs)
    Lmax = 2 * (int(np.ceil(T * 140.0)) // 2) + 1          # A7 with the largest gap, 400 - 260 = 140 Hz
    for i, r in enumerate(p.rows):
        f = freqs[i % len(freqs)]
        assert r.kc == int(np.floor(f * T + 0.5))
        assert r.L == min(2 * int(np.floor(f * T * np.sqrt(11.0) / r.q)) + 1, Lmax)
    x = inputs.white_noise(N, 62)
    _, C = p.frame(-1)
    proj = np.fft.irfft(np.where(C[None, :], np.fft.rfft(x, axis=-1), 0), n=N, axis=-1)
    assert rel_l2(p.inverse(p.forward(x, engine=1), engine=1), proj) <= 1e-12
    with pytest.raises(ValueError):
        RefPlan(fs, N, [4.0], 0.0, 0.0, 0, freqs=[20.0, 20.0, 30.0])      # not ascending


# ---- multi-Q scan: plane metric and optimal-plane selection ----------------------

def test_plane_energy_is_the_per_plane_frame_energy():
    """metric 0 against C36 (:536) restricted to one plane: sum_{k in plane, n} |Y_k[n]|^2 =
    (1/N) sum_f w_f |X[f]|^2 P_plane[f] ... evaluated with numpy's rfft and the plan's own P_plane."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)
    x = inputs.white_noise(p.N, 81, batch=3)
    vals, best = p.plane_metric(p.forward(x, engine=0), "energy")
    X = np.fft.rfft(x, axis=-1)
    for q in range(p.n_planes):
        Pq, _ = p.frame(q)
        expect = np.sum(np.abs(X) ** 2 * Pq[None, :], axis=-1) / p.N
        assert np.max(np.abs(vals[:, q] - expect) / expect) <= 1e-12
    assert np.array_equal(best, np.argmax(vals, axis=1))


def test_plane_peak_of_a_pure_sinusoid_closed_form():
    """metric 1 against P7's closed form: for x = cos(2 pi k0 n/N) every pixel of row k has
    |Y_k[n]|^2 = (N/M_k) W_k[k0 - kc]^2 / 4, so a plane's peak is the largest such value over its rows, and
    the optimal plane is the one that holds it."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)
    k0 = 93
    x = np.cos(2 * np.pi * k0 * np.arange(p.N) / p.N)
    vals, best = p.plane_metric(p.forward(x, engine=0), "peak")
    expect = np.zeros(p.n_planes)
    for k, r in enumerate(p.rows):
        j = k0 - r.kc
        if abs(j) <= r.dk:
            expect[r.plane] = max(expect[r.plane], (p.N / r.M) * p.window(k)[j + r.dk] ** 2 / 4.0)
    assert np.max(np.abs(vals[0] - expect)) <= 1e-12 * expect.max()
    assert best[0] == int(np.argmax(expect))
    # scaling one segment changes its metrics quadratically and not its choice; selection is per segment
    v2, b2 = p.plane_metric(p.forward(np.stack([x, 3.0 * x]), engine=0), "peak")
    assert np.allclose(v2[1], 9.0 * v2[0], rtol=1e-12) and b2[0] == b2[1] == best[0]


# ---- paper-native layouts: uniform tile length, re-modulation ----------------

@pytest.mark.parametrize("tile_length", [-1, 512])
def test_uniform_tile_length_is_an_upsampled_view_of_the_ragged_layout(tile_length):
    """:127-129: "symmetrically zero padded ... so that all the tiles have the same length".  Zero-padding the
    baseband spectrum only resamples the same band-limited envelope: with M' >= M both powers of two,
    Y'[n M'/M] = sqrt(M/M') Y[n] (the factor is C47's (N M)^{-1/2}), the row energy is unchanged (C48 :592),
    and the round trip is still exact on the cover set."""
    args = (1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)
    p = RefPlan(*args)
    u = RefPlan(*args, tile_length=tile_length)
    Mu = {r.M for r in u.rows}
    assert len(Mu) == 1 and Mu.pop() == (128 if tile_length == -1 else 512)
    assert u.ctot == u.n_rows * u.rows[0].M and [r.offset for r in u.rows] == [i * u.rows[0].M for i in range(u.n_rows)]
    x = inputs.white_noise(p.N, 91)
    Y, Yu = p.forward(x, engine=0)[0], u.forward(x, engine=0)[0]
    for k, (r, ru) in enumerate(zip(p.rows, u.rows)):
        assert (r.kc, r.dk, r.L) == (ru.kc, ru.dk, ru.L)
        a, b = Y[p.row_slice(k)], Yu[u.row_slice(k)]
        step = ru.M // r.M
        assert rel_l2(b[::step], np.sqrt(r.M / ru.M) * a) <= 1e-12
        assert abs(np.sum(np.abs(a) ** 2) - np.sum(np.abs(b) ** 2)) <= 1e-12 * np.sum(np.abs(a) ** 2)
    _, C = u.frame(-1)
    proj = np.fft.irfft(np.where(C[None, :], np.fft.rfft(x, axis=-1), 0), n=p.N, axis=-1)
    assert rel_l2(u.inverse(Yu[None, :], engine=0), proj) <= 1e-12
    with pytest.raises(ValueError):
        RefPlan(*args, tile_length=64)          # shorter than the largest window
    with pytest.raises(ValueError):
        RefPlan(*args, tile_length=384)         # not a power of two


def test_remodulation_gives_samples_of_the_dense_tile():
    """Eq. 10a (:113-117) / P2: sqrt(M/N) e^{2 pi i kc n/M} Y_k[n] = T_k[n N/M], against O-dense (pinned by the
    brute-force convolution P1), in the ragged and in the uniform layout."""
    args = (256.0, 256, [4.0, 8.0], 8.0, 100.0, 7)
    for tl in (0, -1):
        p = RefPlan(*args, tile_length=tl)
        x = inputs.white_noise(p.N, 92)
        R = p.remodulate(p.forward(x, engine=0))[0]
        D = p.dense(x, engine=0)[0]
        for k, r in enumerate(p.rows):
            assert rel_l2(R[p.row_slice(k)], D[k][:: p.N // r.M]) <= 1e-12


# ---- instantaneous frequency (Fig. 5) -------------------------------------------------

def test_instantaneous_frequency_of_a_sinusoid_is_its_frequency():
    """closed form: for x = cos(2 pi k0 n/N) the envelope of every row that sees bin k0 is
    ~ e^{2 pi i (k0 - kc) n/M} (P7), so the phase advances by 2 pi (k0 - kc)/M per sample and
    f_inst = (kc + (k0 - kc))/T = k0/T on the whole row -- the carrier comes back exactly."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)
    k0, T = 93, 1.0
    x = np.cos(2 * np.pi * k0 * np.arange(p.N) / p.N)
    F = p.instantaneous_frequency(p.forward(x, engine=0))[0]
    seen = 0
    for k, r in enumerate(p.rows):
        if abs(k0 - r.kc) < r.dk:          # inside the window, away from its zero end points
            assert np.max(np.abs(F[p.row_slice(k)] - k0 / T)) <= 1e-9
            seen += 1
    assert seen >= 6


def test_instantaneous_frequency_vs_numpy_unwrap():
    """the definition through a library routine: diff(unwrap(angle(Y))) M/(2 pi T) + kc/T for n = 0..M-2,
    and the circular last sample; compared on the circle where a difference sits on the branch cut."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0], 16.0, 400.0, 12)
    x = inputs.white_noise(p.N, 95)
    Y = p.forward(x, engine=0)[0]
    F = p.instantaneous_frequency(Y)[0]
    T = p.N / 1024.0
    for k, r in enumerate(p.rows):
        y = Y[p.row_slice(k)]
        ph = np.unwrap(np.angle(np.concatenate([y, y[:1]])))
        want = np.diff(ph) * r.M / (2 * np.pi * T) + r.kc / T
        d = (F[p.row_slice(k)] - want) * T / r.M           # in turns
        assert np.max(np.abs(d - np.round(d))) <= 1e-9
        assert np.mean(np.round(d) != 0) < 0.01            # only exact branch-cut cases may differ by a turn


def test_gathered_optimal_plane_carries_exactly_the_winning_plane():
    """the composite output of the optimal-selection mode (:329): its energy equals the winning plane's metric,
    its leading C_p entries are that plane's rows in layout order, the padding is zero; a different choice per
    segment gives different rows (selection is per signal)."""
    p = RefPlan(1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12)
    x = inputs.white_noise(p.N, 83, batch=3)
    Y = p.forward(x, engine=0)
    vals, _ = p.plane_metric(Y, "energy")
    best = np.array([2, 0, 1], dtype=np.int32)
    out = p.gather_plane(Y, best)
    sizes = p.plane_sizes()
    assert out.shape == (3, sizes.max())
    for b in range(3):
        q = best[b]
        assert abs(np.sum(np.abs(out[b]) ** 2) - vals[b, q]) <= 1e-12 * vals[b, q]
        rows = [k for k, r in enumerate(p.rows) if r.plane == q]
        first = p.rows[rows[0]].offset
        assert np.array_equal(out[b, :sizes[q]], Y[b, first:first + sizes[q]])
        assert np.all(out[b, sizes[q]:] == 0)


# ---- epsilon-regularised windows and single-tile inversion (Eq. 12-13) -------------

def test_single_tile_inversion_recovers_the_signal():
    """Eq. 13: with the window floored at epsilon (Eq. 12, reading R17) ONE dense tile determines the whole
    signal: x = F^{-1}{F[T_k]/W_k}.  Checked for a low, a middle and a high row, and against the same
    construction through numpy's fft / irfft (library routines)."""
    args = (256.0, 256, [4.0, 8.0], 8.0, 100.0, 7)
    eps = 1e-4
    p = RefPlan(*args, epsilon=eps)
    p0 = RefPlan(*args)
    x = inputs.white_noise(p.N, 97, batch=2)
    for k in (0, p.n_rows // 2, p.n_rows - 1):
        T = p.dense(x, engine=0, row_begin=k, row_end=k + 1)[:, 0, :]
        assert rel_l2(p.dense_invert(T, k), x) <= 1e-10          # conditioning 1/eps on the stop band
        # the tile differs from the plain one only by the epsilon-weighted rest of the spectrum
        T0 = p0.dense(x, engine=0, row_begin=k, row_end=k + 1)[:, 0, :]
        assert 0 < rel_l2(T, T0) < 50 * eps
        r = p.rows[k]
        W = np.full(p.n_bins, eps * r.norm)
        w = p0.window(k) / r.norm                                   # unnormalised window values
        for j in range(-r.dk, r.dk + 1):
            if 0 <= r.kc + j < p.n_bins:
                W[r.kc + j] = max(w[j + r.dk], eps) * r.norm
        Xh = np.fft.fft(T, axis=-1)[:, :p.n_bins] / W[None, :]
        Xh[:, 0] = Xh[:, 0].real
        Xh[:, -1] = Xh[:, -1].real
        assert rel_l2(p.dense_invert(T, k), np.fft.irfft(Xh, n=p.N, axis=-1)) <= 1e-10
    with pytest.raises(ValueError):
        p0.dense_invert(np.zeros((1, p0.N), complex), 0)             # epsilon = 0: undefined


# ---- the paper's output-length options (A22) ------------------------------------------------------------------

def test_output_length_options_closed_forms_and_identities():
    """every row at the same number n of samples, n any integer >= the largest
    window.  Pins: the lengths themselves; a pure sinusoid's closed form at a non-power-of-two n; row energy (C48);
    n = the uniform power-of-two tile gives the uniform-tile layout; a numpy construction; re-sampling between any
    two lengths is exact (Fig. 3); the round trip from the minimal image is Pi_C x."""
    N = 512
    p = RefPlan(512.0, N, [4.0, 8.0], 12.0, 200.0, 9)
    n_std, n_min = p.output_length("standard"), p.output_length("minimal")
    assert n_std == N // 2 + 1 == 257 and n_min == max(r.L for r in p.rows)
    x = inputs.white_noise(N, 81, batch=2)
    for n in (n_min, n_std, 100 if 100 >= n_min else n_min + 7):
        Y = p.forward_length(x, n)
        # row energy is that of the dense tile whatever the length (C48)
        X = np.fft.rfft(x, axis=-1)
        for k, r in enumerate(p.rows):
            w = p.window(k)
            f = np.arange(r.kc - r.dk, r.kc + r.dk + 1)
            ok = (f >= 0) & (f < p.n_bins)
            e = np.sum(np.abs(X[:, f[ok]] * w[None, ok]) ** 2, axis=1) / N
            assert np.allclose(np.sum(np.abs(Y[:, k]) ** 2, axis=1), e, rtol=1e-12)
            # numpy construction: the band placed at j mod n of an n-array, inverse DFT of length n
            B = np.zeros((2, n), complex)
            B[:, (f[ok] - r.kc) % n] = X[:, f[ok]] * w[None, ok]
            assert rel_l2(Y[:, k], np.fft.ifft(B, axis=-1) * n / np.sqrt(N * n)) <= 1e-12
    # closed form (P7 at a length that is no power of two): x = cos(2 pi k0 t / T)
    k0 = 61
    t = np.arange(N)
    Yc = p.forward_length(np.cos(2 * np.pi * k0 * t / N), n_std)[0]
    m = np.arange(n_std)
    for k, r in enumerate(p.rows):
        j = k0 - r.kc
        want = 0.0 * m if abs(j) > r.dk else np.sqrt(N / n_std) * 0.5 * p.window(k)[j + r.dk] * np.exp(2j * np.pi * j * m / n_std)
        assert np.max(np.abs(Yc[k] - want)) <= 1e-13
    # n = the uniform power-of-two tile length: the uniform-tile layout of the plan with tile_length = -1
    pu = RefPlan(512.0, N, [4.0, 8.0], 12.0, 200.0, 9, tile_length=-1)
    Mu = pu.rows[0].M
    assert rel_l2(p.forward_length(x, Mu).reshape(2, -1), pu.forward(x)) <= 1e-12
    # re-sampling is exact in both directions, and composes (Fig. 3: down-sample, up-sample, residual ~ rounding)
    Ymin, Ystd = p.forward_length(x, n_min), p.forward_length(x, n_std)
    assert rel_l2(p.resample(Ymin, n_std), Ystd) <= 1e-12
    assert rel_l2(p.resample(Ystd, n_min), Ymin) <= 1e-12
    assert rel_l2(p.resample(p.resample(Ystd, n_min), n_std), Ystd) <= 1e-12
    # round trip from either image
    _, C = p.frame(-1)
    proj = np.fft.irfft(np.where(C[None, :], np.fft.rfft(x, axis=-1), 0), n=N, axis=-1)
    assert rel_l2(p.inverse_length(Ymin), proj) <= 1e-12 and rel_l2(p.inverse_length(Ystd), proj) <= 1e-12
    for plane in (0, 1):
        _, Cp = p.frame(plane)
        projp = np.fft.irfft(np.where(Cp[None, :], np.fft.rfft(x, axis=-1), 0), n=N, axis=-1)
        assert rel_l2(p.inverse_length(Ystd, plane=plane), projp) <= 1e-12
    # a length below the largest window aliases: refused
    with pytest.raises(AssertionError):
        p.forward_length(x, n_min - 1)


# ---- clusters of active pixels -> binary mask ---------------------------------------------------

def test_cluster_labels_hand_built_masks():
    """4-connectivity, time axis circular, frequency axis not, minimum area, canonical labels (1 + smallest pixel
    index): every rule on a mask small enough to check by eye"""
    m = np.zeros((4, 8), np.uint8)
    m[1, 6:8] = 1; m[1, 0] = 1; m[2, 0] = 1      # wraps around the time edge: pixels 14, 15, 8, 16 -> label 9
    m[0, 3] = 1                                   # a single pixel: label 4
    m[3, 4] = 1; m[2, 5] = 1                      # diagonal neighbours are NOT connected: labels 29 and 22
    L, c = cluster_labels(m, 1)
    want = np.zeros((4, 8), np.int32)
    want[1, 6:8] = 9; want[1, 0] = 9; want[2, 0] = 9; want[0, 3] = 4; want[3, 4] = 29; want[2, 5] = 22
    assert np.array_equal(L[0], want) and c[0] == 4
    L, c = cluster_labels(m, 2)                   # minimum area 2 keeps the 4-pixel cluster only
    assert np.array_equal(L[0], np.where(want == 9, 9, 0)) and c[0] == 1
    # the frequency axis does not wrap: top and bottom rows stay apart
    m = np.zeros((3, 4), np.uint8); m[0, 1] = 1; m[2, 1] = 1
    L, c = cluster_labels(m, 1)
    assert L[0, 0, 1] == 2 and L[0, 2, 1] == 10 and c[0] == 2
    # a full row is one ring; an empty mask has no cluster
    m = np.zeros((2, 5), np.uint8); m[1, :] = 1
    L, c = cluster_labels(m, 1)
    assert np.all(L[0, 1] == 6) and np.all(L[0, 0] == 0) and c[0] == 1
    L, c = cluster_labels(np.zeros((2, 5), np.uint8), 1)
    assert not L.any() and c[0] == 0


@pytest.mark.parametrize("density", [0.2, 0.45, 0.6])
def test_cluster_labels_vs_scipy(density):
    """random masks against an outside library's labelling (scipy.ndimage.label, 4-connectivity); the first and
    last time columns are cleared so that no cluster touches the circular edge, which scipy does not have"""
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(int(density * 100))
    m = (rng.random((3, 24, 40)) < density).astype(np.uint8)
    m[:, :, 0] = 0; m[:, :, -1] = 0
    for min_area in (1, 4):
        L, c = cluster_labels(m, min_area)
        for b in range(3):
            lab, n = ndi.label(m[b])
            want = np.zeros_like(L[b]); kept = 0
            for i in range(1, n + 1):
                idx = np.flatnonzero(lab.ravel() == i)
                if idx.size >= min_area:
                    want.ravel()[idx] = idx.min() + 1; kept += 1
            assert np.array_equal(L[b], want) and c[b] == kept
    # with the edge columns active the circular axis joins clusters scipy keeps apart: check against a rolled copy
    m2 = (rng.random((1, 16, 32)) < 0.4).astype(np.uint8)
    L0, c0 = cluster_labels(m2, 1)
    L1, c1 = cluster_labels(np.roll(m2, 5, axis=2), 1)
    assert c0[0] == c1[0]                                    # the partition does not depend on where the edge is
    P0 = (L0[0][:, :, None, None] == L0[0][None, None, :, :]) & (L0[0] > 0)[:, :, None, None]
    R1 = np.roll(L1[0], -5, axis=1)
    P1 = (R1[:, :, None, None] == R1[None, None, :, :]) & (R1 > 0)[:, :, None, None]
    assert np.array_equal(P0, P1)


def test_cluster_mask_pipeline_isolates_a_burst():
    """threshold -> clusters -> binary mask -> inverse (Fig. 8): a strong sine-Gaussian in weak noise is
    the largest cluster of its plane, and inverting its mask alone gives back most of the burst"""
    N = 2048
    p = RefPlan(2048.0, N, [8.0], 32.0, 800.0, 24, tile_length=-1)
    t = np.arange(N) / 2048.0
    burst = inputs.sine_gaussian(t, 300.0, 12.0, 8.0, 0.5)
    x = 0.05 * inputs.white_noise(N, 88)[0] + burst
    Y = p.forward(x)
    Yt = p.threshold(Y, 3.0)
    L, c = p.cluster(Yt, 0, min_area=6)
    assert c[0] >= 1
    ids, areas = np.unique(L[L > 0], return_counts=True)
    big = int(ids[np.argmax(areas)])
    xr = p.inverse(p.apply_mask(Yt, 0, L, label=big), plane=0)[0]
    assert rel_l2(xr, burst) < 0.2
    # every kept cluster together = the thresholded plane restricted to cluster pixels
    allm = p.apply_mask(Yt, 0, L, label=0)
    assert np.count_nonzero(allm) == np.count_nonzero(L)


# ---- composite filter bank: one window family per plane ---------------------------------------------

def test_composite_bank_is_the_concatenation_of_its_single_window_banks():
    """A23: "scanning not only across varying Quality factors Q ... but also across diverse windowing functions and
    their associated shape parameters ... a composite filter bank concatenates all requested configurations".
    Plane p of the composite bank IS the single-window bank of its (Q, family, parameter): windows, coefficients,
    per-plane frame operator and per-plane inverse; the joint frame operator is the sum; P4 and P6 hold jointly."""
    cfgs = [(8.0, "bisquare", 0.0), (8.0, "hann", 0.0), (8.0, "tukey", 0.5), (16.0, "kaiser", 6.0), (16.0, "planck", 0.4)]
    base = (1024.0, 1024)
    p = RefPlan(*base, [c[0] for c in cfgs], 16.0, 400.0, 12, plane_windows=[(c[1], c[2]) for c in cfgs])
    x = inputs.white_noise(1024, 77, batch=2)
    Y = p.forward(x)
    Pj, Cj = p.frame(-1)
    Psum = np.zeros_like(Pj)
    off = 0
    for q, (Q, w, a) in enumerate(cfgs):
        s1 = RefPlan(*base, [Q], 16.0, 400.0, 12, window=w, window_param=a)
        for k in range(s1.n_rows):
            assert np.array_equal(p.window(q * s1.n_rows + k), s1.window(k))
        assert rel_l2(Y[:, off:off + s1.ctot], s1.forward(x)) <= 1e-14
        Pq, Cq = p.frame(q)
        P1, C1 = s1.frame(-1)
        assert np.array_equal(Cq, C1) and np.allclose(Pq, P1, rtol=1e-14)
        assert rel_l2(p.inverse(Y, plane=q), s1.inverse(Y[:, off:off + s1.ctot])) <= 1e-13
        Psum += Pq
        off += s1.ctot
    assert np.allclose(Pj, Psum, rtol=1e-13)
    X = np.fft.rfft(x, axis=-1)
    tot = np.sum(np.abs(Y) ** 2, axis=1)
    assert np.all(np.abs(tot - np.sum(np.abs(X) ** 2 * Pj[None, :], axis=1) / 1024) <= 1e-13 * tot)
    proj = np.fft.irfft(np.where(Cj[None, :], X, 0), n=1024, axis=-1)
    assert rel_l2(p.inverse(Y), proj) <= 1e-12
