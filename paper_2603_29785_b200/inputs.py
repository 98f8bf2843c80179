"""Seeded synthetic inputs and the BASELINE.json configurations.

This module holds NONE of the method's arithmetic (no window, no Q-transform step): it only makes
strain-like time series and names the plan parameters of each configuration.  It is the one module
both the CUDA path's tests/bench and the CPU oracle's tests use.  NumPy only.

The paper's workloads are real detector data (GW150914, GW200129, an 8740 x 24576 tensor of O3 Virgo
glitches) that is not available here; these generators take their shape --
whitened unit-variance strain, 1-64 s segments at 4096 / 16384 Hz, chirps and glitches at SNR ~10-20 --
and stand in for them (recipe: SURVEY.md section 8(d), restated in DESIGN.md "Input recipe").
All generation is fp64; fp32 configurations round once at the end.
"""
import numpy as np

SEED0 = 260329785

# name -> plan parameters + workload shape.  `calls` lists what the configuration exercises.
CONFIGS = {
    "cfg1": dict(idx=1, fs=4096.0, N=4096, batch=1, dtype="f64", Q=[4.0, 8.0, 16.0], rows=32,
                 fmin=16.0, fmax=1024.0, calls=("forward", "inverse", "dense")),
    "cfg2": dict(idx=2, fs=4096.0, N=32768, batch=64, dtype="f32", Q=[4.0, 8.0, 16.0], rows=48,
                 fmin=20.0, fmax=1800.0, calls=("forward",)),
    "cfg3": dict(idx=3, fs=4096.0, N=16384, batch=256, dtype="f32", Q=[4.0, 8.0, 16.0, 32.0, 64.0],
                 rows=64, fmin=16.0, fmax=2000.0, calls=("forward", "inverse")),
    "cfg4": dict(idx=4, fs=16384.0, N=1048576, batch=16, dtype="f32",
                 Q=[4.0, 8.0, 16.0, 32.0, 64.0], rows=96, fmin=5.0, fmax=8000.0,
                 calls=("forward", "inverse")),
    "cfg5": dict(idx=5, fs=4096.0, N=4096, batch=1024, dtype="f32", Q=[8.0, 16.0, 32.0], rows=64,
                 fmin=16.0, fmax=1800.0, calls=("forward", "threshold", "inverse")),
    # not a BASELINE.json configuration: the shape of the paper's own benchmark (Fig. 6), 6 s
    # at 4096 Hz = 24576 = 3 * 2^13 samples, batches of O(10^3) segments, 62 rows (:343).  The paper does not state
    # the Q, the frequency range or the grid that give its 62 rows: one plane, Q = 8, 20-1800 Hz are stand-ins.
    "paper6s": dict(idx=6, fs=4096.0, N=24576, batch=1024, dtype="f32", Q=[8.0], rows=62,
                    fmin=20.0, fmax=1800.0, calls=("forward", "inverse")),
}

GMSUN_C3 = 4.925490947e-6  # G*Msun/c^3 in seconds


def _rng(cfg_idx, segment):
    return np.random.default_rng(SEED0 + 1000 * cfg_idx + segment)


def sine_gaussian(t, f0, q, amp, t0):
    tau = q / (np.sqrt(2.0) * np.pi * f0)
    return amp * np.exp(-((t - t0) ** 2) / tau ** 2) * np.cos(2.0 * np.pi * f0 * (t - t0))


def newtonian_chirp(t, mchirp_msun, f_start, t_c, f_stop=512.0, taper=0.008):
    """Leading-order inspiral: f(tau) = (1/pi)(5/(256 tau))^(3/8) (G Mc/c^3)^(-5/8),
    phi(tau) = -2 (tau/(5 G Mc/c^3))^(5/8), amplitude ~ f^(2/3); tau = t_c - t.  Unit peak scale;
    the caller rescales after whitening."""
    gm = mchirp_msun * GMSUN_C3
    tau = t_c - t
    tau_start = (5.0 / 256.0) * (np.pi * f_start) ** (-8.0 / 3.0) * gm ** (-5.0 / 3.0)
    tau_stop = (5.0 / 256.0) * (np.pi * f_stop) ** (-8.0 / 3.0) * gm ** (-5.0 / 3.0)
    on = (tau <= tau_start) & (tau >= tau_stop)
    ts = np.where(on, tau, tau_start)
    f = (1.0 / np.pi) * (5.0 / (256.0 * ts)) ** 0.375 * gm ** (-0.625)
    phi = -2.0 * (ts / (5.0 * gm)) ** 0.625
    h = np.where(on, f ** (2.0 / 3.0) * np.cos(phi), 0.0)
    # cosine tapers at both ends
    t_on, t_off = t_c - tau_start, t_c - tau_stop
    win = np.ones_like(t)
    a = (t - t_on) / taper
    win = np.where((a >= 0) & (a < 1), 0.5 * (1 - np.cos(np.pi * a)), win)
    b = (t_off - t) / taper
    win = np.where((b >= 0) & (b < 1), 0.5 * (1 - np.cos(np.pi * b)), win)
    return h * win


def _asd(freqs):
    """A(f) = sqrt(S(f)), S = (40/f)^2 below 40 Hz (f clamped at 1 Hz), 1 above."""
    fc = np.maximum(freqs, 1.0)
    return np.where(fc < 40.0, 40.0 / fc, 1.0)


def _colour_whiten(white, signal, fs):
    """white noise coloured by A(f), signal added, the sum whitened by the same A(f); DC zeroed."""
    n = white.shape[-1]
    A = _asd(np.fft.rfftfreq(n, 1.0 / fs))
    W = np.fft.rfft(white, axis=-1) * A
    if signal is not None:
        W = W + np.fft.rfft(signal, axis=-1)
    W = W / A
    W[..., 0] = 0.0
    return np.fft.irfft(W, n=n, axis=-1)


def _whiten_only(signal, fs):
    n = signal.shape[-1]
    A = _asd(np.fft.rfftfreq(n, 1.0 / fs))
    S = np.fft.rfft(signal, axis=-1) / A
    S[..., 0] = 0.0
    return np.fft.irfft(S, n=n, axis=-1)


def _scaled_injection(sig, fs, norm):
    """scale `sig` so that its whitened version has l2 norm `norm`"""
    w = _whiten_only(sig, fs)
    return sig * (norm / np.sqrt(np.sum(w * w)))


def make_segment(name, segment):
    """One segment of configuration `name` (fp64, length N)."""
    c = CONFIGS[name]
    idx, fs, n = c["idx"], c["fs"], c["N"]
    rng = _rng(idx, segment)
    t = np.arange(n) / fs
    white = rng.standard_normal(n)
    if idx == 1:
        return white + sine_gaussian(t, 200.0, 10.0, 5.0, 0.5)
    if idx == 2 or idx == 6:
        return _colour_whiten(white, None, fs)
    if idx == 3:
        t_c = rng.uniform(1.0, 3.0)
        sig = _scaled_injection(newtonian_chirp(t, 26.0, 20.0, t_c), fs, 15.0)
        return _colour_whiten(white, sig, fs)
    if idx == 4:
        sig = _scaled_injection(newtonian_chirp(t, 26.0, 5.0, 40.0), fs, 15.0)
        sig = sig + _scaled_injection(newtonian_chirp(t, 10.0, 10.0, 41.5), fs, 12.0)
        sig = sig + sine_gaussian(t, 300.0, 8.0, 8.0, 40.7)
        return _colour_whiten(white, sig, fs)
    if idx == 5:
        sig = None
        if segment % 4 == 0:
            f0 = rng.uniform(60.0, 500.0)
            q = rng.uniform(4.0, 20.0)
            sig = sine_gaussian(t, f0, q, 6.0, 0.5)
        return _colour_whiten(white, sig, fs)
    raise KeyError(name)


def make_batch(name, batch=None, first_segment=0, dtype=None):
    """[batch][N] array of configuration `name`; dtype defaults to the configuration's."""
    c = CONFIGS[name]
    batch = c["batch"] if batch is None else batch
    out = np.empty((batch, c["N"]), dtype=np.float64)
    for s in range(batch):
        out[s] = make_segment(name, first_segment + s)
    dt = np.float64 if (dtype or c["dtype"]) == "f64" else np.float32
    return out.astype(dt)


def plan_args(name):
    """(fs, N, Q, fmin, fmax, rows) of a configuration."""
    c = CONFIGS[name]
    return c["fs"], c["N"], list(c["Q"]), c["fmin"], c["fmax"], float(c["rows"])


def white_noise(n, seed, batch=1):
    """plain unit white noise for small pin tests"""
    return np.random.default_rng(SEED0 + seed).standard_normal((batch, n))
