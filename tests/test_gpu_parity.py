"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): coefficients <= 1e-12 (fp64) / 2e-5 (fp32) relative L2 per
segment over the whole coefficient vector; round trip <= 1e-12 (fp64) / 1e-5 (fp32) against the
projection Pi_C x (R9).  For fp32 the oracle consumes the same fp32-rounded input
promoted to double.  The threshold step is bit exact on identical inputs.
"""
import numpy as np
import pytest

from conftest import rel_l2
from oracle.qtam_ref import RefPlan
from paper_2603_29785_b200 import binding, inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}
TOL_RT = {"f64": 1e-12, "f32": 1e-5}


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def worst_segment(got, want):
    return max(rel_l2(got[b], want[b]) for b in range(want.shape[0]))


def worst_row(got, want, plan):
    """largest per-(segment, row) relative L2 error: a short row (M = 4..16 is ~1/300 of a segment's energy)
    cannot hide in the norm of the whole coefficient vector"""
    offs = np.array([int(r.offset) for r in plan.rows], dtype=np.int64)
    num = np.add.reduceat(np.abs(got - want) ** 2, offs, axis=-1)
    den = np.add.reduceat(np.abs(want) ** 2, offs, axis=-1)
    return float(np.sqrt((num / np.maximum(den, 1e-300)).max()))


TOL_ROW = {"f64": 1e-11, "f32": 1e-4}


def make_plans(args, dtype, max_batch, **kw):
    g = binding.Plan(args[0], args[1], args[2], args[3], args[4], args[5], dtype=dtype, max_batch=max_batch, **kw)
    r = RefPlan(args[0], args[1], args[2], args[3], args[4], args[5], **kw)
    return g, r


def pi_c(x64, cover):
    X = np.fft.rfft(x64, axis=-1)
    return np.fft.irfft(np.where(cover[None, :], X, 0), n=x64.shape[-1], axis=-1)


def np_rdt(dtype):
    return np.float64 if dtype == "f64" else np.float32


# ---- small plans, both dtypes, every call ---------------------------------------------------------

SMALL = [
    (1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12.0),      # M 8..64
    (256.0, 256, [4.0, 8.0], 8.0, 100.0, 7.0),                # tiny N
    (4096.0, 8192, [5.0, 20.0], 10.0, 1900.0, 24.0),          # M up to 512
]


@pytest.mark.parametrize("args", SMALL)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ov", [1.0, 2.0])
def test_small_forward_inverse_dense(args, dtype, ov):
    g, r = make_plans(args, dtype, 3, clamp_overlap=ov)
    x = inputs.white_noise(args[1], 100 + args[1], batch=3).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x64, engine=0)
    assert worst_segment(Yg, Yr) <= TOL[dtype]
    assert worst_row(Yg, Yr, r) <= TOL_ROW[dtype]
    # inverse of the ORACLE's coefficients (so the two inverses see identical input)
    Yin = Yr.astype(np.complex128 if dtype == "f64" else np.complex64)
    for plane in range(-1, g.n_planes):
        xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
        xr = r.inverse(Yin.astype(np.complex128), plane=plane, engine=0)
        assert worst_segment(xg, xr) <= TOL[dtype], plane
    # round trip through the GPU only
    xrt = g.inverse(g.forward(dev(x))).cpu().numpy()
    _, C = r.frame(-1)
    assert worst_segment(xrt, pi_c(x64, C)) <= TOL_RT[dtype]
    # dense tiles
    Dg = g.dense(dev(x), 0, g.n_rows).cpu().numpy()
    Dr = r.dense(x64, 0, r.n_rows, engine=1)
    assert worst_segment(Dg.reshape(3, -1), Dr.reshape(3, -1)) <= TOL[dtype]


def test_dense_shift_invariance_on_gpu():
    """the check qtam_dense exists for: integer time shifts commute with the tiles"""
    args = SMALL[0]
    g, _ = make_plans(args, "f64", 1)
    x = inputs.white_noise(args[1], 7)[0]
    D = g.dense(dev(x[None, :])).cpu().numpy()[0]
    for s in (1, 17, 500):
        Ds = g.dense(dev(np.roll(x, s)[None, :])).cpu().numpy()[0]
        assert rel_l2(Ds, np.roll(D, s, axis=-1)) <= 1e-12


# ---- BASELINE configurations -------------------------------------------------------------------------

def test_cfg1_fp64_full():
    name = "cfg1"
    g, r = make_plans(inputs.plan_args(name), "f64", 1)
    x = inputs.make_batch(name)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x, engine=0)
    assert worst_segment(Yg, Yr) <= 1e-12
    worst_row = max(rel_l2(Yg[0, r.row_slice(k)], Yr[0, r.row_slice(k)]) for k in range(r.n_rows))
    assert worst_row <= 1e-11
    for plane in (-1, 0, 1, 2):
        xg = g.inverse(dev(Yr), plane=plane).cpu().numpy()
        assert worst_segment(xg, r.inverse(Yr, plane=plane, engine=0)) <= 1e-12
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x, C)) <= 1e-12
    Dg = g.dense(dev(x)).cpu().numpy()
    Dr = r.dense(x, engine=1)
    assert rel_l2(Dg, Dr) <= 1e-12
    # the injected sine-Gaussian (200 Hz) puts the plane's energy peak in a row near 200 Hz
    e = [np.sum(np.abs(Yg[0, r.row_slice(k)]) ** 2) for k in range(32)]
    assert abs(r.rows[int(np.argmax(e))].f_center - 200.0) < 40.0


@pytest.mark.parametrize("name,nseg,ov", [("cfg2", 3, 1.0), ("cfg2", 2, 2.0), ("cfg3", 4, 1.0),
                                          ("cfg3", 2, 2.0), ("cfg5", 8, 1.0), ("cfg5", 4, 2.0)])
def test_config_fp32_forward_inverse(name, nseg, ov):
    g, r = make_plans(inputs.plan_args(name), "f32", nseg, clamp_overlap=ov)
    x = inputs.make_batch(name, batch=nseg)
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Yg, Yr) <= 2e-5
    assert worst_row(Yg, Yr, r) <= TOL_ROW["f32"]
    Yin = Yr.astype(np.complex64)
    xg = g.inverse(dev(Yin)).cpu().numpy()
    xr = r.inverse(Yin.astype(np.complex128), engine=1)
    assert worst_segment(xg, xr) <= 2e-5
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= 1e-5
    # one plane alone (R10)
    pl = g.n_planes - 1
    xg = g.inverse(dev(Yin), plane=pl).cpu().numpy()
    assert worst_segment(xg, r.inverse(Yin.astype(np.complex128), plane=pl, engine=1)) <= 2e-5


@pytest.mark.parametrize("name,ov,dtype", [("cfg2", 1.0, "f32"), ("cfg3", 1.0, "f32"), ("cfg3", 2.0, "f32"),
                                           ("cfg5", 1.0, "f32"), ("cfg4", 1.0, "f32"), ("cfg5", 1.0, "f64"),
                                           ("cfg1", 1.0, "f64")])
def test_inverse_of_arbitrary_coefficients(name, ov, dtype):
    """The inverse is defined for any coefficient array (masked / edited tiles), not only
    for the image of the forward: rows of different Q-planes that share centre bin and window (the
    clamped rows) carry DIFFERENT values here, so a path that merges such rows must add them -- in both
    precisions (the double-precision rows merge leaders and followers too)."""
    nseg = 1 if name == "cfg4" else 2
    g, r = make_plans(inputs.plan_args(name), dtype, nseg, clamp_overlap=ov)
    keys = [(int(a.kc), int(a.dk), int(a.M)) for a in g.rows]
    assert len(set(keys)) < len(keys), "the plan has no identical rows: the merge would not be exercised"
    rng = np.random.default_rng(20260329 + g.ctot % 1000)
    cdt = np.complex64 if dtype == "f32" else np.complex128
    Yin = (rng.standard_normal((nseg, g.ctot)) + 1j * rng.standard_normal((nseg, g.ctot))).astype(cdt)
    # joint, per plane, joint again: no state may survive in the workspaces between the calls
    for plane in (-1, 0, g.n_planes - 1, -1):
        xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
        xr = r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)
        assert worst_segment(xg, xr) <= TOL[dtype], plane


@pytest.mark.parametrize("log2n", [16, 17, 18, 19])
def test_mid_length_segments(log2n):
    """N = 2^16 .. 2^19: the long real FFT runs as the two-kernel transform of long_fft.cu
    (radix 2 .. 16 across stride 2^14, then 2^14-point transforms in shared memory)."""
    N = 1 << log2n
    args = (16384.0, N, [6.0, 24.0], 30.0, 7000.0, 20.0)
    g, r = make_plans(args, "f32", 1)
    rng = np.random.default_rng(log2n)
    x = rng.standard_normal((1, N)).astype(np.float32)
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    assert worst_segment(Yg, r.forward(x64, engine=1)) <= 2e-5
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= 1e-5


@pytest.mark.parametrize("N,dtype,kw", [(96, "f64", {}), (192, "f32", {}), (1536, "f64", dict(clamp_overlap=2.0)),
                                        (12288, "f32", {}), (24576, "f32", {}), (24576, "f64", {}),
                                        (49152, "f32", dict(tile_length=-1)), (3 * 2 ** 17, "f32", {})])
def test_non_power_of_two_segment_length(N, dtype, kw):
    """N = 3 * 2^k (the paper's own benchmark shape is 6 s at 4096 Hz = 24576 samples; SURVEY
    8(f) item 1): the long transforms take a radix-3 step; every call against the oracle."""
    if N >= 1536:
        args = (4096.0, N, [5.0, 20.0], 40.0 if N == 1536 else 10.0, 0.44 * 4096.0, 14.0)
    else:
        args = (float(N), N, [4.0, 8.0], 5.0, 0.42 * N, 7.0)
    g, r = make_plans(args, dtype, 2, **kw)
    assert [(a.kc, a.dk, a.M, a.offset) for a in g.rows] == [(b.kc, b.dk, b.M, b.offset) for b in r.rows]
    x = inputs.white_noise(N, 300 + N % 97, batch=2).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Yg, Yr) <= TOL[dtype]
    assert worst_row(Yg, Yr, r) <= TOL_ROW[dtype]
    rng = np.random.default_rng(N)
    Yin = (rng.standard_normal((2, g.ctot)) + 1j * rng.standard_normal((2, g.ctot))).astype(Yg.dtype)
    for plane in (-1, 1):
        xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
        assert worst_segment(xg, r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)) <= TOL[dtype], plane
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]
    if N <= 1536:
        Dg = g.dense(dev(x)).cpu().numpy()
        assert worst_segment(Dg.reshape(2, -1), r.dense(x64, engine=1).reshape(2, -1)) <= TOL[dtype]
    two = g.threshold_rowmedian(g.forward(dev(x)), 3.0)
    assert torch.equal(torch.view_as_real(g.forward_threshold(dev(x), 3.0)), torch.view_as_real(two))


def test_paper_benchmark_shape():
    """6 s at 4096 Hz, 62 rows at a batch of 64: forward and round trip"""
    name = "paper6s"
    g, r = make_plans(inputs.plan_args(name), "f32", 64)
    x = inputs.make_batch(name, batch=64)
    x64 = x.astype(np.float64)
    Y = g.forward(dev(x))
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Y.cpu().numpy(), Yr) <= 2e-5 and worst_row(Y.cpu().numpy(), Yr, r) <= TOL_ROW["f32"]
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(Y).cpu().numpy(), pi_c(x64, C)) <= 1e-5


@pytest.mark.parametrize("window,par", [("hann", 0.0), ("kaiser", 6.5), ("tukey", 0.4), ("planck", 0.5)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_window_families(window, par, dtype):
    """App. A, A2-A6: the kernels read the plan's window tables, so every family runs the same path."""
    args = (4096.0, 8192, [5.0, 10.0, 20.0], 10.0, 1900.0, 24.0)
    g, r = make_plans(args, dtype, 2, window=window, window_param=par)
    for k in (0, g.n_rows // 2, g.n_rows - 1):
        assert np.abs(g.window(k) - r.window(k)).max() <= 1e-14 * r.window(k).max()
    x = inputs.white_noise(args[1], 71, batch=2).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    assert worst_segment(Yg, r.forward(x64, engine=1)) <= TOL[dtype]
    rng = np.random.default_rng(72)
    Yin = (rng.standard_normal((2, g.ctot)) + 1j * rng.standard_normal((2, g.ctot))).astype(Yg.dtype)
    for plane in (-1, 1):
        xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
        assert worst_segment(xg, r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)) <= TOL[dtype]
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]


def test_manual_frequency_grid_on_gpu():
    freqs = [20.0, 30.0, 47.0, 80.0, 150.0, 260.0, 400.0, 700.0, 1100.0, 1500.0, 1900.0]
    kw = dict(freqs=freqs)
    g = binding.Plan(4096.0, 16384, [4.0, 12.0, 40.0], 0.0, 0.0, 0.0, dtype="f32", max_batch=2, **kw)
    r = RefPlan(4096.0, 16384, [4.0, 12.0, 40.0], 0.0, 0.0, 0.0, **kw)
    assert [(a.kc, a.dk, a.M, a.offset) for a in g.rows] == [(b.kc, b.dk, b.M, b.offset) for b in r.rows]
    x = inputs.white_noise(16384, 73, batch=2).astype(np.float32)
    x64 = x.astype(np.float64)
    assert worst_segment(g.forward(dev(x)).cpu().numpy(), r.forward(x64, engine=1)) <= 2e-5
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= 1e-5


@pytest.mark.parametrize("name,dtype,nseg", [("cfg3", "f32", 6), ("cfg5", "f64", 5), ("cfg2", "f32", 2)])
@pytest.mark.parametrize("metric", ["energy", "peak"])
def test_plane_metric_and_optimal_plane(name, dtype, nseg, metric):
    """Multi-Q scan selection.  Values to the coefficient tolerance; the selected plane is
    compared through what is unique: where the oracle's best and runner-up are separated by more than the
    tolerance the index must be equal, otherwise the kernel's choice must be one of the near-maximal planes."""
    g, r = make_plans(inputs.plan_args(name), dtype, nseg)
    x = inputs.make_batch(name, batch=nseg, dtype=dtype) if dtype == "f64" else inputs.make_batch(name, batch=nseg)
    x = x.astype(np_rdt(dtype))
    Y = g.forward(dev(x))
    vals, best = g.plane_metric(Y, metric)
    vr, br = r.plane_metric(Y.cpu().numpy().astype(np.complex128), metric)
    tol = 1e-12 if dtype == "f64" else 1e-5
    assert np.max(np.abs(vals.cpu().numpy() - vr) / vr) <= tol
    bg = best.cpu().numpy()
    for b in range(nseg):
        top = np.sort(vr[b])[::-1]
        if top[0] - top[1] > 4 * tol * top[0]:
            assert bg[b] == br[b]
        else:
            assert vr[b][bg[b]] >= top[0] * (1 - 4 * tol)
    # a segment with a strong narrow-band line must prefer a different plane than a broadband one does
    if name == "cfg3":
        t = np.arange(g.N) / 4096.0
        xs = np.stack([np.cos(2 * np.pi * 300.0 * t), inputs.white_noise(g.N, 5)[0]]).astype(np.float32)
        _, b2 = g.plane_metric(g.forward(dev(xs)), "peak")
        _, r2 = r.plane_metric(r.forward(xs.astype(np.float64), engine=1), "peak")
        assert np.array_equal(b2.cpu().numpy(), r2) and r2[0] == g.n_planes - 1


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("tile_length", [-1, 2048])
def test_uniform_tile_layout_and_remodulation(dtype, tile_length):
    """the paper's zero-padded layout (every row the same length, :127-129) and the
    carrier re-modulation back to samples of the dense tile (Eq. 10a)."""
    args = (4096.0, 8192, [5.0, 10.0, 20.0], 10.0, 1900.0, 24.0)
    g, r = make_plans(args, dtype, 2, tile_length=tile_length)
    assert {a.M for a in g.rows} == {b.M for b in r.rows} and len({a.M for a in g.rows}) == 1
    assert g.ctot == r.ctot == g.n_rows * g.rows[0].M
    x = inputs.white_noise(args[1], 75, batch=2).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Y = g.forward(dev(x))
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Y.cpu().numpy(), Yr) <= TOL[dtype]
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(Y).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]
    Yin = Yr.astype(Y.cpu().numpy().dtype)
    R = g.remodulate(dev(Yin)).cpu().numpy()
    assert worst_segment(R, r.remodulate(Yin.astype(np.complex128))) <= TOL[dtype]
    # in place, and in the ragged default layout
    Z = dev(Yin.copy())
    g.remodulate(Z, out=Z)
    assert np.array_equal(Z.cpu().numpy(), R)


def test_remodulation_ragged_layout_cfg3():
    g, r = make_plans(inputs.plan_args("cfg3"), "f32", 3)
    rng = np.random.default_rng(76)
    Yin = (rng.standard_normal((3, g.ctot)) + 1j * rng.standard_normal((3, g.ctot))).astype(np.complex64)
    assert worst_segment(g.remodulate(dev(Yin)).cpu().numpy(), r.remodulate(Yin.astype(np.complex128))) <= 2e-5


def test_cfg5_fp64_variant():
    name = "cfg5"
    g, r = make_plans(inputs.plan_args(name), "f64", 4)
    x = inputs.make_batch(name, batch=4, dtype="f64")
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x, engine=1)
    assert worst_segment(Yg, Yr) <= 1e-12
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x, C)) <= 1e-12


@pytest.mark.parametrize("ov", [1.0, 2.0])
def test_cfg4_long_segment(ov):
    """N = 2^20, rows up to M = 65536 (131072 with overlap 2): the multi-pass paths."""
    name = "cfg4"
    g, r = make_plans(inputs.plan_args(name), "f32", 1, clamp_overlap=ov)
    x = inputs.make_batch(name, batch=1)
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Yg, Yr) <= 2e-5
    assert worst_row(Yg, Yr, r) <= TOL_ROW["f32"]
    Yin = Yr.astype(np.complex64)
    xg = g.inverse(dev(Yin)).cpu().numpy()
    xr = r.inverse(Yin.astype(np.complex128), engine=1)
    assert worst_segment(xg, xr) <= 2e-5
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= 1e-5


# ---- threshold (a4): bit exact --------------------------------------------------------------------------

@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_threshold_bit_exact_on_seeded_coefficients(dtype):
    g, r = make_plans(inputs.plan_args("cfg5"), dtype, 5)
    rng = np.random.default_rng(55)
    cdt = np.complex64 if dtype == "f32" else np.complex128
    Y = ((rng.standard_normal((5, r.ctot)) + 1j * rng.standard_normal((5, r.ctot)))
         * rng.uniform(0.05, 4.0, (5, r.ctot))).astype(cdt)
    Y[1, r.row_slice(3)] = 0            # an all-zero row: median 0, nothing is < 0
    Y[2, r.row_slice(5)] = 1 + 1j       # a constant row
    got = g.threshold_rowmedian(dev(Y).clone(), 3.0).cpu().numpy()
    want = r.threshold_f32(Y, 3.0) if dtype == "f32" else r.threshold(Y, 3.0)
    bits = np.uint32 if dtype == "f32" else np.uint64
    assert np.array_equal(got.view(bits), want.view(bits))
    assert 0 < np.count_nonzero(got) < got.size
    # a constant row: every magnitude equals the median m, and m < 3m, so the whole row is zeroed
    assert not got[2, r.row_slice(5)].any()
    assert not got[1, r.row_slice(3)].any()


def test_cfg5_denoise_pipeline_fp32():
    """forward -> zero |c| < 3 x row median -> inverse, each stage against the oracle on the
    oracle's own upstream output, plus the whole chain."""
    name = "cfg5"
    nseg = 8
    g, r = make_plans(inputs.plan_args(name), "f32", nseg)
    x = inputs.make_batch(name, batch=nseg)
    x64 = x.astype(np.float64)
    Yr32 = r.forward(x64, engine=1).astype(np.complex64)
    want_thr = r.threshold_f32(Yr32, 3.0)
    got_thr = g.threshold_rowmedian(dev(Yr32).clone(), 3.0).cpu().numpy()
    assert np.array_equal(got_thr.view(np.uint32), want_thr.view(np.uint32))
    xg = g.inverse(dev(want_thr)).cpu().numpy()
    xr = r.inverse(want_thr.astype(np.complex128), engine=1)
    assert worst_segment(xg, xr) <= 2e-5
    # whole chain on the GPU; a coefficient within rounding of the threshold may flip, so compare
    # the masks' agreement and the outputs loosely
    Yg = g.forward(dev(x))
    g.threshold_rowmedian(Yg, 3.0)
    mask_g = (Yg.cpu().numpy() != 0)
    mask_r = (want_thr != 0)
    assert np.mean(mask_g != mask_r) < 1e-4
    xchain = g.inverse(Yg).cpu().numpy()
    assert worst_segment(xchain, xr) <= 5e-3
    kept = mask_r.mean()
    # Rayleigh magnitudes: P(|c| > 3 median) = 2^-9 ~ 0.2 % for pure noise, more where a glitch sits
    assert 1e-3 < kept < 0.05


# ---- edge cases and properties -------------------------------------------------------------------------

def test_empty_batch_and_batch_limit():
    g, _ = make_plans(SMALL[0], "f32", 2)
    x = torch.zeros((0, g.N), dtype=torch.float32, device="cuda")
    out = torch.empty((0, g.ctot), dtype=torch.complex64, device="cuda")
    assert binding.lib().qtam_forward(g._h, x.data_ptr() or 16, 0, out.data_ptr() or 16, None) == 0
    big = torch.zeros((3, g.N), dtype=torch.float32, device="cuda")
    with pytest.raises(binding.QtamError) as e:
        g.forward(big)
    assert e.value.code == 1


def test_inputs_are_not_modified_and_output_fully_written():
    g, r = make_plans(inputs.plan_args("cfg3"), "f32", 2)
    x = dev(inputs.make_batch("cfg3", batch=2))
    x0 = x.clone()
    out = torch.full((2, g.ctot), float("nan"), dtype=torch.complex64, device="cuda")
    g.forward(x, out=out)
    assert torch.equal(x, x0)
    assert not torch.isnan(out.real).any() and not torch.isnan(out.imag).any()
    c0 = out.clone()
    xo = torch.full((2, g.N), float("nan"), dtype=torch.float32, device="cuda")
    g.inverse(out, out=xo)
    assert torch.equal(out, c0) and not torch.isnan(xo).any()


def _frame_energy_err(Y, x64, r, N):
    """P6 on every segment: sum|Y|^2 = (1/N) sum_f |X[f]|^2 P[f]"""
    P, _ = r.frame(-1)
    X = np.fft.rfft(x64, axis=-1)
    want = (np.abs(X) ** 2 * P[None, :]).sum(axis=1) / N
    got = (Y.abs().double() ** 2).sum(dim=1).cpu().numpy()
    return float(np.max(np.abs(got - want) / want))


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5"])
def test_full_batch_every_segment_against_the_oracle(name):
    """BASELINE configs 2-5 at their full batch, in the launch configuration bench.py times: EVERY segment is
    compared with the oracle element by element -- the forward on the same input, the inverse (where the
    configuration calls it) on the oracle's coefficients -- with a bound on the whole vector of every segment
    and on every single row; then the round trip, the frame-energy identity P6 and linearity P5 as extras."""
    cfg = inputs.CONFIGS[name]
    B = cfg["batch"]
    g, r = make_plans(inputs.plan_args(name), "f32", B)
    x = inputs.make_batch(name, batch=B)
    dx = dev(x)
    Y = g.forward(dx)
    xo = g.inverse(Y) if "inverse" in cfg["calls"] else None
    Yin_dev = torch.empty_like(Y)
    chunk = 4 if name == "cfg4" else 64
    worst = worst_r = 0.0
    for b0 in range(0, B, chunk):
        b1 = min(B, b0 + chunk)
        Yr = r.forward(x[b0:b1].astype(np.float64), engine=1)
        Yg = Y[b0:b1].cpu().numpy()
        worst = max(worst, worst_segment(Yg, Yr))
        worst_r = max(worst_r, worst_row(Yg, Yr, r))
        Yin_dev[b0:b1] = dev(Yr.astype(np.complex64))
    assert worst <= 2e-5 and worst_r <= TOL_ROW["f32"], (worst, worst_r)
    assert _frame_energy_err(Y, x.astype(np.float64), r, g.N) <= 1e-5
    a, b = 0.7, -1.9
    h = min(8, B // 2)
    comb = g.forward((a * dx[:h] + b * dx[h:2 * h]).contiguous())
    assert rel_l2(comb.cpu().numpy(), (a * Y[:h] + b * Y[h:2 * h]).cpu().numpy()) <= 1e-5
    if xo is None:
        return
    # the inverse of the ORACLE's coefficients (rounded to complex64), every segment, at the full batch
    xg = g.inverse(Yin_dev).cpu().numpy()
    worst = 0.0
    for b0 in range(0, B, chunk):
        b1 = min(B, b0 + chunk)
        xr = r.inverse(Yin_dev[b0:b1].cpu().numpy().astype(np.complex128), engine=1)
        worst = max(worst, worst_segment(xg[b0:b1], xr))
    assert worst <= 2e-5, worst
    _, C = r.frame(-1)
    assert worst_segment(xo.cpu().numpy(), pi_c(x.astype(np.float64), C)) <= 1e-5


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_cfg5_denoise_chain_full_batch(dtype):
    """BASELINE config 5 (complex64 plus the fp64 variant) at its full batch of 1024 segments, as bench.py
    launches it: forward (every segment, every row), threshold bit for bit on the kernel's own coefficients
    (every segment), inverse of the thresholded coefficients (every segment), and the fused
    forward+threshold call = the two calls."""
    name = "cfg5"
    B = inputs.CONFIGS[name]["batch"]
    g, r = make_plans(inputs.plan_args(name), dtype, B)
    x = inputs.make_batch(name, batch=B, dtype=dtype).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Y = g.forward(dev(x))
    Yh = Y.cpu().numpy()
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Yh, Yr) <= TOL[dtype]
    assert worst_row(Yh, Yr, r) <= TOL_ROW[dtype]
    assert _frame_energy_err(Y, x64, r, g.N) <= (1e-5 if dtype == "f32" else 1e-12)
    fused = g.forward_threshold(dev(x), 3.0)
    g.threshold_rowmedian(Y, 3.0)
    assert torch.equal(torch.view_as_real(fused), torch.view_as_real(Y))
    Yt = Y.cpu().numpy()
    want_thr = r.threshold_f32(Yh, 3.0) if dtype == "f32" else r.threshold(Yh, 3.0)
    bits = np.uint32 if dtype == "f32" else np.uint64
    assert np.array_equal(Yt.view(bits), want_thr.view(bits))
    kept = float((Yt != 0).mean())
    assert 1e-3 < kept < 0.05
    xg = g.inverse(Y).cpu().numpy()
    xr = r.inverse(want_thr.astype(np.complex128), engine=1)
    assert worst_segment(xg, xr) <= TOL[dtype]


@pytest.mark.parametrize("name,dtype", [("cfg3", "f32"), ("cfg1", "f64"), ("cfg2", "f32")])
def test_instantaneous_frequency(name, dtype):
    """PAPER.md:176 / Fig. 5.  The phase difference is compared on the circle (a value on the branch cut may
    come out as +pi or -pi: both are the same angle), in turns per sample: |d - round(d)| small."""
    nseg = 2
    g, r = make_plans(inputs.plan_args(name), dtype, nseg)
    x = inputs.make_batch(name, batch=nseg).astype(np_rdt(dtype))
    Y = g.forward(dev(x))
    F = g.instantaneous_frequency(Y).cpu().numpy().astype(np.float64)
    Fr = r.instantaneous_frequency(Y.cpu().numpy().astype(np.complex128))
    T = g.N / inputs.CONFIGS[name]["fs"]
    tol = 1e-11 if dtype == "f64" else 2e-5
    for k, row in enumerate(r.rows):
        sl = slice(row.offset, row.offset + row.M)
        d = (F[:, sl] - Fr[:, sl]) * T / row.M                    # turns per sample
        assert np.max(np.abs(d - np.round(d))) <= tol, k
    # the chirp / sinusoid check of the closed form on the GPU: a pure tone reads back its own frequency
    t = np.arange(g.N) / inputs.CONFIGS[name]["fs"]
    k0 = 300
    tone = np.cos(2 * np.pi * (k0 / T) * t)[None, :].astype(np_rdt(dtype))
    Ft = g.instantaneous_frequency(g.forward(dev(np.repeat(tone, nseg, axis=0)))).cpu().numpy()
    hit = [k for k, row in enumerate(r.rows) if abs(k0 - row.kc) < row.dk // 2]
    assert hit
    for k in hit:
        row = r.rows[k]
        assert np.max(np.abs(Ft[0, row.offset:row.offset + row.M] - k0 / T)) <= (1e-6 if dtype == "f64" else 2e-2)


def test_forward_inverse_under_cuda_graph_capture():
    """The calls never allocate or synchronise (include/qtam.h), so a step can be captured into a CUDA graph
    and replayed; the replay on new input contents equals the eager result bit for bit."""
    name = "cfg3"
    nseg = 4
    g, _ = make_plans(inputs.plan_args(name), "f32", nseg)
    x0 = dev(inputs.make_batch(name, batch=nseg))
    x1 = dev(inputs.make_batch(name, batch=nseg, first_segment=nseg))
    xin = x0.clone()
    Y = torch.empty((nseg, g.ctot), dtype=torch.complex64, device="cuda")
    out = torch.empty_like(xin)
    vals = None
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        g.forward(xin, out=Y); g.inverse(Y, out=out)          # warm-up outside the capture
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        g.forward(xin, out=Y)
        g.inverse(Y, out=out)
    for src in (x1, x0):
        xin.copy_(src)
        graph.replay()
        torch.cuda.synchronize()
        got_Y, got_x = Y.clone(), out.clone()
        ref_Y = g.forward(src)
        ref_x = g.inverse(ref_Y)
        assert torch.equal(got_Y, ref_Y) and torch.equal(got_x, ref_x)


@pytest.mark.parametrize("name,dtype,nseg", [("cfg5", "f32", 16), ("cfg3", "f32", 3), ("cfg2", "f32", 2), ("cfg5", "f64", 3),
                                             ("cfg5", "f32", 1), ("cfg4", "f32", 1)])
def test_forward_threshold_fused_equals_the_two_calls(name, dtype, nseg):
    """qtam_forward_threshold = qtam_forward then qtam_threshold_rowmedian, bit for bit (the decisions are taken
    on the same binary32 values, in registers instead of after a round trip through memory)."""
    g, _ = make_plans(inputs.plan_args(name), dtype, nseg)
    x = dev(inputs.make_batch(name, batch=nseg).astype(np_rdt(dtype)))
    two = g.threshold_rowmedian(g.forward(x), 3.0)
    one = g.forward_threshold(x, 3.0)
    assert torch.equal(torch.view_as_real(one), torch.view_as_real(two))
    assert 0 < (one != 0).float().mean().item() < 0.2


def _random_plan_cases():
    """seeded sweep over plan shapes: segment lengths 2^8..2^17, 1-4 planes, clamp settings, window families,
    tile-length modes, bins-per-octave grids -- the dispatch takes different kernels for different shapes"""
    rng = np.random.default_rng(20260329785 % (2 ** 32))
    cases = []
    for i in range(14):
        log2n = int(rng.integers(8, 18))
        N = 1 << log2n
        fs = float(rng.choice([1024.0, 4096.0, 16384.0]))
        nq = int(rng.integers(1, 5))
        Q = sorted(float(q) for q in rng.uniform(3.4, 60.0, size=nq))
        fmax = float(rng.uniform(0.2, 0.49)) * fs
        T = N / fs
        fmin = max(float(rng.uniform(2.0, 30.0)) * max(Q) / (np.sqrt(11.0) * T), 2.0 / T)   # half-width >= 1 bin
        if fmin >= 0.5 * fmax:
            fmin = 0.25 * fmax
        kw = dict(clamp_overlap=float(rng.choice([1.0, 1.5, 2.0])))
        mode = int(rng.integers(0, 4))
        if mode == 1:
            kw["window"], kw["window_param"] = "tukey", float(rng.uniform(0.2, 0.9))
        elif mode == 2:
            kw["window"], kw["window_param"] = "kaiser", float(rng.uniform(2.0, 9.0))
        elif mode == 3:
            kw["tile_length"] = -1
        if rng.integers(0, 3) == 0:
            kw["rows_are_bins_per_octave"] = 1
            spacing = float(rng.integers(3, 12))
        else:
            spacing = float(rng.integers(5, 40))
        cases.append((i, fs, N, Q, fmin, fmax, spacing, "f64" if i % 3 == 2 else "f32", kw))
    return cases


@pytest.mark.parametrize("case", _random_plan_cases(), ids=lambda c: f"case{c[0]}-N{c[2]}-{c[7]}")
def test_random_plan_shapes(case):
    i, fs, N, Q, fmin, fmax, spacing, dtype, kw = case
    try:
        r = RefPlan(fs, N, Q, fmin, fmax, spacing, **kw)
    except ValueError:
        with pytest.raises(binding.QtamError):
            binding.Plan(fs, N, Q, fmin, fmax, spacing, dtype=dtype, max_batch=2, **kw)
        return
    g = binding.Plan(fs, N, Q, fmin, fmax, spacing, dtype=dtype, max_batch=2, **kw)
    assert [(a.kc, a.dk, a.M, a.offset) for a in g.rows] == [(b.kc, b.dk, b.M, b.offset) for b in r.rows]
    x = inputs.white_noise(N, 1000 + i, batch=2).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    Y = g.forward(dev(x))
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Y.cpu().numpy(), Yr) <= TOL[dtype]
    assert worst_row(Y.cpu().numpy(), Yr, r) <= TOL_ROW[dtype]
    rng = np.random.default_rng(2000 + i)
    Yin = (rng.standard_normal((2, g.ctot)) + 1j * rng.standard_normal((2, g.ctot))).astype(Y.cpu().numpy().dtype)
    for plane in (-1, g.n_planes - 1):
        xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
        xr = r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)
        assert worst_segment(xg, xr) <= TOL[dtype], plane
    _, C = r.frame(-1)
    assert worst_segment(g.inverse(Y).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]
    two = g.threshold_rowmedian(g.forward(dev(x)), 2.5)
    one = g.forward_threshold(dev(x), 2.5)
    assert torch.equal(torch.view_as_real(one), torch.view_as_real(two))


@pytest.mark.parametrize("name,dtype", [("cfg3", "f32"), ("cfg5", "f64")])
def test_gather_of_the_optimal_plane(name, dtype):
    nseg = 5
    g, r = make_plans(inputs.plan_args(name), dtype, nseg)
    x = inputs.make_batch(name, batch=nseg).astype(np_rdt(dtype))
    Y = g.forward(dev(x))
    _, best = g.plane_metric(Y, "peak")
    out = g.gather_plane(Y, best).cpu().numpy()
    want = r.gather_plane(Y.cpu().numpy().astype(np.complex128), best.cpu().numpy())
    assert out.shape == want.shape and np.array_equal(out.astype(np.complex128), want)     # a copy: bit exact
    forced = torch.tensor([i % g.n_planes for i in range(nseg)], dtype=torch.int32, device="cuda")
    out2 = g.gather_plane(Y, forced).cpu().numpy()
    assert np.array_equal(out2.astype(np.complex128), r.gather_plane(Y.cpu().numpy().astype(np.complex128), forced.cpu().numpy()))


@pytest.mark.parametrize("dtype,eps,tol", [("f64", 1e-5, 1e-9), ("f32", 1e-2, 2e-4)])
def test_epsilon_windows_and_single_tile_inversion(dtype, eps, tol):
    """Eq. 12-13 (:140-148): dense tiles with the epsilon-floored window against the oracle, and the whole signal
    back from ONE tile by spectral division (errors of the tile are amplified by up to 1/epsilon, hence the
    tolerances)."""
    args = (1024.0, 1024, [4.0, 8.0, 16.0], 16.0, 400.0, 12.0)
    g, r = make_plans(args, dtype, 2, epsilon=eps)
    x = inputs.white_noise(args[1], 99, batch=2).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    for k in (1, g.n_rows // 2, g.n_rows - 1):
        T = g.dense(dev(x), row_begin=k, row_end=k + 1)
        Tr = r.dense(x64, row_begin=k, row_end=k + 1, engine=1)
        assert worst_segment(T.cpu().numpy()[:, 0, :], Tr[:, 0, :]) <= TOL[dtype]
        xg = g.dense_invert(T[:, 0, :].contiguous(), k).cpu().numpy()
        assert worst_segment(xg, x64) <= tol
        # against the oracle's inversion of the oracle's tile
        assert worst_segment(xg, r.dense_invert(Tr[:, 0, :], k)) <= tol
    g0, _ = make_plans(args, dtype, 2)
    with pytest.raises(binding.QtamError):
        g0.dense_invert(torch.zeros((2, args[1]), dtype=torch.complex128 if dtype == "f64" else torch.complex64, device="cuda"), 0)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("mode", ["minimal", "standard", 300])
def test_output_length_options(dtype, mode):
    """The paper's output-resolution options: [rows][n] images at a length n
    that is no power of two, the inverse from such an image, and the re-sampling to / from the standard length
    (Fig. 3) -- against the oracle's naive sums."""
    args = (512.0, 512, [4.0, 8.0], 12.0, 200.0, 9.0)
    g, r = make_plans(args, dtype, 3)
    g.close()
    g = binding.Plan(*args[:5], args[5], dtype=dtype, max_batch=3, out_length=mode)
    n = g.output_length()
    assert n == (r.output_length(mode) if isinstance(mode, str) else mode)
    assert g.output_length("standard") == 257 and g.output_length("minimal") == r.output_length("minimal")
    x = inputs.white_noise(512, 91, batch=3).astype(np_rdt(dtype))
    x64 = x.astype(np.float64)
    img = g.forward_length(dev(x))
    want = r.forward_length(x64, n, engine=1)
    assert worst_segment(img.cpu().numpy().reshape(3, -1), want.reshape(3, -1)) <= TOL[dtype]
    # inverse of the oracle's image, joint and one plane; round trip through the GPU
    cdt = np.complex64 if dtype == "f32" else np.complex128
    for plane in (-1, 1):
        xg = g.inverse_length(dev(want.astype(cdt)), plane=plane).cpu().numpy()
        assert worst_segment(xg, r.inverse_length(want.astype(cdt).astype(np.complex128), plane=plane, engine=1)) <= TOL[dtype]
    _, C = r.frame(-1)
    assert worst_segment(g.inverse_length(img).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]
    # up-sampling to the standard length and back
    up = g.resample(img, to_standard=True)
    assert up.shape[-1] == 257
    assert worst_segment(up.cpu().numpy().reshape(3, -1), r.forward_length(x64, 257, engine=1).reshape(3, -1)) <= 4 * TOL[dtype]
    back = g.resample(up, to_standard=False)
    assert worst_segment(back.cpu().numpy().reshape(3, -1), want.reshape(3, -1)) <= 4 * TOL[dtype]
    g0 = binding.Plan(*args[:5], args[5], dtype=dtype, max_batch=3)
    with pytest.raises(ValueError):
        g0.forward_length(dev(x))


def test_output_length_at_the_papers_shape():
    """6 s at 4096 Hz (N = 24576): the 62 x 669-like minimal image and its 62 x 12289 standard one (:343)"""
    name = "paper6s"
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
    g = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype="f32", max_batch=2, out_length="minimal")
    r = RefPlan(fs, N, Q, fmin, fmax, rows)
    n = g.output_length()
    assert n == r.output_length("minimal") and g.output_length("standard") == 12289 and g.n_rows == 62
    x = inputs.make_batch(name, batch=2)
    img = g.forward_length(dev(x))
    want = r.forward_length(x.astype(np.float64), n, engine=1)
    assert worst_segment(img.cpu().numpy().reshape(2, -1), want.reshape(2, -1)) <= 2e-5
    up = g.resample(img, to_standard=True).cpu().numpy()
    k = 40
    w12289 = r.forward_length(x[:1].astype(np.float64), 12289, engine=1)
    assert rel_l2(up[0, k], w12289[0, k]) <= 1e-4 and rel_l2(up[0], w12289[0]) <= 1e-4


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_clusters_and_masks(dtype):
    """threshold -> clusters -> binary mask -> inverse: labels and counts equal the oracle's flood fill
    exactly (canonical numbering), on the thresholded transform of bursts in noise and on random patterns; the mask
    of a cluster and its inverse against the oracle"""
    N = 4096
    args = (4096.0, N, [6.0, 12.0], 32.0, 1600.0, 24.0)
    nseg = 3
    g, r = make_plans(args, dtype, nseg, tile_length=-1)
    t = np.arange(N) / 4096.0
    x = 0.3 * inputs.white_noise(N, 97, batch=nseg)
    x[0] += inputs.sine_gaussian(t, 300.0, 10.0, 6.0, 0.4) + inputs.sine_gaussian(t, 900.0, 20.0, 5.0, 0.7)
    x[1] += inputs.sine_gaussian(t, 150.0, 6.0, 8.0, 0.999)          # wraps around the circular time axis
    x = x.astype(np_rdt(dtype))
    Y = g.forward_threshold(dev(x), 2.5)
    Yh = Y.cpu().numpy()
    cdt = torch.complex64 if dtype == "f32" else torch.complex128
    for plane in (0, 1):
        for min_area in (1, 5):
            L, c = g.cluster(Y, plane, min_area)
            Lr, cr = r.cluster(Yh, plane, min_area)
            assert np.array_equal(L.cpu().numpy().reshape(Lr.shape), Lr) and np.array_equal(c.cpu().numpy(), cr)
            assert cr.max() >= 1
    plane = 1
    L, c = g.cluster(Y, plane, 5)
    Lr, _ = r.cluster(Yh, plane, 5)
    ids, areas = np.unique(Lr[0][Lr[0] > 0], return_counts=True)
    big = int(ids[np.argmax(areas)])
    for label in (big, 0):
        Mg = g.mask(Y, plane, L, label)
        Mr = r.apply_mask(Yh, plane, Lr, label)
        assert np.array_equal(Mg.cpu().numpy(), Mr)
        Yc = Y.clone()                                   # in place: qtam.h allows d_out == d_coef
        g.mask(Yc, plane, L, label, out=Yc)
        assert torch.equal(Yc, Mg)
        xg = g.inverse(Mg, plane=plane).cpu().numpy()
        assert worst_segment(xg, r.inverse(Mr.astype(np.complex128), plane=plane, engine=1)) <= TOL[dtype] * 10
    # random patterns at several densities (most clusters merge into a few snakes around 0.5-0.6)
    rng = np.random.default_rng(5)
    for density in (0.15, 0.45, 0.6, 0.95):
        Z = torch.zeros((nseg, g.ctot), dtype=cdt, device="cuda")
        sl, R, M = r.plane_slice(0)
        pat = (rng.random((nseg, R * M)) < density)
        Z[:, sl] = torch.from_numpy(pat.astype(np.complex64 if dtype == "f32" else np.complex128)).cuda()
        L, c = g.cluster(Z, 0, 3)
        Lr, cr = r.cluster(Z.cpu().numpy(), 0, 3)
        assert np.array_equal(L.cpu().numpy().reshape(Lr.shape), Lr) and np.array_equal(c.cpu().numpy(), cr)
    # a plan in the ragged layout has no image to label
    g0, _ = make_plans(args, dtype, nseg)
    with pytest.raises(ValueError):
        g0.cluster(g0.forward(dev(x)), 0)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_composite_bank_with_a_window_family_per_plane(dtype):
    """A23: the planes of one bank differ in window family and shape parameter as well as in Q.  Planes
    0-2 share Q = 8 (same centre bins and half-widths, different windows: such rows must NOT be merged), planes 3-4
    share Q and window (identical rows under the clamp: merged).  Long rows included (N = 2^16)."""
    cfgs = [(8.0, "bisquare", 0.0), (8.0, "hann", 0.0), (8.0, "tukey", 0.5), (16.0, "kaiser", 6.0), (16.0, "kaiser", 6.0)]
    for N, fs in ((8192, 4096.0), (65536, 16384.0)):
        args = (fs, N, [c[0] for c in cfgs], 20.0, 0.44 * fs, 20.0)
        kw = dict(plane_windows=[(c[1], c[2]) for c in cfgs])
        g, r = make_plans(args, dtype, 2, **kw)
        for k in range(0, g.n_rows, 7):
            assert np.abs(g.window(k) - r.window(k)).max() <= 1e-14 * r.window(k).max()
        x = inputs.white_noise(N, 120, batch=2).astype(np_rdt(dtype))
        x64 = x.astype(np.float64)
        Yg = g.forward(dev(x)).cpu().numpy()
        Yr = r.forward(x64, engine=1)
        assert worst_segment(Yg, Yr) <= TOL[dtype] and worst_row(Yg, Yr, r) <= TOL_ROW[dtype]
        rng = np.random.default_rng(121)
        Yin = (rng.standard_normal((2, g.ctot)) + 1j * rng.standard_normal((2, g.ctot))).astype(Yg.dtype)
        for plane in (-1, 1, 4, -1):
            xg = g.inverse(dev(Yin), plane=plane).cpu().numpy()
            assert worst_segment(xg, r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)) <= TOL[dtype], plane
        _, C = r.frame(-1)
        assert worst_segment(g.inverse(g.forward(dev(x))).cpu().numpy(), pi_c(x64, C)) <= TOL_RT[dtype]


# ---- long rows as a dataflow of work items (rows_split.cu) ------------------------------------------------------------

def test_long_rows_partial_batches_and_two_plans_at_once():
    """Rows of 2^15 / 2^16 points run as work items popped from a counter, with completion counts between the
    stages (rows_split.cu).  The schedule must not depend on how many CTAs are resident: two plans running at the
    same time on two streams (each takes part of the SMs) give what they give alone; a plan sized for a larger batch
    works on a smaller one, call after call (counters and partial sums are reset by every call)."""
    args_a = (16384.0, 1 << 19, [4.0, 8.0], 5.0, 8000.0, 32.0)
    args_b = (16384.0, 1 << 19, [4.0, 6.0, 12.0], 6.0, 7900.0, 24.0)
    ga, ra = make_plans(args_a, "f32", 3)
    gb, _ = make_plans(args_b, "f32", 3)
    assert max(int(r.M) for r in ga.rows) >= 1 << 15 and max(int(r.M) for r in gb.rows) >= 1 << 15
    rng = np.random.default_rng(77)
    x = rng.standard_normal((3, 1 << 19)).astype(np.float32)
    dx = dev(x)
    # alone, full batch and a partial one, twice
    Ya = ga.forward(dx)
    Yr = ra.forward(x[:1].astype(np.float64), engine=1)
    assert worst_segment(Ya[:1].cpu().numpy(), Yr) <= 2e-5
    for nb in (1, 2, 3, 2):
        Yp = ga.forward(dx[:nb])
        assert torch.equal(Yp, Ya[:nb])
    xa = ga.inverse(Ya)
    xr = ra.inverse(Ya[:1].cpu().numpy().astype(np.complex128), engine=1)
    assert worst_segment(xa[:1].cpu().numpy(), xr) <= 2e-5
    for nb in (2, 1, 3):
        assert torch.equal(ga.inverse(Ya[:nb]), xa[:nb])
    Yb = gb.forward(dx)
    xb = gb.inverse(Yb)
    torch.cuda.synchronize()
    # the two plans at once on two streams, several rounds
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(s1):
            Ya2 = ga.forward(dx); xa2 = ga.inverse(Ya2)
        with torch.cuda.stream(s2):
            Yb2 = gb.forward(dx); xb2 = gb.inverse(Yb2)
        s1.synchronize(); s2.synchronize()
        assert torch.equal(Ya2, Ya) and torch.equal(Yb2, Yb)
        assert torch.equal(xa2, xa) and torch.equal(xb2, xb)
    ga.close(); gb.close()


def test_longest_segment_without_long_rows():
    """N = 2^20 with rows of at most 2^14 points: no residue-sorted spectrum, so the long transforms take the two-pass
    path whose second pass writes with stride 64 (long_fft.cu), not the residue-order one of config 4."""
    args = (16384.0, 1 << 20, [200.0], 2000.0, 7000.0, 24.0)
    g, r = make_plans(args, "f32", 1)
    assert max(int(a.M) for a in g.rows) <= 1 << 14
    x = np.random.default_rng(5).standard_normal((1, 1 << 20)).astype(np.float32)
    x64 = x.astype(np.float64)
    Yg = g.forward(dev(x)).cpu().numpy()
    Yr = r.forward(x64, engine=1)
    assert worst_segment(Yg, Yr) <= 2e-5 and worst_row(Yg, Yr, r) <= TOL_ROW["f32"]
    xg = g.inverse(dev(Yr.astype(np.complex64))).cpu().numpy()
    assert worst_segment(xg, r.inverse(Yr.astype(np.complex64).astype(np.complex128), engine=1)) <= 2e-5
    g.close()
