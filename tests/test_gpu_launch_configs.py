"""GPU parity at the launch configurations bench.py's largest-batch records time, and plans of different shape alive
at the same time.

north_star: ">= 60 % of the HBM roofline ... at the largest batch".  A plan's tile lengths, ring sizes and groups adapt
to `max_batch`, so the largest-batch numbers are only worth something if those very configurations are compared with
the oracle.  PAPER.md:208 (Sec. V) alternates a low-Q and a high-Q transform: several plans live in one process, and
what one plan sets on a kernel (its dynamic shared-memory limit is per kernel and per process) must not break another.
"""
import numpy as np
import pytest

import bench
from conftest import rel_l2
from oracle.qtam_ref import RefPlan
from paper_2603_29785_b200 import binding, inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}
TOL_RT = {"f64": 1e-12, "f32": 1e-5}
TOL_ROW = {"f64": 1e-11, "f32": 1e-4}


def worst_row(got, want, plan):
    offs = np.array([int(r.offset) for r in plan.rows], dtype=np.int64)
    num = np.add.reduceat(np.abs(got - want) ** 2, offs, axis=-1)
    den = np.add.reduceat(np.abs(want) ** 2, offs, axis=-1)
    return float(np.sqrt((num / np.maximum(den, 1e-300)).max()))


def largest_cases():
    """(configuration, dtype, batch) exactly as bench.py builds its largest-batch workloads"""
    out = []
    for name, big in sorted(bench.LARGEST.items()):
        out.append((name, "f32", big))
        if name == "cfg5":
            out.append((name, "f64", big // 2))
    return out


@pytest.mark.parametrize("name,dtype,B", largest_cases(), ids=lambda v: str(v))
def test_largest_batch_against_the_oracle(name, dtype, B):
    """plans created with bench.py's max_batch; a strided sample of >= 16 segments plus the first and the last is
    compared with the oracle element by element (forward on the same input; inverse, run at the full batch, on the
    oracle's coefficients); the round trip is checked on EVERY segment against the projection Pi_C x"""
    cfg = inputs.CONFIGS[name]
    fs, N, Q, fmin, fmax, rows = inputs.plan_args(name)
    g = binding.Plan(fs, N, Q, fmin, fmax, rows, dtype=dtype, max_batch=B)
    r = RefPlan(fs, N, Q, fmin, fmax, rows)
    rdt = np.float64 if dtype == "f64" else np.float32
    cdt = np.complex128 if dtype == "f64" else np.complex64
    # the configuration's own segments, repeated with a different circular shift per repetition (distinct data in
    # every slot without generating thousands of coloured-noise segments)
    nb = min(cfg["batch"], 64, B)
    base = inputs.make_batch(name, batch=nb, dtype=dtype)
    x = np.empty((B, N), dtype=rdt)
    for b in range(B):
        x[b] = np.roll(base[b % nb], 977 * (b // nb))
    dx = torch.from_numpy(x).cuda()
    has_inv = "inverse" in cfg["calls"]
    Y = g.forward(dx)
    sample = sorted(set([0, B - 1] + list(range(0, B, max(1, B // 16)))))
    assert len(sample) >= min(B, 16)
    Yin = Y.clone() if has_inv else None
    want_inv = {}
    worst = worst_r = 0.0
    for b in sample:
        x64 = x[b:b + 1].astype(np.float64)
        Yr = r.forward(x64, engine=1)
        Yg = Y[b:b + 1].cpu().numpy()
        worst = max(worst, rel_l2(Yg[0], Yr[0]))
        worst_r = max(worst_r, worst_row(Yg, Yr, r))
        if has_inv:
            Yc = Yr.astype(cdt)
            Yin[b:b + 1] = torch.from_numpy(Yc).cuda()
            want_inv[b] = r.inverse(Yc.astype(np.complex128), engine=1)[0]
    assert worst <= TOL[dtype] and worst_r <= TOL_ROW[dtype], (worst, worst_r)
    if not has_inv:
        g.close()
        return
    xo = g.inverse(Yin)                                  # the whole batch, oracle coefficients in the sampled slots
    worst = max(rel_l2(xo[b].cpu().numpy(), want_inv[b]) for b in sample)
    assert worst <= TOL[dtype], worst
    # round trip of every segment (cfg5's step has a threshold between the two calls; the plain round trip is what
    # pins the two launch configurations against each other)
    xrt = g.inverse(Y)
    _, cover = g.frame(-1)
    cov = torch.from_numpy(cover.astype(bool)).cuda()
    worst = 0.0
    for b0 in range(0, B, 64):
        xs = dx[b0:b0 + 64].double()
        X = torch.fft.rfft(xs, dim=-1)
        proj = torch.fft.irfft(torch.where(cov[None, :], X, torch.zeros_like(X)), n=N, dim=-1)
        err = (xrt[b0:b0 + 64].double() - proj).norm(dim=-1) / proj.norm(dim=-1)
        worst = max(worst, float(err.max().item()))
    assert worst <= TOL_RT[dtype], worst
    g.close()


def _run(plan, dx, calls):
    Y = plan.forward_threshold(dx, 3.0) if "threshold" in calls else plan.forward(dx)
    return Y, plan.inverse(Y)


def test_two_live_plans_of_different_shape():
    """a cfg3-shaped and a cfg5-shaped float plan and a double plan alive together, calls alternated A, B, C, A, B, C:
    every result is bit-identical to what the plan gives when it is the only plan of the process.  Both creation
    orders, so that whichever plan needs less shared memory for a shared kernel is once created last."""
    specs = [("cfg3", "f32", 5), ("cfg5", "f32", 24), ("cfg5", "f64", 7), ("cfg2", "f32", 3)]
    data, alone = [], []
    for name, dtype, nseg in specs:
        x = torch.from_numpy(inputs.make_batch(name, batch=nseg, dtype=dtype)).cuda()
        p = binding.Plan(*inputs.plan_args(name), dtype=dtype, max_batch=nseg)
        alone.append(_run(p, x, list(inputs.CONFIGS[name]["calls"]) + ["inverse"]))
        data.append(x)
        p.close()
    for order in (list(range(len(specs))), list(reversed(range(len(specs))))):
        plans = {}
        for i in order:
            name, dtype, nseg = specs[i]
            plans[i] = binding.Plan(*inputs.plan_args(name), dtype=dtype, max_batch=nseg)
        for _ in range(2):
            for i in range(len(specs)):
                Y, xo = _run(plans[i], data[i], list(inputs.CONFIGS[specs[i][0]]["calls"]) + ["inverse"])
                assert torch.equal(Y, alone[i][0]) and torch.equal(xo, alone[i][1]), (order, specs[i])
        # a plan created and destroyed in between must not disturb the live ones either
        tmp = binding.Plan(1024.0, 1024, [4.0, 8.0], 16.0, 400.0, 12.0, dtype="f32", max_batch=2)
        tmp.forward(torch.zeros((2, 1024), dtype=torch.float32, device="cuda"))
        tmp.close()
        for i in reversed(range(len(specs))):
            Y, xo = _run(plans[i], data[i], list(inputs.CONFIGS[specs[i][0]]["calls"]) + ["inverse"])
            assert torch.equal(Y, alone[i][0]) and torch.equal(xo, alone[i][1]), (order, specs[i])
        for p in plans.values():
            p.close()


class Guarded:
    """a tensor of `shape` in the middle of a larger allocation whose two margins hold a fixed bit pattern"""
    PAD = 1 << 20          # bytes on either side

    def __init__(self, shape, dtype):
        n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        self.raw = torch.full((self.PAD + n + self.PAD,), 0xA5, dtype=torch.uint8, device="cuda")
        self.t = self.raw[self.PAD:self.PAD + n].view(dtype).view(shape)

    def intact(self):
        return bool((self.raw[:self.PAD] == 0xA5).all() and (self.raw[-self.PAD:] == 0xA5).all())


@pytest.mark.parametrize("name,dtype,nseg", [("cfg3", "f32", 5), ("cfg5", "f32", 33), ("cfg5", "f64", 6), ("cfg2", "f32", 3),
                                             ("cfg4", "f32", 2), ("paper6s", "f32", 3), ("cfg1", "f64", 1)])
def test_no_write_outside_the_callers_buffers(name, dtype, nseg):
    """compute-sanitizer is closed on this pool, so out-of-bounds WRITES into caller memory are
    looked for directly: every buffer a call is given sits between two 1 MiB margins of a known pattern, the batch is
    smaller than the plan's max_batch (the rows after it must stay untouched as well), and the margins and the unused
    rows are compared bit for bit after forward, threshold, fused forward + threshold and inverse (joint and one plane)"""
    g = binding.Plan(*inputs.plan_args(name), dtype=dtype, max_batch=nseg + 2)
    rdt = torch.float64 if dtype == "f64" else torch.float32
    cdt = torch.complex128 if dtype == "f64" else torch.complex64
    X, Y, Y2, O = (Guarded((nseg + 1, g.N), rdt), Guarded((nseg + 1, g.ctot), cdt), Guarded((nseg + 1, g.ctot), cdt),
                   Guarded((nseg + 1, g.N), rdt))
    X.t[:nseg] = torch.from_numpy(inputs.make_batch(name, batch=nseg, dtype=dtype)).cuda()
    spare = [b.t[nseg].clone() for b in (X, Y, Y2, O)]
    g.forward(X.t[:nseg], out=Y.t[:nseg])
    g.forward_threshold(X.t[:nseg], 3.0, out=Y2.t[:nseg])
    g.threshold_rowmedian(Y.t[:nseg], 3.0)
    assert torch.equal(Y.t[:nseg].view(rdt), Y2.t[:nseg].view(rdt))          # and the fused call equals the two calls
    g.inverse(Y.t[:nseg], out=O.t[:nseg])
    g.inverse(Y2.t[:nseg], plane=g.n_planes - 1, out=O.t[:nseg])
    torch.cuda.synchronize()
    for b, s in zip((X, Y, Y2, O), spare):
        assert b.intact()
        assert torch.equal(b.t[nseg].view(torch.uint8), s.view(torch.uint8))
    g.close()


def test_composite_bank_with_more_than_64_window_identities():
    """66 planes with 66 different Kaiser windows at one Q: the float row tables are keyed on (half-width, window
    identity), and a key that packs the identity into 6 bits would hand plane 64 + b the window of plane b at the next
    half-width.  Rows dense enough that consecutive half-widths occur; every row against the oracle."""
    nP = 66
    fs, N = 2048.0, 4096
    args = (fs, N, [8.0] * nP, 16.0, 900.0, 40.0)
    kw = dict(plane_windows=[("kaiser", 3.0 + 0.125 * i) for i in range(nP)])
    g = binding.Plan(*args, dtype="f32", max_batch=2, **kw)
    r = RefPlan(*args, **kw)
    dks = sorted({int(a.dk) for a in g.rows})
    assert any(b - a == 1 for a, b in zip(dks, dks[1:])) and g.n_planes == nP
    x = inputs.white_noise(N, 4242, batch=2).astype(np.float32)
    Y = g.forward(torch.from_numpy(x).cuda()).cpu().numpy()
    Yr = r.forward(x.astype(np.float64), engine=1)
    assert max(rel_l2(Y[b], Yr[b]) for b in range(2)) <= TOL["f32"]
    assert worst_row(Y, Yr, r) <= TOL_ROW["f32"]
    Yin = Yr.astype(np.complex64)
    for plane in (-1, 1, 64, 65):
        xg = g.inverse(torch.from_numpy(Yin).cuda(), plane=plane).cpu().numpy()
        xr = r.inverse(Yin.astype(np.complex128), plane=plane, engine=1)
        assert max(rel_l2(xg[b], xr[b]) for b in range(2)) <= TOL["f32"], plane
    g.close()
