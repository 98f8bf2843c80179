"""qtam_cluster_noalloc: cluster labelling for a caller that cannot allocate device memory.

Why the entry point exists: every other compute call wants a qtam_plan, and making a plan calls cudaMalloc.  A stage of
a running low-latency pipeline (cudaMalloc / cudaFree stall the whole device), a plug-in whose host application already
owns the free device memory through its own pool, or code that is only lent its buffers cannot do that.  For them the
library keeps the one piece of scratch the labelling needs (a pixel counter per component root) in a fixed 4 MiB array
inside libqtam.so, so the call takes no plan and allocates nothing; in exchange the problem size is bounded
(batch * rows * samples <= 2^20) and calls that overlap on one GPU would race on that array.

What is checked: the labels and counts equal those of the existing path (Plan.cluster, whose scratch is in the plan's
workspace) bit for bit -- that is the tolerance the cluster tests use -- on two calls in a row.  The second call
labels a different, sparser image with a larger minimum area right after a dense one, so counters left in the shared
array by the first call would show up as clusters that survive the area filter.  The size limit is checked without a
GPU.  This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process (the first call then does the per-device set-up) and after the
other tests.
"""
import numpy as np
import pytest

from paper_2603_29785_b200 import binding


def test_noalloc_rejects_what_does_not_fit():
    """the size check comes before any CUDA call, so it can be seen on a box without a GPU: a clear status, not a
    launch failure, and nothing is read or written"""
    L = binding.lib()
    limit = binding.CLUSTER_NOALLOC_MAX_PIXELS
    fake = 256            # a non-null address that is never dereferenced: the call must return before touching it
    rows, samples = 64, 4096
    batch = limit // (rows * samples) + 1
    s = L.qtam_cluster_noalloc(0, fake, rows * samples, batch, rows, samples, 1, fake, fake, None)
    assert s == 6 and b"scratch" in L.qtam_status_string(s)
    assert L.qtam_cluster_noalloc(0, fake, 2 * limit, 1, 2, limit, 1, fake, fake, None) == 6
    # argument errors are still argument errors
    assert L.qtam_cluster_noalloc(0, None, 16, 1, 4, 4, 1, fake, fake, None) == 1
    assert L.qtam_cluster_noalloc(0, fake, 15, 1, 4, 4, 1, fake, fake, None) == 1      # stride shorter than an image
    assert L.qtam_cluster_noalloc(0, fake, 16, 1, 4, 4, 0, fake, fake, None) == 1      # min_area < 1
    assert L.qtam_cluster_noalloc(7, fake, 16, 1, 4, 4, 1, fake, fake, None) == 1      # no such dtype
    # an empty batch is fine and does nothing
    assert L.qtam_cluster_noalloc(0, fake, 16, 0, 4, 4, 1, fake, fake, None) == 0


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_noalloc_equals_the_plan_path_on_two_calls_in_a_row(dtype):
    import torch
    assert torch.cuda.is_available(), "GPU test on a box without a CUDA device"
    torch.cuda.set_device(0)
    N, nseg, plane = 4096, 3, 1
    g = binding.Plan(4096.0, N, [6.0, 12.0], 32.0, 1600.0, 24.0, dtype=dtype, max_batch=nseg, tile_length=-1)
    rows = [r for r in g.rows if r.plane == plane]
    R, M, first = len(rows), int(rows[0].M), int(rows[0].offset)
    assert all(int(r.M) == M for r in rows) and R * M == int(binding.lib().qtam_plane_pixels(g._h, plane))
    assert nseg * R * M <= binding.CLUSTER_NOALLOC_MAX_PIXELS
    cdt = torch.complex64 if dtype == "f32" else torch.complex128
    rng = np.random.default_rng(11)
    # the caller's buffers, made once: the entry point itself is handed pointers only
    labels = torch.empty((nseg, R * M), dtype=torch.int32, device="cuda")
    count = torch.empty((nseg,), dtype=torch.int32, device="cuda")
    for call, (density, min_area) in enumerate(((0.7, 1), (0.25, 6))):
        Z = torch.zeros((nseg, g.ctot), dtype=cdt, device="cuda")
        pat = rng.random((nseg, R * M)) < density
        pat[:, :3] = True                                   # something in the corner that wraps in time
        pat[:, M - 2:M] = True
        vals = (rng.standard_normal((nseg, R * M)) + 1j * rng.standard_normal((nseg, R * M))) * pat
        Z[:, first:first + R * M] = torch.from_numpy(vals).to(cdt).cuda()
        want_labels, want_count = g.cluster(Z, plane, min_area)          # existing path: scratch in the plan
        labels.fill_(-7)
        count.fill_(-7)
        binding.cluster_noalloc(Z.view(-1)[first:], g.ctot, nseg, R, M, min_area, labels, count)
        torch.cuda.synchronize()
        assert torch.equal(labels, want_labels.view(nseg, R * M)), f"labels differ on call {call}"
        assert torch.equal(count, want_count), f"counts differ on call {call}"
        assert int(want_count.min()) >= 1
        if call == 1:                                       # the filter really dropped something
            assert int(g.cluster(Z, plane, 1)[1].sum()) > int(want_count.sum())
    # a bare stack of images (stride = one image) of another shape, same call, same array
    R2, M2 = 5, 96
    img = torch.from_numpy((rng.random((2, R2 * M2)) < 0.5).astype(np.complex64)).cuda()
    lab2 = torch.empty((2, R2 * M2), dtype=torch.int32, device="cuda")
    cnt2 = torch.empty((2,), dtype=torch.int32, device="cuda")
    binding.cluster_noalloc(img, R2 * M2, 2, R2, M2, 2, lab2, cnt2)
    got = lab2.cpu().numpy().reshape(2, R2, M2)
    act = img.cpu().numpy().reshape(2, R2, M2) != 0
    for b in range(2):
        kept = got[b] > 0
        assert not kept[~act[b]].any()
        ids, areas = np.unique(got[b][kept], return_counts=True)
        assert len(ids) == int(cnt2[b]) and areas.min() >= 2
        # a label is 1 + the smallest pixel index of its cluster, and neighbours share a label
        for i in ids:
            assert np.flatnonzero(got[b].ravel() == i)[0] == i - 1
        both = act[b] & np.roll(act[b], -1, axis=1)
        assert np.array_equal(got[b][both], np.roll(got[b], -1, axis=1)[both])
    # too large is refused with its own status and leaves the outputs alone
    with pytest.raises(binding.QtamError) as e:
        big = binding.CLUSTER_NOALLOC_MAX_PIXELS // (R * M) + 1
        binding.cluster_noalloc(torch.zeros((big, R * M), dtype=cdt, device="cuda"), R * M, big, R, M, 1,
                                torch.empty((big, R * M), dtype=torch.int32, device="cuda"),
                                torch.empty((big,), dtype=torch.int32, device="cuda"))
    assert e.value.code == 6
    g.close()
