"""fredopt_volume_histogram_no_alloc (include/fredopt.h): the entry point that allocates nothing -- its bin counters are a fixed
array in device memory -- against the existing path, fredopt_volume_histogram, on the same plan and weights.  Collected last
on purpose (the file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the other tests.

Tolerance: the one tests/test_gpu_parity.py uses for the volume histograms (1.5 voxels of the structure + 1e-6 per bin): the
new call bins the fp32 outputs of fredopt_dose_let, the existing one its own fp64 products, so a value within fp32 rounding of
a bin edge may move one voxel.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fredopt():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2509_20012_b200 import fredopt as f
    return f


def test_no_alloc_histogram_matches_the_plan_path_on_calls_in_a_row(fredopt, plan0):
    f = fredopt
    gp = f.from_plan(plan0)
    x = plan0.x0
    n = plan0.n_rows
    dose = torch.empty(n, dtype=torch.float32, device="cuda")
    letd = torch.empty(n, dtype=torch.float32, device="cuda")
    gp.dose_let(x, dose, letd)
    labels = plan0.labels.to(device="cuda", dtype=torch.int32).contiguous()
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    f.no_alloc_setup()
    # calls in a row on the shared scratch: more bins, then fewer (stale counters above them), the other quantity, and again
    cases = [(0, 1, 200), (0, 2, 64), (2, 2, 64), (2, 1, 31), (0, 1, 200), (0, 2, 64)]
    hists = [torch.full((nb,), -1.0, dtype=torch.float32, device="cuda") for _, _, nb in cases]
    refs = []
    for q, label, nb in cases:
        _, _, mx, nvox = gp.structure_stats(q, label, x)
        assert nvox > 0 and mx > 0
        ref = np.empty(nb, np.float32)
        gp.volume_histogram(q, label, nb, mx * 1.05, ref, x)            # the existing path (plan-owned scratch)
        refs.append((ref, mx * 1.05, nvox))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (q, label, nb), h, (ref, vmax, nvox) in zip(cases, hists, refs):
        f.volume_histogram_no_alloc(dose if q == 0 else letd, labels, label, nb, vmax, h, count)
        got = h.cpu().numpy()                                           # synchronises
        assert int(count.item()) == nvox
        assert np.all(np.abs(got - ref) <= 1.5 / nvox + 1e-6), (q, label, nb, float(np.abs(got - ref).max()))
        assert got[0] == 1.0 and np.all(np.diff(got) <= 0)
    # two calls enqueued back to back without a synchronisation in between
    f.volume_histogram_no_alloc(dose, labels, 1, 200, refs[0][1], hists[0])
    f.volume_histogram_no_alloc(dose, labels, 2, 64, refs[1][1], hists[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                         # no device memory was taken by any of the calls
    for i in (0, 1):
        assert np.all(np.abs(hists[i].cpu().numpy() - refs[i][0]) <= 1.5 / refs[i][2] + 1e-6)
    # labels = NULL: every voxel of the caller's array; the same counts as the labelled call on the masked values
    sel = dose[labels == 2].contiguous()
    h2 = torch.empty(64, dtype=torch.float32, device="cuda")
    f.volume_histogram_no_alloc(sel, None, 0, 64, refs[1][1], h2, count)
    assert np.array_equal(h2.cpu().numpy(), hists[1].cpu().numpy()) and int(count.item()) == refs[1][2]
    # an empty structure gives zeros
    f.volume_histogram_no_alloc(dose, labels, 12345, 64, 1.0, h2, count)
    assert not h2.cpu().numpy().any() and int(count.item()) == 0
    gp.destroy()


def test_no_alloc_histogram_rejects_sizes_beyond_the_scratch(fredopt):
    f = fredopt
    v = torch.ones(16, dtype=torch.float32, device="cuda")
    h = torch.empty(f.NO_ALLOC_MAX_BINS + 1, dtype=torch.float32, device="cuda")
    with pytest.raises(f.FredoptError) as e:
        f.volume_histogram_no_alloc(v, None, 0, f.NO_ALLOC_MAX_BINS + 1, 1.0, h)
    assert e.value.code == f.INVALID_ARG and "4096" in str(e.value)
    f.volume_histogram_no_alloc(v, None, 0, f.NO_ALLOC_MAX_BINS, 2.0, h)     # the maximum is accepted
    assert h[:f.NO_ALLOC_MAX_BINS // 2 + 1].eq(1.0).all() and h[f.NO_ALLOC_MAX_BINS // 2 + 1:f.NO_ALLOC_MAX_BINS].eq(0.0).all()
    torch.cuda.synchronize()
    for bad in (dict(n_bins=0, vmax=1.0), dict(n_bins=8, vmax=0.0), dict(n_bins=8, vmax=float("inf"))):
        with pytest.raises(f.FredoptError):
            f.volume_histogram_no_alloc(v, None, 0, bad["n_bins"], bad["vmax"], h)
