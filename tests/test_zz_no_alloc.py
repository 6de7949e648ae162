"""semb_field_minmax_hist_noalloc: the min / max / histogram consumer through the entry point that allocates nothing (its
accumulators live in a file-scope device array, include/semb200.h) against the existing semb_field_minmax_hist, on calls in a
row that share that array.  Integer counts and min / max: the bar is equality, as in test_export_field_and_consumer.

Collected last on purpose (the name sorts after every other test file): the suite runs with `pytest -x`.
Runs alone in a fresh process (`pytest tests/test_zz_no_alloc.py -m gpu`) and after the other tests alike: it builds its own
inputs and depends on no state left by them."""
import ctypes as C

import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def semb(torch_cuda):
    from paper_2501_13240_b200 import semb as S
    S.lib()                                             # fails loudly if the CUDA library is missing
    return S


def desc_of(semb, t, count=None, stride=1):
    """a device fp64 field descriptor over tensor t (what semb_export_field hands out: dtype 1 = fp64, memspace 1 = device)"""
    return semb.FieldDesc(name=b"synthetic", ptr=C.c_void_p(t.data_ptr()), dtype=1, memspace=1,
                          count=t.numel() // stride if count is None else count, stride=stride, cycle=0, time=0.0)


def fields(torch, n):
    """temperature-like field of the RBC workload (conduction profile 1 - z plus fluctuations, DESIGN.md input recipe) and a
    signed, wider one"""
    z = I.uniform(I.seed_for(9, 1), n, 0.0, 1.0)
    T = (1.0 - z) + 0.05 * I.uniform(I.seed_for(9, 2), n)
    w = 3.0 * I.uniform(I.seed_for(9, 3), n)
    return torch.from_numpy(T).cuda(), torch.from_numpy(w).cuda(), T, w


CASES = [  # (field, nbins, lo, hi, stride): the second and third follow a call that left MORE bins and other min / max behind
    ("T", 256, 0.0, 1.0, 1),
    ("w", 64, 0.0, 0.0, 1),          # lo >= hi: the range is found on the device (two passes)
    ("w", 4096, -1.0, 2.0, 1),       # the maximum size; values outside the range go to the end bins
    ("T", 100, 0.25, 0.75, 2),       # every second value
    ("T", 256, 0.0, 1.0, 1),         # the first call again
]


def run(semb, torch, fn, d, nbins, lo, hi):
    mm = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")        # garbage: the call must write every output word
    h = torch.full((nbins,), -1, dtype=torch.int64, device="cuda")
    fn(d, nbins, lo, hi, mm, h)
    return mm, h


def test_noalloc_minmax_hist_matches_existing_path(torch_cuda, semb, orc):
    torch = torch_cuda
    n = 300007                                           # 147 blocks of 2048 and a ragged tail
    dT, dw, T, w = fields(torch, n)
    host = {"T": T, "w": w}; devt = {"T": dT, "w": dw}
    # one untimed pass of both paths first: the driver loads kernel images lazily on the first launch (context growth, not an
    # allocation of the call)
    for name, nbins, lo, hi, stride in CASES[:2]:
        d = desc_of(semb, devt[name], stride=stride)
        run(semb, torch, semb.field_minmax_hist, d, nbins, lo, hi); run(semb, torch, semb.field_minmax_hist_noalloc, d, nbins, lo, hi)
    torch.cuda.synchronize()
    # the calls in a row on one stream, no synchronisation in between; outputs allocated beforehand
    outs = [(torch.full((2,), -7.0, dtype=torch.float64, device="cuda"), torch.full((c[1],), -1, dtype=torch.int64, device="cuda"))
            for c in CASES]
    descs = [desc_of(semb, devt[c[0]], stride=c[4]) for c in CASES]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (name, nbins, lo, hi, stride), d, (mm, h) in zip(CASES, descs, outs):
        semb.field_minmax_hist_noalloc(d, nbins, lo, hi, mm, h)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0         # nothing allocated by the calls
    for (name, nbins, lo, hi, stride), d, (mm, h) in zip(CASES, descs, outs):
        mm_ref, h_ref = run(semb, torch, semb.field_minmax_hist, d, nbins, lo, hi)     # the existing path, same arguments
        torch.cuda.synchronize()
        assert torch.equal(mm, mm_ref), (name, nbins, mm, mm_ref)
        assert torch.equal(h, h_ref), (name, nbins)
        assert int(h.sum().item()) == d.count
        v = host[name][::stride][:d.count]               # and the CPU oracle, as the existing path's own test does
        mn, mx, ho = orc.minmax_hist(v, nbins, lo if lo < hi else v.min(), hi if lo < hi else v.max())
        assert mm[0].item() == mn and mm[1].item() == mx
        assert np.array_equal(h.cpu().numpy().astype(np.uint64), ho)


def test_noalloc_rejects_sizes_beyond_the_static_scratch(torch_cuda, semb):
    torch = torch_cuda
    t = torch.zeros(1000, dtype=torch.float64, device="cuda")
    mm = torch.zeros(2, dtype=torch.float64, device="cuda")
    assert semb.NOALLOC_MAX_BINS == 4096
    h = torch.full((semb.NOALLOC_MAX_BINS + 1,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(semb.SembError) as ei:
        semb.field_minmax_hist_noalloc(desc_of(semb, t), semb.NOALLOC_MAX_BINS + 1, 0.0, 1.0, mm, h)
    assert ei.value.code == -1 and "4096" in str(ei.value) and "4097" in str(ei.value)
    torch.cuda.synchronize()
    assert int((h == -1).sum().item()) == h.numel()      # rejected before anything was launched
    with pytest.raises(semb.SembError):
        semb.field_minmax_hist_noalloc(desc_of(semb, t), 0, 0.0, 1.0, mm, h)
    semb.field_minmax_hist_noalloc(desc_of(semb, t), semb.NOALLOC_MAX_BINS, 0.0, 1.0, mm, h)      # the limit itself is accepted
    torch.cuda.synchronize()
    assert h[0].item() == 1000 and int(h[:semb.NOALLOC_MAX_BINS].sum().item()) == 1000 and mm[0].item() == 0.0 and mm[1].item() == 0.0
