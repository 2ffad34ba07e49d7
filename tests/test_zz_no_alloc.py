"""GPU test of the entry point that allocates no device memory (fiesta_partial_sums_noalloc_async: per-shift sums of
one real sector with the partial records in a static device array; fx_kernels_noalloc.cu).

Collected last (file name), because the suite runs with pytest -x.  Passes alone in a fresh process and after the
other tests: it makes its own context, and the only state it shares with them is the static array, which the entry
point itself prepares."""
import numpy as np
import pytest

from workloads import make_workload

pytestmark = pytest.mark.gpu

TOL_SUM = 1e-10      # tests/helpers.py: the bar of the per-shift sums (R15)


def _device_buffers(torch, shape):
    sums = torch.full(shape, float("nan"), dtype=torch.float64, device="cuda:0")
    nonfinite = torch.full((1,), 12345, dtype=torch.int64, device="cuda:0")
    return sums, nonfinite


def test_no_alloc_entry_point_matches_partial_sums(lib):
    import torch
    fb = lib
    ctx = fb.Context(0)                      # stream 0: torch.cuda.synchronize() below waits for it
    wl = make_workload("C3", nsectors=3, npoints=1 << 16, n_shifts=8)
    prog = ctx.compile(wl.sectors, wl.dim)
    lattice = fb.Rule.from_workload(wl)
    mc = fb.Rule(kind=fb.RULE_MC)
    K = wl.K
    # two calls in a row, the second with fewer records than the first left behind in the shared array,
    # then the first again
    cases = [(2, lattice, wl.npoints, wl.seed), (0, mc, 70001, 5), (2, lattice, wl.npoints, wl.seed), (1, mc, 3, 9)]
    first = None
    for sector, rule, npoints, seed in cases:
        R = rule.n_shifts if rule.kind == fb.RULE_LATTICE else 1
        sums, nonfinite = _device_buffers(torch, (R, K, 2))
        ctx.partial_sums_noalloc_async(prog, sector, npoints, rule, seed, sums.data_ptr(), nonfinite.data_ptr())
        torch.cuda.synchronize()
        got = sums.cpu().numpy()
        ref = ctx.partial_sums(prog, npoints, rule, seed, sectors=[sector], tier=fb.TIER_INTERPRETER)[0, :, :, 0, :]
        assert np.all(np.isfinite(got))
        assert np.all(np.abs(got - ref) <= TOL_SUM * np.abs(ref))
        assert np.array_equal(got, ref)      # same chunking, same order of additions: the same bits
        assert int(nonfinite.item()) == 0
        if first is None:
            first = got.copy()
        elif sector == 2:
            assert np.array_equal(got, first)
    # without the optional counter
    sums, _ = _device_buffers(torch, (1, K, 2))
    ctx.partial_sums_noalloc_async(prog, 0, 70001, mc, 5, sums.data_ptr())
    torch.cuda.synchronize()
    assert np.array_equal(sums.cpu().numpy(), ctx.partial_sums(prog, 70001, mc, 5, sectors=[0], tier=0)[0, :, :, 0, :])
    prog.close()
    ctx.close()


def test_no_alloc_entry_point_counts_nonfinite_and_rejects_what_it_does_not_cover(lib):
    import torch
    from workloads import SectorText
    fb = lib
    ctx = fb.Context(0)
    # log of a negative number on half of the cube: NaN values are counted, and the counter starts from zero each call
    bad = SectorText(sector_id=4, texts=["2;\n0;\nl[x[1]-0.5]*x[2];\n|"])
    prog = ctx.compile([bad], 2)
    mc = fb.Rule(kind=fb.RULE_MC)
    counts = []
    for _ in range(2):
        sums, nonfinite = _device_buffers(torch, (1, 1, 2))
        ctx.partial_sums_noalloc_async(prog, 0, 4096, mc, 1, sums.data_ptr(), nonfinite.data_ptr())
        torch.cuda.synchronize()
        counts.append(int(nonfinite.item()))
    assert counts[0] == counts[1] and 1500 < counts[0] < 2600
    sums, nonfinite = _device_buffers(torch, (8, 1, 2))
    # beyond the static array: 8 shifts x 2^27 points = 8 x 1024 chunks of 2^17 points > 4096 records
    big = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=12345, periodize_r=3)
    with pytest.raises(fb.FiestaError) as ei:
        ctx.partial_sums_noalloc_async(prog, 0, 8 << 27, big, 1, sums.data_ptr(), nonfinite.data_ptr())
    assert "4096" in str(ei.value)
    with pytest.raises(fb.FiestaError):
        ctx.partial_sums_noalloc_async(prog, 0, 4096, fb.Rule(kind=fb.RULE_VEGAS), 1, sums.data_ptr())
    with pytest.raises(fb.FiestaError):
        ctx.partial_sums_noalloc_async(prog, 1, 4096, mc, 1, sums.data_ptr())          # no such sector
    prog.close()
    wl = make_workload("C4", nsectors=1, npoints=1 << 12)
    cplx = ctx.compile(wl.sectors, wl.dim)
    with pytest.raises(fb.FiestaError):
        ctx.partial_sums_noalloc_async(cplx, 0, 4096, mc, 1, sums.data_ptr())          # complex sector
    cplx.close()
    ctx.close()
