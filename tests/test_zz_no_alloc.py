"""qlp_bls_grid_noalloc: the grid stage (S1) with its scratch in a file-scope __device__ array of the library, for
callers that cannot call cudaMalloc (include/qlp_bls.h).  Collected last on purpose (pytest -x).

The existing path, qlp_bls_grid, is the reference: same kernels, so grid descriptors, freq_ptr and the two totals
must be identical bit for bit -- on two calls in a row that share the static array (a larger batch first, then a
smaller one, so stale contents of the array would show), with the device's free memory unchanged across the calls,
and with a clear error beyond QLP_BLS_NOALLOC_MAX_STARS."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

NOALLOC_MAX_STARS = 262144


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2302_01293_b200 import build, bls
    build.build()
    return bls


def _batches():
    from paper_2302_01293_b200 import synth
    ts = synth.sector_times(0, 1800.0)
    one = lambda t: (t, np.ones(t.size), np.full(t.size, 1e-3))
    bad = ts.copy(); bad[10] = bad[9]                                   # status 7: skipped, n_freq = 0
    first = synth.make_batch(5, star_ids=np.arange(48))                  # ragged multi-sector stars
    odd = synth.from_arrays([one(ts[:1]), one(ts[:2]), one(ts), one(bad),
                             one(np.concatenate([ts[:300], ts[:300] + 400.0]))],
                            rho=np.array([1.0, 0.3, 5.0, 1.0, 0.1]))
    second = synth.make_batch(2, n_stars=7)                              # fewer stars than the call before
    return [first, odd, second]


def _noalloc(gpu, ctx, dev, out):
    """out = (grid, freq_ptr, totals) device tensors owned by the caller; returns them as numpy."""
    ctx.grid_noalloc(dev[0], dev[1], dev[4], *out)
    S = int(dev[0].numel()) - 1
    return out[0][:S].cpu().numpy().tobytes(), out[1][:S + 1].cpu().numpy(), out[2].cpu().numpy()


def test_grid_noalloc_matches_grid_on_calls_in_a_row(gpu):
    import torch
    batches = _batches()
    devs = [gpu.upload(b) for b in batches]
    ref_ctx, ctx = gpu.QlpBls(), gpu.QlpBls()       # the no-alloc calls get a context whose workspace stays empty
    try:
        want = []
        for dev in devs:
            grid, fp, tf, tb = ref_ctx.grid(dev[0], dev[1], dev[4], dev[5])
            want.append((grid.cpu().numpy().tobytes(), fp.cpu().numpy(), tf, tb))
        s_max = max(b.n_stars for b in batches)
        # outputs are the caller's: allocated once, reused by every call (filled with junk first)
        out = (torch.full((s_max, gpu.GRID_DTYPE.itemsize), 0xAB, dtype=torch.uint8, device="cuda"),
               torch.full((s_max + 1,), -7, dtype=torch.int64, device="cuda"),
               torch.full((2,), -7, dtype=torch.int64, device="cuda"))
        _noalloc(gpu, ctx, devs[0], out)             # first call on the device: resolves the array's address
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for rep in range(2):                         # the whole sequence twice: every batch follows another one
            for dev, w in zip(devs, want):
                ctx.grid_noalloc(dev[0], dev[1], dev[4], *out)
                torch.cuda.synchronize()
                assert torch.cuda.mem_get_info()[0] == free0      # the call took no device memory
                S = int(dev[0].numel()) - 1
                assert out[0][:S].cpu().numpy().tobytes() == w[0]                 # descriptors bit for bit
                assert np.array_equal(out[1][:S + 1].cpu().numpy(), w[1])         # freq_ptr
                assert out[2].cpu().numpy().tolist() == [w[2], w[3]]              # total_freq, total_bins
        assert want[1][2] > 0 and want[2][3] > 0
        # the grids are usable downstream: the spectrum of the last batch from the no-alloc grid = from the other
        dev, b = devs[2], batches[2]
        sr_a, best_a = ref_ctx.spectrum(dev[0], dev[1], dev[2], dev[3], out[0][:b.n_stars], out[1][:b.n_stars + 1],
                                        want[2][2])
        grid, fp, tf, _ = ref_ctx.grid(dev[0], dev[1], dev[4], dev[5])
        sr_b, best_b = ref_ctx.spectrum(dev[0], dev[1], dev[2], dev[3], grid, fp, tf)
        assert torch.equal(sr_a, sr_b) and torch.equal(best_a, best_b)
    finally:
        ctx.close()
        ref_ctx.close()


def test_grid_noalloc_empty_batch_and_limit(gpu):
    import torch
    ctx = gpu.QlpBls()
    try:
        z = torch.zeros(1, dtype=torch.int64, device="cuda")
        fp = torch.full((1,), -7, dtype=torch.int64, device="cuda")
        totals = torch.full((2,), -7, dtype=torch.int64, device="cuda")
        ctx.grid_noalloc(z, z.double(), z.double(), z.to(torch.uint8), fp, totals)    # S = 0 is legal
        assert fp.tolist() == [0] and totals.tolist() == [0, 0]
        # one star more than the static array holds: refused, nothing enqueued, outputs untouched
        n = NOALLOC_MAX_STARS + 1
        row_ptr = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        grid = torch.zeros((n, gpu.GRID_DTYPE.itemsize), dtype=torch.uint8, device="cuda")
        fp = torch.full((n + 1,), -7, dtype=torch.int64, device="cuda")
        totals.fill_(-7)
        with pytest.raises(gpu.QlpBlsError, match=r"static scratch.*\(-6\)"):
            ctx.grid_noalloc(row_ptr, z.double(), row_ptr[:n].double(), grid, fp, totals)
        torch.cuda.synchronize()
        assert totals.tolist() == [-7, -7] and int(fp[0]) == -7
        # exactly the maximum is accepted (stars without points: status != 0, n_freq = 0)
        ctx.grid_noalloc(row_ptr[:n], z.double(), row_ptr[:n - 1].double(), grid, fp, totals)
        assert totals.tolist() == [0, 0] and int(fp[n - 1]) == 0
    finally:
        ctx.close()
