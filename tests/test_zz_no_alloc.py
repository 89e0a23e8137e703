"""dmpt_spectral_bounds_noalloc (include/dmpt.h): step a1 with its scratch in a static device array,
for callers that cannot allocate.  Checked against the existing path (dmpt_spectral_bounds through a context) on calls
in a row that share the static scratch, and against the oracle's Gershgorin bounds.

This file is named to be collected last: the run uses `pytest -x`.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

TOL = 2e-6          # tests/test_gpu_parity.py, test_a1_gershgorin_matches_oracle: fp32 partial sums per lane


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda:0")


def _sym(n, seed):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((n, n))
    return ((a + a.T) / 2).astype(np.float32)


def _existing(h0_dev, n, dev):
    from paper_2203_09621_b200 import Dmpt
    s = Dmpt(n, device=dev)
    lo, hi = s.spectral_bounds(h0_dev)
    s.close()
    return lo, hi


def test_no_alloc_bounds_match_existing_path_on_calls_in_a_row(dev):
    """Two (and more) calls in a row on one stream, sizes going down as well as up so that rows left in the scratch by
    the call before would show; aligned and unaligned leading dimensions.  The arithmetic is that of the existing
    kernel, so the results are equal; the tolerance of the a1 parity test is what is asserted against the oracle."""
    from oracle.dnn_sp2_pt import gershgorin
    from paper_2203_09621_b200 import spectral_bounds_noalloc

    out = torch.full((2,), float("nan"), dtype=torch.float64, device=dev)
    for k, n in enumerate([1000, 333, 1, 37, 2048, 128]):
        h0 = _sym(n, 7 + n)
        m = torch.from_numpy(h0).to(dev)
        pad = torch.zeros((n, n + 5), dtype=torch.float32, device=dev)
        pad[:, :n] = m
        want = _existing(m, n, dev)
        rlo, rhi = gershgorin(h0)
        scale = max(abs(rlo), abs(rhi), 1.0)
        for mat in (pad[:, :n], m):
            out.fill_(float("nan"))
            spectral_bounds_noalloc(mat, out)
            got = out.cpu().numpy()
            assert abs(got[0] - want[0]) <= TOL * scale and abs(got[1] - want[1]) <= TOL * scale, (n, got, want)
            assert abs(got[0] - rlo) <= TOL * scale and abs(got[1] - rhi) <= TOL * scale, (n, got, (rlo, rhi))
        # the same matrix (m, the last of the two above) again: identical bits, and those of the existing path
        assert got[0] == want[0] and got[1] == want[1]
        spectral_bounds_noalloc(m, out)
        again = out.cpu().numpy()
        assert np.array_equal(got, again)


def test_no_alloc_allocates_nothing_and_rejects_sizes_beyond_the_limit(dev):
    from paper_2203_09621_b200 import binding as B

    n = 512
    m = torch.from_numpy(_sym(n, 3)).to(dev)
    out = torch.zeros(2, dtype=torch.float64, device=dev)
    B.spectral_bounds_noalloc(m, out)                  # first call on this device: module load, symbol address
    torch.cuda.synchronize(dev)
    first = out.clone()
    free0, _ = torch.cuda.mem_get_info(dev)
    alloc0 = torch.cuda.memory_allocated(dev)
    for _ in range(20):
        B.spectral_bounds_noalloc(m, out)
    torch.cuda.synchronize(dev)
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 >= free0 and torch.cuda.memory_allocated(dev) == alloc0
    assert torch.equal(out, first)
    # on a side stream, ordered after the default stream
    side = torch.cuda.Stream(device=dev)
    side.wait_stream(torch.cuda.current_stream(dev))
    out2 = torch.zeros(2, dtype=torch.float64, device=dev)
    B.spectral_bounds_noalloc(m, out2, stream=side)
    side.synchronize()
    assert torch.equal(out2, first)
    # limits and argument errors: nothing is enqueued, the pointers are not touched
    assert B.dmpt_spectral_bounds_noalloc(m.data_ptr(), B.DMPT_NOALLOC_MAX_N + 1, B.DMPT_NOALLOC_MAX_N + 1,
                                          out.data_ptr()) == B.DMPT_ELIMIT
    assert "limit" in B.dmpt_strerror(B.DMPT_ELIMIT)
    assert B.dmpt_spectral_bounds_noalloc(m.data_ptr(), 0, 0, out.data_ptr()) == B.DMPT_EINVAL
    assert B.dmpt_spectral_bounds_noalloc(m.data_ptr(), n, n - 1, out.data_ptr()) == B.DMPT_EINVAL
    assert B.dmpt_spectral_bounds_noalloc(0, n, n, out.data_ptr()) == B.DMPT_EINVAL
    assert B.dmpt_spectral_bounds_noalloc(m.data_ptr(), n, n, 0) == B.DMPT_EINVAL
    with pytest.raises(ValueError):
        B.spectral_bounds_noalloc(m.double(), out)
    torch.cuda.synchronize(dev)
    assert torch.equal(out, first)


def test_no_alloc_largest_rows(dev):
    """BASELINE.json's size, n = 16384 (1 GiB of fp32, 2048 row blocks over 1184 resident ones: the grid-stride loop and
    the last-block reduction over all rows), against the existing path."""
    from paper_2203_09621_b200 import spectral_bounds_noalloc

    n = 16384
    g = torch.Generator(device=dev).manual_seed(5)
    a = torch.randn((n, n), dtype=torch.float32, device=dev, generator=g)
    m = (a + a.T) * 0.5
    del a
    out = torch.zeros(2, dtype=torch.float64, device=dev)
    spectral_bounds_noalloc(m, out)
    got = out.cpu().numpy()
    want = _existing(m, n, dev)
    scale = max(abs(want[0]), abs(want[1]), 1.0)
    assert abs(got[0] - want[0]) <= TOL * scale and abs(got[1] - want[1]) <= TOL * scale
