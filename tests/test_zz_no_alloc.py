"""mcdc_tallies_get_noalloc: the tally read-out for callers that cannot allocate device memory.

Some programs that embed libmcdc.so must never see it call cudaMalloc: all of the GPU's memory has already been
given to a pool (PyTorch's caching allocator, a fixed per-rank budget), or the read-out sits in a timing-critical
loop where cudaMalloc / cudaFree would make the host wait for the whole device.  For them the library keeps the
scratch of its statistics kernel in a fixed 16 MiB array of its own device image (include/mcdc.h).  These tests
hold that entry point to the ordinary one, mcdc_tallies_get, at the bars the other GPU tests use for tallies
(mean 1e-9 relative, sdev 1e-6 relative), on calls made back to back: the array is shared by every handle and
keeps the previous call's contents, so a call must not be able to see what the one before it left behind.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process (the first call does the one-time
address look-up) and after the other tests (the library is then already loaded and used).
"""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(300)]


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()                       # fails loudly if libmcdc.so is missing
    return M


def _same(got, ref):
    (mg, sg), (mr, sr) = got, ref
    scale = np.abs(mr).max()
    assert scale > 0.0 and np.count_nonzero(mr) > 10                      # a run that scored: not zeros against zeros
    assert np.all(np.abs(mg - mr) <= 1e-9 * np.maximum(np.abs(mr), np.abs(mg)) + 1e-13 * scale)
    assert np.allclose(sg, sr, rtol=1e-6, atol=1e-12 * scale)


def _large_mesh_problem():
    """The duct of config 2 on a 30 x 50 x 30 x 20 mesh: 900 000 bins, large enough that mcdc_tallies_get itself
    computes on the device (>= 2^18 bins) and just under the fixed array's 2^20."""
    from workloads import configs as W
    p = W.config2_lduct(n_histories=40_000, n_batches=4)
    p.mesh_n = np.array([30, 50, 30], dtype=np.int32)
    return p


def test_noalloc_readout_equals_tallies_get_on_calls_in_a_row(M):
    import torch
    from workloads import configs as W
    pa = _large_mesh_problem()
    assert (1 << 18) <= pa.n_bins <= M.NOALLOC_MAX_BINS
    pb = W.config3_pin_lattice(n_histories=20_000, n_batches=4)        # 40 460 bins: a shorter read-out into the same array
    a, b = M.Problem(pa), M.Problem(pb)
    a.run(); b.run()
    ref_a, ref_b = a.tallies(), b.tallies()                             # the existing path
    assert not np.array_equal(ref_a[0].ravel()[:pb.n_bins], ref_b[0].ravel())
    # two calls in a row on the same handle, then a smaller problem into the array that still holds a's numbers,
    # then a again over b's
    _same(a.tallies_noalloc(), ref_a)
    _same(a.tallies_noalloc(), ref_a)
    _same(b.tallies_noalloc(), ref_b)
    _same(a.tallies_noalloc(), ref_a)
    # more histories change the accumulators; the read-out follows them (nothing is cached from the earlier calls)
    b.run(seed=pb.seed + 1)
    ref_b2 = b.tallies()
    assert not np.array_equal(ref_b2[0], ref_b[0])
    _same(b.tallies_noalloc(), ref_b2)
    # and the point of it: with the caller's result arrays in place, a call leaves the GPU's free memory as it found it
    out = (np.empty(pa.n_bins), np.empty(pa.n_bins))
    M.mcdc_tallies_get_noalloc(a._h, pa.n_bins, out=out)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    M.mcdc_tallies_get_noalloc(a._h, pa.n_bins, out=out)
    assert torch.cuda.mem_get_info()[0] == free_before
    _same((out[0].reshape(ref_a[0].shape), out[1].reshape(ref_a[1].shape)), ref_a)
    a.close(); b.close()


def test_noalloc_readout_refuses_what_the_fixed_array_cannot_hold(M):
    from workloads import configs as W
    p = W.config2_lduct(n_histories=1_000, n_batches=1)                # BASELINE config 2's mesh: 7.2e6 bins
    assert p.n_bins > M.NOALLOC_MAX_BINS
    g = M.Problem(p, max_batches_in_flight=1)
    with pytest.raises(M.McdcError) as e:
        g.tallies_noalloc()
    assert e.value.code == -4 and "MCDC_NOALLOC_MAX_BINS" in str(e.value) and str(p.n_bins) in str(e.value)
    g.close()
    q = W.config0_infinite_medium(n_histories=1_000, n_batches=2)
    h = M.Problem(q)
    with pytest.raises(M.McdcError) as e:
        h.tallies_noalloc()                                             # nothing has run yet: as mcdc_tallies_get
    assert e.value.code == -1
    h.run()
    with pytest.raises(M.McdcError) as e:
        M.mcdc_tallies_get_noalloc(h._h, q.n_bins + 1)                  # not this problem's bin count
    assert e.value.code == -4
    m, s = h.tallies_noalloc()
    mr, sr = h.tallies()
    assert np.allclose(m, mr, rtol=1e-9, atol=0.0) and np.allclose(s, sr, rtol=1e-6, atol=1e-12 * np.abs(mr).max())
    h.close()
