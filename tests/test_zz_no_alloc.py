"""of_field_minmax_static (include/optflow.h): the min / max step of eq. 3 for callers that cannot
allocate.  Its scratch is a static device array shared by every call, so the test makes TWO calls in a row with different
sizes (the second smaller: stale partials of the first stay in the array behind it) and compares each with the existing path,
of_field_minmax, bit for bit (integer min / max on both sides: the tolerance of the other eq. 3 tests is equality).

Collected last on purpose (the suite runs with pytest -x).  Runs alone in a fresh process or after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def B():
    from paper_1306_2461_b200 import binding
    binding.lib()          # fails loudly if liboptflow.so is missing
    return binding


def _field(torch, W, H, seed):
    g = np.random.default_rng(13062461 + seed)
    f = g.normal(0.0, 3.0, (H, W)).astype(np.float32)
    m = (g.random((H, W)) < 0.9).astype(np.uint8)
    f[H // 3, W // 2] = np.nan                       # ignored by both paths
    iy, ix = np.unravel_index(np.nanargmax(f), f.shape)
    m[iy, ix] = 0                                    # the global maximum is not an available vector
    return torch.from_numpy(f).cuda(), torch.from_numpy(m).cuda(), f, m


def test_static_minmax_matches_handle_path_on_two_calls_in_a_row(torch, B):
    out = torch.empty(2, dtype=torch.float32, device="cuda")          # the caller's output buffer
    # 1283 x 1021 = 1 309 943 pixels: 320 chunks with a ragged tail; then 333 x 251 = 83 583: 21 chunks
    for call, (W, H) in enumerate([(1283, 1021), (333, 251)]):
        fd, md, fh, mh = _field(torch, W, H, call)
        with B.OpticalFlow(W, H, 1, 4, 1, 0) as of:
            for valid_d, valid_h in ((md, mh != 0), (None, np.ones_like(mh, bool))):
                ref = of.field_minmax(fd, valid_d)
                out.fill_(123.0)
                B.field_minmax_static(fd, out, valid_d)
                torch.cuda.synchronize()
                assert torch.equal(out.view(torch.int32), ref.view(torch.int32)), (call, W, H, out.tolist(), ref.tolist())
                sel = fh[valid_h & ~np.isnan(fh)]
                assert out[0].item() == float(sel.min()) and out[1].item() == float(sel.max())
                # unaligned views take the scalar loop: same values
                flat = fd.reshape(-1)[1:]
                vflat = valid_d.reshape(-1)[1:] if valid_d is not None else None
                B.field_minmax_static(flat, out, vflat)
                torch.cuda.synchronize()
                s2 = fh.reshape(-1)[1:][(valid_h.reshape(-1) & ~np.isnan(fh.reshape(-1)))[1:]]
                assert out[0].item() == float(s2.min()) and out[1].item() == float(s2.max())


def test_static_minmax_rejects_sizes_beyond_the_scratch_array(torch, B):
    out = torch.empty(2, dtype=torch.float32, device="cuda")
    small = torch.zeros(16, dtype=torch.float32, device="cuda")
    L = B.lib()
    rc = L.of_field_minmax_static(small.data_ptr(), None, B.OF_STATIC_MAX_PIXELS + 1, out.data_ptr(), None)
    assert rc == B.OF_ERR_INVALID_ARG and "OF_STATIC_MAX_PIXELS" in B.last_error() and str(B.OF_STATIC_MAX_PIXELS) in B.last_error()
    assert L.of_field_minmax_static(small.data_ptr(), None, 0, out.data_ptr(), None) == B.OF_ERR_INVALID_ARG
    assert L.of_field_minmax_static(None, None, 16, out.data_ptr(), None) == B.OF_ERR_INVALID_ARG
    # and the array still works afterwards
    B.field_minmax_static(small, out)
    torch.cuda.synchronize()
    assert out.tolist() == [0.0, 0.0]
